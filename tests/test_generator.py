"""Pins for the seeded scene generator: counts and track statistics match BASELINE.json `configs`
(SURVEY.md 8(d) table), inputs are float32, valid and reproducible."""
import numpy as np
import pytest

from ba_scenes import CONFIGS, make_scene, scene_summary


@pytest.mark.parametrize("name", ["tiny", "small", "mid"])
def test_full_observation_table(scene_cache, name):
    from ba_scenes import FULL_OBSERVATIONS
    assert scene_cache(name).num_observations == FULL_OBSERVATIONS[name]   # large / skewed: tests/test_gpu_golden.py


def test_tiny_counts(scene_cache):
    s = scene_cache("tiny")
    m = scene_summary(s)
    assert (m["num_cameras"], m["num_points"]) == (16, 1000)
    assert 5500 <= m["num_observations"] <= 6500            # "~6,000 observations"
    assert m["track_min"] >= 4 and m["track_max"] <= 8      # "seen by 4-8 uniformly chosen cameras"
    assert s.lm_iterations == 10 and s.pcg_max_iter == 50 and s.pcg_rel_tol == 1e-6


def test_small_counts(scene_cache):
    s = scene_cache("small")
    m = scene_summary(s)
    assert (m["num_cameras"], m["num_points"]) == (64, 20000)
    assert 125_000 <= m["num_observations"] <= 135_000      # "~130,000 observations"
    assert m["track_min"] >= 3 and m["track_max"] <= 10
    assert s.lm_iterations == 20 and s.pcg_max_iter == 100


def test_mid_counts(scene_cache):
    s = scene_cache("mid")
    m = scene_summary(s)
    assert (m["num_cameras"], m["num_points"]) == (1800, 1_000_000)
    assert 4_800_000 <= m["num_observations"] <= 5_200_000  # "~5,000,000 observations"
    assert m["track_min"] >= 2 and m["track_max"] <= 12
    # banded camera-camera coupling: a point's cameras lie in a 4 x 4 block of the 30 x 60 grid
    k = np.argsort(s.point_index, kind="stable")
    cam, pt = s.camera_index[k], s.point_index[k]
    gx, gy = cam // 60, cam % 60
    first = np.r_[True, pt[1:] != pt[:-1]]
    seg = np.cumsum(first) - 1
    span_x = np.maximum.reduceat(gx, np.nonzero(first)[0]) - np.minimum.reduceat(gx, np.nonzero(first)[0])
    span_y = np.maximum.reduceat(gy, np.nonzero(first)[0]) - np.minimum.reduceat(gy, np.nonzero(first)[0])
    assert seg.max() + 1 == 1_000_000
    assert span_x.max() <= 3 and span_y.max() <= 3


def test_large_and_skewed_recipes_shrunk():
    """The full Large / Skewed scenes take ~30-60 s to draw; their recipes are pinned on shrunken copies,
    and the full-size counts are checked where the scenes are built anyway (GPU tests, bench)."""
    s = make_scene("large", grid=(20, 27), num_points=200_000)
    m = scene_summary(s)
    assert m["num_cameras"] == 540
    assert abs(m["track_mean"] - 6.4) < 0.1                 # geometric, mean 6.4, truncated to [2, 50]
    assert m["track_min"] >= 2 and m["track_max"] <= 50
    s = make_scene("skewed", num_cameras=1000, num_points=100_000)
    m = scene_summary(s)
    assert m["track_min"] >= 2 and m["track_max"] <= 200
    per_cam = np.bincount(s.camera_index, minlength=1000)
    assert per_cam[0] == per_cam.max()                      # Zipf: rank-1 camera is the most popular
    assert per_cam[:10].sum() > 5 * per_cam[500:510].sum()
    assert s.robust_loss == 1 and s.robust_scale == 2.0
    # ~10 % of pixels are uniform outliers in [-300, 300]^2
    twin = make_scene("skewed", num_cameras=1000, num_points=100_000, noise_free=True, shuffle=False)
    noisy = make_scene("skewed", num_cameras=1000, num_points=100_000, shuffle=False)
    far = np.abs(noisy.observations - twin.observations).max(axis=1) > 8.0
    assert 0.07 < far.mean() < 0.12


def test_config_table_matches_baseline_text():
    assert CONFIGS["large"]["grid"][0] * CONFIGS["large"]["grid"][1] == 13_700
    assert CONFIGS["large"]["num_points"] == 4_500_000
    assert CONFIGS["mid"]["grid"][0] * CONFIGS["mid"]["grid"][1] == 1_800
    assert CONFIGS["skewed"]["num_cameras"] == 5_000 and CONFIGS["skewed"]["num_points"] == 2_000_000
    assert [CONFIGS[k]["seed"] for k in ("tiny", "small", "mid", "large", "skewed")] == [0, 1, 2, 3, 4]


def test_inputs_are_float32_valid_and_reproducible(scene_cache):
    s = scene_cache("tiny")
    for a in (s.cameras, s.points, s.observations):
        assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"] and np.isfinite(a).all()
    assert s.camera_index.dtype == np.int32 and s.point_index.dtype == np.int32
    assert s.camera_index.min() >= 0 and s.camera_index.max() < s.num_cameras
    assert s.point_index.min() >= 0 and s.point_index.max() < s.num_points
    # a (camera, point) pair is observed at most once
    key = s.point_index.astype(np.int64) * s.num_cameras + s.camera_index
    assert np.unique(key).size == key.size
    again = make_scene("tiny")
    assert np.array_equal(again.observations, s.observations) and np.array_equal(again.cameras, s.cameras)
    # start is a perturbation of the truth: N(0, 0.01) on rotation and camera centre (in the camera's own
    # frame, reading C16), N(0, 0.05) on points
    from scipy.spatial.transform import Rotation
    r0 = Rotation.from_rotvec(s.cameras[:, :3].astype(np.float64))
    r1 = Rotation.from_rotvec(s.cameras_true[:, :3].astype(np.float64))
    assert 0.005 < np.std((r0 * r1.inv()).as_rotvec()) < 0.02
    c0 = -r0.inv().apply(s.cameras[:, 3:6].astype(np.float64))
    c1 = -r1.inv().apply(s.cameras_true[:, 3:6].astype(np.float64))
    assert 0.005 < np.std(c0 - c1) < 0.02
    assert 0.04 < np.std(s.points - s.points_true) < 0.06
    assert np.array_equal(s.cameras[:, 6:], s.cameras_true[:, 6:])


@pytest.mark.parametrize("name,kw", [("tiny", {}), ("mid", dict(grid=(8, 10), num_points=3000)),
                                     ("large", dict(grid=(100, 137), num_points=60_000)),
                                     ("skewed", dict(num_cameras=300, num_points=5000))])
def test_points_in_front_of_cameras(name, kw):
    """Reading C7: no epsilon guard, so every generated observation must have P_z well below zero, at the
    true parameters (<= -5) and at the perturbed start (large keeps the full 100 x 137 grid extent here:
    the far cameras are the ones a careless start perturbation would break)."""
    from scipy.spatial.transform import Rotation
    s = make_scene(name, **kw)
    for cams, pts, bound in ((s.cameras_true, s.points_true, -5.0 + 1e-4), (s.cameras, s.points, -4.0)):
        rot = Rotation.from_rotvec(cams[:, :3].astype(np.float64)).as_matrix()
        pc = np.einsum("nij,nj->ni", rot[s.camera_index], pts[s.point_index].astype(np.float64))
        pc += cams[s.camera_index, 3:6]
        assert pc[:, 2].max() < bound
