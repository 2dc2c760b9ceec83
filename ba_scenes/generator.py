"""Seeded synthetic bundle-adjustment scenes shaped like BASELINE.json `configs`.

Recipe.  The paper measures on
the BAL dataset, which is not available here; these scenes
stand in for it with BAL-like shapes (N_c << N_p, mean track 5-8, 9-parameter
cameras) and reproduce no dataset record.

All arrays are rounded to float32 ONCE; the oracle up-casts those float32 values
to float64 and the CUDA path uses them as they are, so both sides see
bit-identical inputs.

Nothing here is solver arithmetic.  The only model evaluation is the forward
projection needed to synthesise pixel measurements; it uses
`scipy.spatial.transform.Rotation` and is imported by neither the oracle nor
the CUDA kernels for their own computation.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional, Tuple

import numpy as np
from scipy.spatial.transform import Rotation

# ---------------------------------------------------------------------------
# Config table: BASELINE.json `configs[0..4]`, readings per SURVEY.md 8(d).
# ---------------------------------------------------------------------------
CONFIGS: Dict[str, dict] = {
    # configs[0]
    "tiny": dict(seed=0, geometry="ring", num_cameras=16, num_points=1_000,
                 track="uniform", track_lo=4, track_hi=8,
                 lm_iterations=10, pcg_max_iter=50, pcg_rel_tol=1e-6,
                 robust_loss=0, robust_scale=0.0, outlier_fraction=0.0),
    # configs[1]
    "small": dict(seed=1, geometry="ring", num_cameras=64, num_points=20_000,
                  track="uniform", track_lo=3, track_hi=10,
                  lm_iterations=20, pcg_max_iter=100, pcg_rel_tol=1e-6,
                  robust_loss=0, robust_scale=0.0, outlier_fraction=0.0),
    # configs[2]: 1,800 cameras on a 30 x 60 grid; L = min(12, 2 + Geom(0.235))
    "mid": dict(seed=2, geometry="grid", grid=(30, 60), num_points=1_000_000,
                track="geometric", track_p=0.235, track_lo=2, track_hi=12,
                lm_iterations=20, pcg_max_iter=100, pcg_rel_tol=1e-6,
                robust_loss=0, robust_scale=0.0, outlier_fraction=0.0),
    # configs[3]: 13,700 cameras on a 100 x 137 grid; L = 2 + Geom(0.185) in [2, 50]
    "large": dict(seed=3, geometry="grid", grid=(100, 137), num_points=4_500_000,
                  track="geometric", track_p=0.185, track_lo=2, track_hi=50,
                  lm_iterations=10, pcg_max_iter=100, pcg_rel_tol=1e-6,
                  robust_loss=0, robust_scale=0.0, outlier_fraction=0.0),
    # configs[4]: Zipf(1.1) camera popularity, P(L) ~ L^-2 on [2, 200], 10 % outliers, Cauchy c = 2 px
    "skewed": dict(seed=4, geometry="ring", num_cameras=5_000, num_points=2_000_000,
                   track="powerlaw", track_alpha=2.0, track_lo=2, track_hi=200,
                   popularity="zipf", zipf_s=1.1,
                   lm_iterations=20, pcg_max_iter=100, pcg_rel_tol=1e-6,
                   robust_loss=1, robust_scale=2.0, outlier_fraction=0.10,
                   outlier_range=300.0),
}

# Observations each full config yields (after the grazing cull; pinned by tests/test_generator.py and by the full-size
# GPU tests): lets a caller size a sample against the full workload without generating it.
FULL_OBSERVATIONS = {"tiny": 5_990, "small": 129_449, "mid": 5_035_057, "large": 28_810_876, "skewed": 15_213_972}

GRID_SPACING = 2.0
GRID_HEIGHT = 10.0
RING_RADIUS = 10.0
MAX_DEPTH = -5.0            # every generated observation has P_z <= MAX_DEPTH at the true parameters


@dataclasses.dataclass
class Scene:
    """One BA problem.  `cameras`/`points` are the perturbed START values."""
    name: str
    seed: int
    cameras: np.ndarray          # float32 [Nc, 9]: w0 w1 w2 t0 t1 t2 f k1 k2
    points: np.ndarray           # float32 [Np, 3]
    observations: np.ndarray     # float32 [N, 2] pixels
    camera_index: np.ndarray     # int32 [N]
    point_index: np.ndarray      # int32 [N]
    cameras_true: np.ndarray     # float32 [Nc, 9]
    points_true: np.ndarray      # float32 [Np, 3]
    robust_loss: int
    robust_scale: float
    lm_iterations: int
    pcg_max_iter: int
    pcg_rel_tol: float
    noise_free: bool

    @property
    def num_cameras(self) -> int:
        return int(self.cameras.shape[0])

    @property
    def num_points(self) -> int:
        return int(self.points.shape[0])

    @property
    def num_observations(self) -> int:
        return int(self.observations.shape[0])


# ---------------------------------------------------------------------------
# geometry
# ---------------------------------------------------------------------------
def _ring_cameras(rng: np.random.Generator, n: int) -> Tuple[np.ndarray, np.ndarray]:
    """Camera centres on a radius-10 ring, optical (-z) axis through the origin."""
    phi = 2.0 * math.pi * np.arange(n) / n
    centres = np.stack([RING_RADIUS * np.cos(phi), RING_RADIUS * np.sin(phi), np.zeros(n)], axis=1)
    z_cam = centres / np.linalg.norm(centres, axis=1, keepdims=True)   # points away from the scene
    up = np.array([0.0, 0.0, 1.0])
    x_cam = np.cross(up, z_cam)
    x_cam /= np.linalg.norm(x_cam, axis=1, keepdims=True)
    y_cam = np.cross(z_cam, x_cam)
    r_look = np.stack([x_cam, y_cam, z_cam], axis=1)                    # rows: world -> camera
    return centres, r_look


def _grid_cameras(nx: int, ny: int) -> Tuple[np.ndarray, np.ndarray]:
    """Cameras on a planar nx x ny grid at height 10, looking straight down (-z)."""
    gx, gy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")
    centres = np.stack([GRID_SPACING * gx.ravel(), GRID_SPACING * gy.ravel(),
                        np.full(nx * ny, GRID_HEIGHT)], axis=1).astype(np.float64)
    r_look = np.broadcast_to(np.eye(3), (nx * ny, 3, 3)).copy()
    return centres, r_look


def _camera_params(rng: np.random.Generator, centres: np.ndarray, r_look: np.ndarray) -> np.ndarray:
    n = centres.shape[0]
    eps = rng.normal(0.0, 0.1, size=(n, 3))
    rot = Rotation.from_rotvec(eps) * Rotation.from_matrix(r_look)      # R_j = Exp(eps_j) R_look
    omega = rot.as_rotvec()
    trans = -rot.apply(centres)                                         # t_j = -R_j C_j
    f = rng.uniform(400.0, 600.0, size=n)
    k1 = rng.normal(0.0, 1e-2, size=n)
    k2 = rng.normal(0.0, 1e-4, size=n)
    return np.concatenate([omega, trans, f[:, None], k1[:, None], k2[:, None]], axis=1)


# ---------------------------------------------------------------------------
# track lengths
# ---------------------------------------------------------------------------
def _track_lengths(rng: np.random.Generator, cfg: dict, n_points: int, n_cameras: int) -> np.ndarray:
    lo, hi = cfg["track_lo"], min(cfg["track_hi"], n_cameras)
    if cfg.get("popularity") == "zipf":           # shrunken test scenes: keep the coupon collector finite
        hi = min(hi, max(lo, n_cameras // 4))
    kind = cfg["track"]
    if kind == "uniform":
        length = rng.integers(lo, hi + 1, size=n_points)
    elif kind == "geometric":
        length = lo + (rng.geometric(cfg["track_p"], size=n_points) - 1)
        length = np.minimum(length, hi)
    elif kind == "powerlaw":
        support = np.arange(lo, hi + 1)
        pmf = support.astype(np.float64) ** (-cfg["track_alpha"])
        pmf /= pmf.sum()
        length = rng.choice(support, size=n_points, p=pmf)
    else:
        raise ValueError(kind)
    return length.astype(np.int64)


# ---------------------------------------------------------------------------
# visibility
# ---------------------------------------------------------------------------
def _first_k_of_shuffled(rng, candidates: np.ndarray, length: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Per row: pick `length[i]` of the row's candidates uniformly without replacement.
    Returns (row ids, chosen candidate values), flattened, rows ascending."""
    n, k = candidates.shape
    keys = rng.random((n, k), dtype=np.float32)
    order = np.argsort(keys, axis=1)
    shuffled = np.take_along_axis(candidates, order, axis=1)
    mask = np.arange(k)[None, :] < length[:, None]
    rows = np.broadcast_to(np.arange(n)[:, None], (n, k))[mask]
    return rows, shuffled[mask]


def _visibility_uniform(rng, n_cameras: int, length: np.ndarray, chunk: int = 1 << 18):
    pts, cams = [], []
    for s in range(0, length.shape[0], chunk):
        ln = length[s:s + chunk]
        cand = np.broadcast_to(np.arange(n_cameras, dtype=np.int32)[None, :], (ln.shape[0], n_cameras))
        r, c = _first_k_of_shuffled(rng, cand, ln)
        pts.append(r + s)
        cams.append(c)
    return np.concatenate(pts), np.concatenate(cams)


def _visibility_grid(rng, nx: int, ny: int, xy: np.ndarray, length: np.ndarray, chunk: int = 1 << 19):
    """Each point chooses its cameras among the K x K block of grid cameras centred on it
    (K = 4 -> the 16 horizontally nearest; K = 8 when the track is longer than 16)."""
    pts, cams = [], []
    n = xy.shape[0]
    for k_side, sel in ((4, length <= 16), (8, length > 16)):
        idx_all = np.nonzero(sel)[0]
        kx, ky = min(k_side, nx), min(k_side, ny)
        for s in range(0, idx_all.shape[0], chunk):
            idx = idx_all[s:s + chunk]
            cx = np.floor(xy[idx, 0] / GRID_SPACING).astype(np.int64)
            cy = np.floor(xy[idx, 1] / GRID_SPACING).astype(np.int64)
            x0 = np.clip(cx - (kx // 2 - 1), 0, nx - kx)
            y0 = np.clip(cy - (ky // 2 - 1), 0, ny - ky)
            ox, oy = np.meshgrid(np.arange(kx), np.arange(ky), indexing="ij")
            cand = ((x0[:, None] + ox.ravel()[None, :]) * ny + (y0[:, None] + oy.ravel()[None, :])).astype(np.int32)
            ln = np.minimum(length[idx], kx * ky)
            r, c = _first_k_of_shuffled(rng, cand, ln)
            pts.append(idx[r])
            cams.append(c)
    pts = np.concatenate(pts)
    cams = np.concatenate(cams)
    order = np.argsort(pts, kind="stable")
    assert n >= 0
    return pts[order], cams[order]


def _visibility_zipf(rng, n_cameras: int, length: np.ndarray, s: float):
    """Weighted sampling without replacement (successive sampling): popularity ~ rank^-s.
    Draw with replacement, drop repeats within a point, redraw the shortfall."""
    w = np.arange(1, n_cameras + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(w / w.sum())
    cdf[-1] = 1.0
    n = length.shape[0]
    chosen = np.empty(0, dtype=np.int64)          # point * n_cameras + camera, unique, sorted
    need = length.copy()
    for _ in range(64):
        todo = np.nonzero(need > 0)[0]
        if todo.size == 0:
            break
        # the distinct items of an i.i.d. stream, in order of first appearance, ARE a successive
        # sample without replacement; oversample the stream, keep the first `need` new items.
        rep = np.repeat(todo, 3 * need[todo] + 16)
        draw = np.searchsorted(cdf, rng.random(rep.shape[0]), side="right").astype(np.int64)
        key = rep * n_cameras + np.minimum(draw, n_cameras - 1)
        uniq, first = np.unique(key, return_index=True)
        fresh = ~np.isin(uniq, chosen, assume_unique=True)
        uniq, first = uniq[fresh], first[fresh]
        order = np.argsort(first)                 # stream order (point-major, then draw position)
        uniq = uniq[order]
        pt = uniq // n_cameras
        start = np.searchsorted(pt, pt, side="left")
        keep = (np.arange(pt.shape[0]) - start) < need[pt]
        chosen = np.union1d(chosen, uniq[keep])
        need = length - np.bincount(chosen // n_cameras, minlength=n)
    else:
        raise RuntimeError("zipf visibility did not converge")
    return chosen // n_cameras, (chosen % n_cameras).astype(np.int32)


# ---------------------------------------------------------------------------
# forward projection (measurement synthesis only)
# ---------------------------------------------------------------------------
def _project(cameras: np.ndarray, points: np.ndarray, cam_idx: np.ndarray, pt_idx: np.ndarray,
             chunk: int = 1 << 21) -> Tuple[np.ndarray, np.ndarray]:
    """uv = f r p with p = -P_xy / P_z, r = 1 + k1 |p|^2 + k2 |p|^4 (configs[0]).
    Returns (uv [N, 2], depth P_z [N])."""
    rot = Rotation.from_rotvec(cameras[:, 0:3]).as_matrix()
    out = np.empty((cam_idx.shape[0], 2), dtype=np.float64)
    depth = np.empty(cam_idx.shape[0], dtype=np.float64)
    for s in range(0, cam_idx.shape[0], chunk):
        c = cam_idx[s:s + chunk]
        k = pt_idx[s:s + chunk]
        pc = np.einsum("nij,nj->ni", rot[c], points[k]) + cameras[c, 3:6]
        p = -pc[:, 0:2] / pc[:, 2:3]
        n2 = np.sum(p * p, axis=1)
        r = 1.0 + cameras[c, 7] * n2 + cameras[c, 8] * n2 * n2
        out[s:s + chunk] = (cameras[c, 6] * r)[:, None] * p
        depth[s:s + chunk] = pc[:, 2]
    return out, depth


# ---------------------------------------------------------------------------
# public entry point
# ---------------------------------------------------------------------------
def make_scene(name: str, *, noise_free: bool = False, seed: Optional[int] = None,
               num_cameras: Optional[int] = None, num_points: Optional[int] = None,
               grid: Optional[Tuple[int, int]] = None, shuffle: bool = True) -> Scene:
    """Build config `name` ("tiny" | "small" | "mid" | "large" | "skewed").

    `num_cameras`, `num_points`, `grid` shrink a config for tests (same recipe, smaller counts).
    `noise_free=True` gives the zero-pixel-noise twin (same perturbed start, no outliers).
    `shuffle=True` delivers observations in random order (the caller's order is arbitrary).
    """
    cfg = dict(CONFIGS[name])
    if seed is not None:
        cfg["seed"] = seed
    if num_points is not None:
        cfg["num_points"] = num_points
    if grid is not None:
        cfg["grid"] = grid
    if num_cameras is not None:
        if cfg["geometry"] == "grid":
            raise ValueError("grid scenes take grid=(nx, ny), not num_cameras")
        cfg["num_cameras"] = num_cameras
    rng = np.random.default_rng(cfg["seed"])

    # --- cameras and points (truth), rounded to float32 once -----------------------------
    if cfg["geometry"] == "ring":
        centres, r_look = _ring_cameras(rng, cfg["num_cameras"])
        n_cam = cfg["num_cameras"]
        cams_true = _camera_params(rng, centres, r_look)
        pts_true = rng.uniform(-2.0, 2.0, size=(cfg["num_points"], 3))
    else:
        nx, ny = cfg["grid"]
        centres, r_look = _grid_cameras(nx, ny)
        n_cam = nx * ny
        cams_true = _camera_params(rng, centres, r_look)
        n_pts = cfg["num_points"]
        pts_true = np.stack([rng.uniform(0.0, GRID_SPACING * (nx - 1), size=n_pts),
                             rng.uniform(0.0, GRID_SPACING * (ny - 1), size=n_pts),
                             rng.uniform(-1.0, 1.0, size=n_pts)], axis=1)
    cams_true = cams_true.astype(np.float32)
    pts_true = pts_true.astype(np.float32)
    n_pts = pts_true.shape[0]

    # --- visibility ---------------------------------------------------------------------
    length = _track_lengths(rng, cfg, n_pts, n_cam)
    if cfg["geometry"] == "grid":
        pt_idx, cam_idx = _visibility_grid(rng, nx, ny, pts_true[:, 0:2].astype(np.float64), length)
    elif cfg.get("popularity") == "zipf":
        pt_idx, cam_idx = _visibility_zipf(rng, n_cam, length, cfg["zipf_s"])
    else:
        pt_idx, cam_idx = _visibility_uniform(rng, n_cam, length)
    pt_idx = pt_idx.astype(np.int32)
    cam_idx = cam_idx.astype(np.int32)
    n_obs = pt_idx.shape[0]

    # --- measurements -------------------------------------------------------------------
    uv, depth = _project(cams_true.astype(np.float64), pts_true.astype(np.float64), cam_idx, pt_idx)
    # visibility cull (reading G2; C7: no depth guard in the model, so scenes keep P_z <= -5): drop the few
    # grazing observations, never taking a point below two observations
    graze = depth > MAX_DEPTH
    if graze.any():
        left = np.bincount(pt_idx, minlength=n_pts) - np.bincount(pt_idx[graze], minlength=n_pts)
        keep = ~(graze & (left[pt_idx] >= 2))
        uv, cam_idx, pt_idx = uv[keep], cam_idx[keep], pt_idx[keep]
        n_obs = pt_idx.shape[0]
    noise = rng.normal(0.0, 1.0, size=(n_obs, 2))
    outlier = rng.random(n_obs) < cfg["outlier_fraction"]
    outlier_px = rng.uniform(-cfg.get("outlier_range", 300.0), cfg.get("outlier_range", 300.0), size=(n_obs, 2))
    if not noise_free:
        uv = uv + noise
        uv[outlier] = outlier_px[outlier]
    obs = uv.astype(np.float32)

    # --- perturbed start ----------------------------------------------------------------
    # N(0, 0.01) on rotation / translation, applied in the camera's own frame (reading G1):
    # R0 = Exp(d_w) R about the camera centre, C0 = C + d_c, t0 = -R0 C0.  Adding the noise to (w, t) of
    # P = R X + t literally would turn far cameras about the WORLD origin and throw their points by
    # |X| * 0.01 (up to ~8 units on the large grid), putting hundreds of observations behind the camera.
    cams0 = cams_true.astype(np.float64)
    rot_true = Rotation.from_rotvec(cams0[:, 0:3])
    centre = -rot_true.inv().apply(cams0[:, 3:6])
    rot0 = Rotation.from_rotvec(rng.normal(0.0, 0.01, size=(n_cam, 3))) * rot_true
    centre0 = centre + rng.normal(0.0, 0.01, size=(n_cam, 3))
    cams0[:, 0:3] = rot0.as_rotvec()
    cams0[:, 3:6] = -rot0.apply(centre0)
    pts0 = pts_true.astype(np.float64) + rng.normal(0.0, 0.05, size=(n_pts, 3))

    if shuffle:
        perm = rng.permutation(n_obs)
        obs, cam_idx, pt_idx = obs[perm], cam_idx[perm], pt_idx[perm]

    return Scene(name=name, seed=cfg["seed"],
                 cameras=np.ascontiguousarray(cams0.astype(np.float32)),
                 points=np.ascontiguousarray(pts0.astype(np.float32)),
                 observations=np.ascontiguousarray(obs),
                 camera_index=np.ascontiguousarray(cam_idx),
                 point_index=np.ascontiguousarray(pt_idx),
                 cameras_true=cams_true, points_true=pts_true,
                 robust_loss=cfg["robust_loss"], robust_scale=float(cfg["robust_scale"]),
                 lm_iterations=cfg["lm_iterations"], pcg_max_iter=cfg["pcg_max_iter"],
                 pcg_rel_tol=cfg["pcg_rel_tol"], noise_free=noise_free)


def scene_summary(scene: Scene) -> dict:
    """Counts used by the generator pins."""
    track = np.bincount(scene.point_index, minlength=scene.num_points)
    per_cam = np.bincount(scene.camera_index, minlength=scene.num_cameras)
    return dict(name=scene.name, seed=scene.seed, num_cameras=scene.num_cameras,
                num_points=scene.num_points, num_observations=scene.num_observations,
                track_mean=float(track.mean()), track_min=int(track.min()), track_max=int(track.max()),
                cam_obs_max=int(per_cam.max()), cam_obs_min=int(per_cam.min()),
                top_camera_share=float(per_cam.max() / max(1, scene.num_observations)))
