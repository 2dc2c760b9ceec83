"""GPU edge cases through the C ABI: empty and degenerate problems, unobserved nodes, the longest supported
track, every tile size, both Schur-matvec kernels, error codes of include/caspar_ba.h."""
import numpy as np
import pytest

import oracle
import paper_2605_30583_b200 as pkg
from oracle import binding as ob

pytestmark = pytest.mark.gpu

LAM = float(np.float32(1e-2))


def rel_l2(a, b):
    a, b = np.asarray(a, np.float64).ravel(), np.asarray(b, np.float64).ravel()
    den = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / den) if den > 0 else float(np.linalg.norm(a))


def _step_matches(g, o, iters=25, tol=1e-4):
    cg, co = g.linearize(), o.linearize()
    assert abs(cg - co) <= 1e-5 * max(co, 1e-30)
    g.pcg_solve(LAM, 0.0, iters)
    o.pcg_solve(LAM, 0.0, iters)
    d_g, d_o = g.export(pkg.DELTA), o.export(ob.DELTA)
    assert rel_l2(d_g, d_o) <= tol, rel_l2(d_g, d_o)
    return d_g, d_o


def test_empty_problems():
    z2, zi = np.zeros((0, 2), np.float32), np.zeros(0, np.int32)
    g = pkg.CasparBA(np.zeros((2, 9), np.float32), np.zeros((3, 3), np.float32), z2, zi, zi)
    assert g.linearize() == 0.0
    info = g.pcg_solve(LAM, 1e-6, 10)
    assert info.iterations == 0 and info.converged
    assert np.all(g.export(pkg.DELTA) == 0.0)
    st = g.lm_step(LAM, 1e-6, 10, accept_mode=1)
    assert st.cost_before == 0.0 and st.cost_after == 0.0
    g.close()
    g = pkg.CasparBA(np.zeros((0, 9), np.float32), np.zeros((0, 3), np.float32), z2, zi, zi)
    assert g.linearize() == 0.0 and g.cost() == 0.0
    g.close()


def test_error_codes():
    one9, one3 = np.zeros((1, 9), np.float32), np.zeros((1, 3), np.float32)
    with pytest.raises(pkg.CasparError) as e:      # index out of range (the binding hands DEVICE index arrays over)
        pkg.CasparBA(one9, one3, np.zeros((1, 2), np.float32), np.array([1], np.int32), np.array([0], np.int32))
    assert e.value.code == -1 and "observation 0 (validated on the device)" in str(e.value)
    ci = np.zeros(5000, np.int32)
    pi = np.zeros(5000, np.int32)
    pi[[4321, 777]] = 9                            # the LOWEST offending observation is reported
    with pytest.raises(pkg.CasparError) as e:
        pkg.CasparBA(one9, one3, np.zeros((5000, 2), np.float32), ci, pi)
    assert e.value.code == -1 and "observation 777 (validated on the device)" in str(e.value)
    with pytest.raises(pkg.CasparError) as e:      # negative index
        pkg.CasparBA(one9, one3, np.zeros((1, 2), np.float32), np.array([0], np.int32), np.array([-1], np.int32))
    assert e.value.code == -1
    with pytest.raises(pkg.CasparError) as e:      # Cauchy without a scale
        pkg.CasparBA(one9, one3, np.zeros((0, 2), np.float32), np.zeros(0, np.int32), np.zeros(0, np.int32),
                     robust_loss=1, robust_scale=0.0)
    assert e.value.code == -1
    g = pkg.CasparBA(one9, one3, np.zeros((0, 2), np.float32), np.zeros(0, np.int32), np.zeros(0, np.int32))
    with pytest.raises(pkg.CasparError) as e:      # pcg_solve before linearize
        g.pcg_solve(LAM, 1e-6, 1)
    assert e.value.code == -5
    with pytest.raises(pkg.CasparError) as e:      # export before linearize
        g.export(pkg.RESIDUALS)
    assert e.value.code == -5
    with pytest.raises(pkg.CasparError) as e:      # negative damping
        g.linearize()
        g.pcg_solve(-1.0, 1e-6, 1)
    assert e.value.code == -1
    g.close()


def test_depth_zero_is_a_numeric_error():
    """Reading C7: P_z = 0 is not guarded -> non-finite cost -> ENUMERIC, as in the oracle."""
    cam = np.r_[0, 0, 0, 0, 0, 0, 500.0, 0, 0][None, :].astype(np.float32)
    g = pkg.CasparBA(cam, np.array([[1.0, 1.0, 0.0]], np.float32), np.zeros((1, 2), np.float32),
                     np.array([0], np.int32), np.array([0], np.int32))
    with pytest.raises(pkg.CasparError) as e:
        g.linearize()
    assert e.value.code == -4
    g.close()


def test_unobserved_nodes_get_zero_step(scene_cache):
    s = scene_cache("tiny")
    cams = np.vstack([s.cameras[:1], s.cameras, s.cameras[:1]])         # cameras 0 and 17: no observations
    pts = np.vstack([s.points[:1], s.points, s.points[:2]])             # points 0, 1001, 1002: none
    ci, pi = s.camera_index + 1, s.point_index + 1
    g = pkg.CasparBA(cams, pts, s.observations, ci, pi)
    o = oracle.OracleBA(cams, pts, s.observations, ci, pi)
    d_g, d_o = _step_matches(g, o)
    nc9 = 9 * 18
    assert np.all(d_g[:9] == 0.0) and np.all(d_g[9 * 17:nc9] == 0.0)
    assert np.all(d_g[nc9:nc9 + 3] == 0.0) and np.all(d_g[nc9 + 3 * 1001:] == 0.0)
    before = g.points.cpu().numpy().copy()
    g.lm_step(LAM, 0.0, 10, accept_mode=1)
    after = g.points.cpu().numpy()
    assert np.array_equal(before[0], after[0]) and np.array_equal(before[1001:], after[1001:])
    g.close()


def _long_track_scene(track, seed=7):
    """One point seen by `track` cameras on the ring plus ordinary points (ragged tiles around a full one);
    ~20 ordinary points per camera keep every camera block well conditioned (>= 100 observations each)."""
    from ba_scenes import make_scene
    s = make_scene("small", num_cameras=max(track, 16), num_points=20 * track + 1, seed=seed)
    nc = s.num_cameras
    keep = s.point_index != 0
    cam_true, X = s.cameras_true.astype(np.float64), s.points_true[0].astype(np.float64)
    from scipy.spatial.transform import Rotation
    P = Rotation.from_rotvec(cam_true[:track, :3]).apply(X) + cam_true[:track, 3:6]
    p = -P[:, :2] / P[:, 2:3]
    n2 = (p * p).sum(1)
    uv = (cam_true[:track, 6] * (1 + cam_true[:track, 7] * n2 + cam_true[:track, 8] * n2 * n2))[:, None] * p
    obs = np.vstack([s.observations[keep], uv.astype(np.float32)])
    ci = np.r_[s.camera_index[keep], np.arange(track, dtype=np.int32)].astype(np.int32)
    pi = np.r_[s.point_index[keep], np.zeros(track, np.int32)].astype(np.int32)
    assert nc >= track
    return s.cameras, s.points, obs, ci, pi


@pytest.mark.parametrize("track", [257, 512, 1024])
def test_longest_tracks(track):
    """A track longer than 256 / 512 forces T = 512 / 1024; CASPAR_BA_MAX_TRACK = 1024 is the limit."""
    args = _long_track_scene(track)
    g = pkg.CasparBA(*args)
    o = oracle.OracleBA(*args)
    assert g.stats().tile_slots == (512 if track <= 512 else 1024)
    _step_matches(g, o)
    p = np.random.default_rng(3).normal(size=9 * g.nc).astype(np.float32).astype(np.float64)
    assert rel_l2(g.schur_matvec(LAM, p), o.schur_matvec(LAM, p)) <= 1e-4
    g.close()


def test_track_over_the_limit_is_rejected():
    args = _long_track_scene(1025)
    with pytest.raises(pkg.CasparError) as e:
        pkg.CasparBA(*args)
    assert e.value.code == -1


@pytest.mark.parametrize("tile", [128, 192, 256, 512, 1024])
@pytest.mark.parametrize("pipeline", ["0", "1"])
def test_every_tile_size_and_both_matvec_kernels(scene_cache, monkeypatch, tile, pipeline):
    """CASPAR_BA_TILE / CASPAR_BA_PIPELINE are read at create: T in {128, 192, 256, 512, 1024}; the one-block-per-tile
    Schur pass and the persistent TMA-pipelined one (tiles of <= 256 slots) must both match the oracle."""
    monkeypatch.setenv("CASPAR_BA_TILE", str(tile))
    monkeypatch.setenv("CASPAR_BA_PIPELINE", pipeline)
    monkeypatch.setenv("CASPAR_BA_LIN_PIPELINE", pipeline)     # the same choice for linearize / cost
    s = scene_cache("mid", grid=(10, 12), num_points=40_000)
    g = pkg.CasparBA.from_scene(s)
    o = oracle.OracleBA.from_scene(s)
    assert g.stats().tile_slots == tile
    assert g.stats().matvec_pipelined == (1 if pipeline == "1" and tile <= 256 else 0)
    assert g.stats().linearize_pipelined == (1 if pipeline == "1" and tile <= 256 else 0)
    assert abs(g.cost() - o.cost()) <= 1e-9 * o.cost()         # the residual-only instantiation
    _step_matches(g, o)
    p = np.random.default_rng(3).normal(size=9 * g.nc).astype(np.float32).astype(np.float64)
    assert rel_l2(g.schur_matvec(LAM, p), o.schur_matvec(LAM, p)) <= 1e-4
    g.close()


def test_rejected_step_keeps_the_linearization_and_parameters(scene_cache):
    s = scene_cache("tiny")
    g = pkg.CasparBA.from_scene(s)
    cams0, pts0 = g.cameras.clone(), g.points.clone()
    a = g.lm_step(LAM, 0.0, 20, accept_mode=2)
    assert not a.accepted and (g.cameras == cams0).all() and (g.points == pts0).all()
    launches = g.stats().kernels_launched
    b = g.lm_step(LAM, 0.0, 20, accept_mode=2)              # same lambda: same step, no re-linearization
    assert abs(b.cost_after - a.cost_after) <= 1e-6 * a.cost_after and b.cost_before == a.cost_before
    assert g.stats().kernels_launched - launches < launches  # linearize kernels were skipped
    c = g.lm_step(LAM, 0.0, 20, accept_mode=1)
    assert c.accepted and not (g.cameras == cams0).all()
    assert abs(g.cost() - c.cost_after) <= 1e-6 * c.cost_after
    g.close()


def test_host_parameter_round_trip(scene_cache):
    import torch
    s = scene_cache("tiny")
    g = pkg.CasparBA.from_scene(s)
    cam_h = torch.from_numpy(s.cameras.copy()).pin_memory()
    pts_h = torch.from_numpy(s.points.copy()).pin_memory()
    g.set_parameters_host(cam_h, pts_h)
    st = g.lm_step(LAM, 0.0, 20, accept_mode=1)
    g.get_parameters_host(cam_h, pts_h)
    assert torch.equal(cam_h, g.cameras.cpu()) and torch.equal(pts_h, g.points.cpu())
    o = oracle.OracleBA.from_scene(s)
    so = o.lm_step(LAM, 0.0, 20, accept_mode=1)
    assert abs(st.cost_after - so.cost_after) <= 1e-4 * so.cost_after
    g.close()


@pytest.mark.parametrize("graph", ["0", "1"])
def test_pcg_chunks_as_a_cuda_graph_and_kernel_by_kernel_agree(scene_cache, monkeypatch, graph):
    """CASPAR_BA_GRAPH=0 launches every PCG kernel on its own; by default whole chunks of 8 iterations are one
    CUDA-graph launch and the remainder (25 = 3 x 8 + 1) goes kernel by kernel.  Same iteration counts, same step;
    the tolerance-driven run stops at the same place."""
    monkeypatch.setenv("CASPAR_BA_GRAPH", graph)
    s = scene_cache("small")
    g = pkg.CasparBA.from_scene(s)
    o = oracle.OracleBA.from_scene(s)
    _step_matches(g, o, iters=25)
    ig, io = g.pcg_solve(LAM, 1e-6, 100), o.pcg_solve(LAM, 1e-6, 100)
    assert ig.converged and io.converged and abs(ig.iterations - io.iterations) <= 1
    assert rel_l2(g.export(pkg.DELTA), o.export(ob.DELTA)) <= 1e-4
    g.close()
    o.close()
