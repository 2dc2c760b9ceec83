"""GPU parity of the paper's own variants against the oracle's, through the C ABI:

  N3  the Pose3 camera (rotation linearised in its tangent space, retraction on an accepted step) and the d_safe
      depth guard: residuals, Jacobians, blocks, one LM step, a replayed schedule;
  N4  the Schur-Jacobi preconditioner (diagonal blocks of S): the blocks themselves, the PCG step at equal
      iteration counts, iterations to tolerance;
  N1  the full-system PCG with normal residual, no Schur elimination: the step at equal
      iteration counts per parameter class, and its limit against the Schur path's.
Tolerances are test_gpu_parity.py's."""
import numpy as np
import pytest

import oracle
import paper_2605_30583_b200 as pkg
from oracle import binding as ob
from parity_util import (TAIL_CAMERA_TOL, assert_cameras_match, assert_per_class, per_class_rel_l2, rel_l2,
                         scaled_block_rel, significant_step)

pytestmark = pytest.mark.gpu

LAM = float(np.float32(1e-2))
SCENES = {
    "tiny": ("tiny", {}),
    "small": ("small", {}),
    "large": ("large", dict(grid=(12, 16), num_points=30_000)),
    "skewed": ("skewed", dict(num_cameras=300, num_points=30_000)),
}


# ------------------------------------------------------------------ N3: Pose3 camera + d_safe
@pytest.mark.parametrize("key", list(SCENES))
@pytest.mark.parametrize("eps", [0.0, 1e-3])
def test_pose3_linearize_parity(scene_cache, key, eps):
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    g = pkg.CasparBA.from_scene(s, camera_model=1, depth_epsilon=eps)
    o = oracle.OracleBA.from_scene(s, camera_model=1, depth_epsilon=eps)
    cg, co = g.linearize(), o.linearize()
    assert abs(cg - co) <= 1e-5 * co
    r_g, r_o = g.export(pkg.RESIDUALS), o.export(ob.RESIDUALS)
    assert (np.abs(r_g - r_o) <= 1e-6 + 1e-5 * np.abs(r_o)).all()
    for what_g, what_o in ((pkg.JC, ob.JC), (pkg.JP, ob.JP)):
        j_g, j_o = g.export(what_g), o.export(what_o)
        row_scale = np.abs(j_o).max(axis=2, keepdims=True)
        assert (np.abs(j_g - j_o) <= 1e-6 + 1e-5 * np.maximum(np.abs(j_o), row_scale)).all()
        assert rel_l2(j_g, j_o) <= 1e-5
    u_g, u_o = g.export(pkg.U), o.export(ob.U)
    assert scaled_block_rel(u_g, u_o).max() <= 1e-5
    assert_per_class(g.export(pkg.G)[:9 * s.num_cameras], o.export(ob.G)[:9 * s.num_cameras], 1e-4, "g_c")
    if eps > 0:   # the guard changes the model: the residuals differ from the unguarded ones by ~eps/depth
        o0 = oracle.OracleBA.from_scene(s, camera_model=1)
        o0.linearize()
        assert rel_l2(o0.export(ob.RESIDUALS), r_o) > 1e-6
    g.close()
    o.close()


@pytest.mark.parametrize("key", ["tiny", "small", "large"])
def test_pose3_lm_schedule_parity(scene_cache, key):
    """The oracle's adaptive run with the Pose3 camera, replayed on the GPU: cost at every step to 1e-4, and the
    cameras after every significant step (accepted steps RETRACT the rotation: w <- Log(Exp(w) Exp(d_w)))."""
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    eps = 1e-6
    o = oracle.OracleBA.from_scene(s, camera_model=1, depth_epsilon=eps)
    ref = o.solve(s.lm_iterations, 1e-2, 1e-10, s.pcg_max_iter)
    o.close()
    o = oracle.OracleBA.from_scene(s, camera_model=1, depth_epsilon=eps)   # the same run again, step by step
    g = pkg.CasparBA.from_scene(s, camera_model=1, depth_epsilon=eps)
    resolved = True
    for t, st in enumerate(ref):
        mode = 1 if st.accepted else 2
        got = g.lm_step(float(np.float32(st.lam)), 1e-10, s.pcg_max_iter, accept_mode=mode)
        o.lm_step(st.lam, 1e-10, s.pcg_max_iter, accept_mode=mode)
        assert abs(got.cost_before - st.cost_before) <= 1e-4 * st.cost_before, t
        assert abs(got.cost_after - st.cost_after) <= 1e-4 * st.cost_after, t
        resolved &= st.pcg_rel_residual <= 1e-2
        # C16: 1e-4 per class after every significant step; the converged tail only drifts along the gauge
        if resolved and significant_step(st):
            assert_cameras_match(g.cameras, o.cameras, 1e-4, ("cameras after step", t))
    if resolved:
        assert_cameras_match(g.cameras, o.cameras, TAIL_CAMERA_TOL, "final cameras")
    g.close()
    o.close()


def test_pose3_step_is_a_retraction(scene_cache):
    s = scene_cache("tiny")
    g = pkg.CasparBA.from_scene(s, camera_model=1)
    before = g.cameras.cpu().numpy().astype(np.float64)
    g.lm_step(LAM, 0.0, 20, accept_mode=1)
    d = g.export(pkg.DELTA)[:9 * s.num_cameras].reshape(-1, 9)
    after = g.cameras.cpu().numpy().astype(np.float64)
    want = np.stack([oracle.retract_camera(1, before[j], d[j]) for j in range(s.num_cameras)])
    assert np.abs(after - want).max() <= 2e-7 * np.abs(want).max()         # fp32 storage of the result
    assert np.abs(after[:, :3] - (before + d)[:, :3]).max() > 1e-6         # ... and it is not the additive update
    g.close()


# ------------------------------------------------------------------ N4: Schur-Jacobi preconditioner
@pytest.mark.parametrize("key", list(SCENES))
def test_schur_jacobi_preconditioner_parity(scene_cache, key):
    """The blocks (diagonal 9x9 blocks of S) against the oracle's, scaled per parameter class; the PCG step at equal
    iteration counts per class; and the number of iterations to the config's tolerance against the oracle's."""
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    g = pkg.CasparBA.from_scene(s)
    o = oracle.OracleBA.from_scene(s)
    g.linearize()
    o.linearize()
    g.set_preconditioner(1)
    o.set_preconditioner(1)
    nc9 = 9 * s.num_cameras
    ig, io = g.pcg_solve(LAM, 0.0, 30), o.pcg_solve(LAM, 0.0, 30)
    assert ig.iterations == io.iterations == 30
    blk_g, blk_o = g.export(pkg.PRECONDITIONER), o.preconditioner_blocks()
    assert scaled_block_rel(blk_g, blk_o).max() <= 1e-4               # a cancelling fp32 term per observation (I - B)
    d_g, d_o = g.export(pkg.DELTA), o.export(ob.DELTA)
    assert_per_class(d_g[:nc9], d_o[:nc9], 1e-4, "delta_c, 30 iterations")
    assert rel_l2(d_g[nc9:], d_o[nc9:]) <= 1e-4
    # At lambda = 1e-4 the weights I - B_i of two-view points are ~1e-4 and carry the rounding of the fp32 V'^-1
    # (relative 1e-3): the blocks still agree to 1e-4 after scaling.  (The STEP is not compared there: at that
    # damping the fp32 and fp64 solutions of the linear system themselves differ by ~6e-4 in the rotation and
    # translation classes on the ring scenes, whatever the preconditioner: conditioning of S, N4.)
    lam = float(np.float32(1e-4))
    g.pcg_solve(lam, 0.0, 5)
    o.pcg_solve(lam, 0.0, 5)
    assert scaled_block_rel(g.export(pkg.PRECONDITIONER), o.preconditioner_blocks()).max() <= 1e-4
    ig, io = g.pcg_solve(LAM, s.pcg_rel_tol, 300), o.pcg_solve(LAM, s.pcg_rel_tol, 300)
    assert ig.converged and io.converged and abs(ig.iterations - io.iterations) <= 2
    # switching back restores the U' blocks (C9)
    g.set_preconditioner(0)
    o.set_preconditioner(0)
    g.pcg_solve(LAM, 0.0, 5)
    o.pcg_solve(LAM, 0.0, 5)
    assert scaled_block_rel(g.export(pkg.PRECONDITIONER), o.preconditioner_blocks()).max() <= 1e-5
    g.close()
    o.close()


# ------------------------------------------------------------------ N1: full-system PCGNR, no Schur
@pytest.mark.parametrize("key", list(SCENES))
def test_pcgnr_step_parity(scene_cache, key):
    """PCG with normal residual on the full camera + point system.  The step after 30 passes
    over the Jacobians (tol 0: equal counts) per parameter class, the recursive residual, and -- run to
    convergence -- the same solution as the Schur path (the exact solutions coincide)."""
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    g = pkg.CasparBA.from_scene(s)
    o = oracle.OracleBA.from_scene(s)
    g.linearize()
    o.linearize()
    nc9 = 9 * s.num_cameras
    ig, io = g.pcgnr_solve(LAM, 0.0, 30), o.pcgnr_solve(LAM, 0.0, 30)
    assert ig.iterations == io.iterations == 30
    d_g, d_o = g.export(pkg.DELTA), o.export(ob.DELTA)
    assert_per_class(d_g[:nc9], d_o[:nc9], 1e-4, "PCGNR delta_c")
    assert rel_l2(d_g[nc9:], d_o[nc9:]) <= 1e-4
    assert abs(ig.rel_residual - io.rel_residual) <= 1e-3 * io.rel_residual + 1e-9
    assert abs(ig.rz0 - io.rz0) <= 1e-5 * io.rz0
    if key in ("tiny", "small"):
        info = g.pcgnr_solve(LAM, 1e-7, 2000)
        assert info.converged
        full = g.export(pkg.DELTA)
        g.pcg_solve(LAM, 1e-8, 500)
        schur = g.export(pkg.DELTA)
        assert rel_l2(full[:nc9], schur[:nc9]) <= 1e-4 and rel_l2(full[nc9:], schur[nc9:]) <= 1e-4
    g.close()
    o.close()


@pytest.mark.parametrize("key", ["tiny", "small"])
def test_lm_step_with_pcgnr(scene_cache, key):
    """One LM step with the paper's linear solve: cost, model decrease (|J delta|^2 from one more pass over the
    Jacobians with delta as the direction) and gain ratio against the oracle's."""
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    g = pkg.CasparBA.from_scene(s)
    o = oracle.OracleBA.from_scene(s)
    g.set_linear_solver(1)
    o.set_linear_solver(1)
    sg, so = g.lm_step(LAM, 0.0, 40, accept_mode=1), o.lm_step(LAM, 0.0, 40, accept_mode=1)
    assert abs(sg.cost_after - so.cost_after) <= 1e-4 * so.cost_after
    assert abs(sg.model_decrease - so.model_decrease) <= 1e-3 * so.model_decrease
    assert abs(sg.rho - so.rho) <= 1e-3
    cams = g.cameras.cpu().numpy().astype(np.float64)
    assert max(per_class_rel_l2(cams, o.cameras).values()) <= 1e-4
    g.close()
    o.close()


# ------------------------------------------------------------------ N2: speculative trial linearization
@pytest.mark.parametrize("key", ["tiny", "small", "large"])   # (the shrunken skewed scene is chaotic even at 10 iterations)
@pytest.mark.parametrize("camera_model", [0, 1])
def test_fused_trial_linearization_matches_the_default_path(scene_cache, key, camera_model):
    """caspar_ba_set_fusion(1): S9 runs the FULL linearize kernel at the trial point into a second
    set of arrays and an accepted step swaps the sets instead of linearizing again.  The same kernel at the same
    point, so the two paths differ only by what two runs of ONE path differ by: the order of the fp64 REDs inside
    the Schur matvec (C14, ~1e-16 per solve).  A fixed schedule of forced accepts and rejects at lambda = 1e-2
    (rejected steps throw the speculative Jacobians away and solve again from the kept linearization): step records
    to 1e-6, parameters and the linearization left behind to 1e-4."""
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    decisions = [1, 1, 2, 1, 2, 2, 1, 1]
    runs = []
    for fusion in (0, 1):
        g = pkg.CasparBA.from_scene(s, camera_model=camera_model)
        g.set_fusion(fusion)
        # five PCG iterations, no tolerance: a long unconverged CG run amplifies the last-bit differences of the RED order
        # (two runs of the DEFAULT path differ by up to 2e-5 in the residuals after eight 10-iteration steps on "large")
        steps = [g.lm_step(LAM * 0.5 ** t, 0.0, 5, mode) for t, mode in enumerate(decisions)]
        stats = g.stats()
        if fusion == 0:      # the linearization the next step would start from
            g.linearize()
        arrays = [g.export(w) for w in (pkg.RESIDUALS, pkg.JC, pkg.JP, pkg.U, pkg.V, pkg.G)]
        runs.append((steps, g.cameras.cpu().numpy(), g.points.cpu().numpy(), arrays, stats))
        g.close()
    (s0, c0, p0, a0, st0), (s1, c1, p1, a1, st1) = runs
    for x, y, mode in zip(s0, s1, decisions):
        assert x.accepted == y.accepted == (mode == 1) and x.pcg_iterations == y.pcg_iterations
        assert x.cost_before == pytest.approx(y.cost_before, rel=1e-6)
        assert x.cost_after == pytest.approx(y.cost_after, rel=1e-6)
        if x.model_decrease > 1e-6 * x.cost_before:
            assert x.model_decrease == pytest.approx(y.model_decrease, rel=1e-4)
    assert np.abs(c0 - c1).max() <= 1e-4 * np.abs(c0).max() and np.abs(p0 - p1).max() <= 1e-4 * np.abs(p0).max()
    assert st0.speculative_hits == 0 and st0.speculative_misses == 0 and st0.arena2_bytes == 0
    assert st1.speculative_hits == decisions.count(1) and st1.speculative_misses == decisions.count(2)
    assert st1.arena2_bytes > 0
    for x, y in zip(a0, a1):  # the fused run already holds the linearization at the new point
        assert rel_l2(x, y) <= 1e-4


def test_fusion_survives_a_parameter_reset_and_the_graph_chunks(scene_cache):
    """After set_parameters_host the speculative linearization is stale and must not be used; the CUDA-graph PCG
    chunks hold the pointers of ONE set of Jacobians, so both sets need their own graph."""
    import torch
    s = scene_cache("small")
    g = pkg.CasparBA.from_scene(s)
    g.set_fusion(1)
    ref = pkg.CasparBA.from_scene(s)
    a = [g.lm_step(LAM, 1e-6, s.pcg_max_iter, 0) for _ in range(3)]       # three accepted steps: sets swap 3 times
    b = [ref.lm_step(LAM, 1e-6, s.pcg_max_iter, 0) for _ in range(3)]
    for x, y in zip(a, b):
        assert x.accepted and y.accepted and x.pcg_iterations == y.pcg_iterations
        assert x.cost_after == pytest.approx(y.cost_after, rel=1e-6)
    cam_h = torch.from_numpy(s.cameras.copy()).pin_memory()
    pts_h = torch.from_numpy(s.points.copy()).pin_memory()
    g.set_parameters_host(cam_h, pts_h)
    ref.set_parameters_host(cam_h, pts_h)
    x, y = g.lm_step(LAM, 1e-6, s.pcg_max_iter, 0), ref.lm_step(LAM, 1e-6, s.pcg_max_iter, 0)
    assert x.pcg_iterations == y.pcg_iterations
    assert x.cost_before == pytest.approx(y.cost_before, rel=1e-12) and x.cost_after == pytest.approx(y.cost_after, rel=1e-6)
    assert x.cost_before == pytest.approx(b[0].cost_before, rel=1e-12)
    g.close()
    ref.close()
