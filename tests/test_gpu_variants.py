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
from parity_util import assert_per_class, per_class_rel_l2, rel_l2, scaled_block_rel

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
    cameras after the run (accepted steps RETRACT the rotation: w <- Log(Exp(w) Exp(d_w)))."""
    name, kw = SCENES[key]
    s = scene_cache(name, **kw)
    eps = 1e-6
    o = oracle.OracleBA.from_scene(s, camera_model=1, depth_epsilon=eps)
    ref = o.solve(s.lm_iterations, 1e-2, 1e-10, s.pcg_max_iter)
    g = pkg.CasparBA.from_scene(s, camera_model=1, depth_epsilon=eps)
    for t, st in enumerate(ref):
        got = g.lm_step(float(np.float32(st.lam)), 1e-10, s.pcg_max_iter, accept_mode=1 if st.accepted else 2)
        assert abs(got.cost_before - st.cost_before) <= 1e-4 * st.cost_before, t
        assert abs(got.cost_after - st.cost_after) <= 1e-4 * st.cost_after, t
    cams = g.cameras.cpu().numpy().astype(np.float64)
    assert max(per_class_rel_l2(cams, o.cameras).values()) <= 1e-4
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
