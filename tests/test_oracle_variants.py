"""Pins of the oracle's remaining branches and of the paper's own variants, each against something
other than the oracle itself:

  C15 breakdown branch           an operator made indefinite by construction (negative lambda I), checked on the dense S
  damping_mode = 1               the dense Schur complement with lambda I
  N1 full-system PCGNR           dense Cholesky of the 3,144^2 damped system; the first iterate in closed form
  N3 Pose3 tangent + d_safe      central differences THROUGH the retraction; scipy's rotation composition;
                                 the d_safe formula of PAPER.md:196-198 by hand
  N4 Schur-Jacobi preconditioner the diagonal 9x9 blocks of the dense 144x144 Schur complement
"""
import numpy as np
import pytest
import scipy.sparse as sp
from scipy.spatial.transform import Rotation

import oracle
from oracle import binding as ob

LAM = 1e-2


def _dense_normal_matrix(o):
    jc, jp = o.export(ob.JC), o.export(ob.JP)
    n, nc = o.n, o.nc
    rows_c = (2 * np.arange(n)[:, None, None] + np.arange(2)[None, :, None] + np.zeros((1, 1, 9), int)).ravel()
    cols_c = (9 * o.camera_index[:, None, None] + np.zeros((1, 2, 1), int) + np.arange(9)[None, None, :]).ravel()
    rows_p = (2 * np.arange(n)[:, None, None] + np.arange(2)[None, :, None] + np.zeros((1, 1, 3), int)).ravel()
    cols_p = (9 * nc + 3 * o.point_index[:, None, None] + np.zeros((1, 2, 1), int)
              + np.arange(3)[None, None, :]).ravel()
    J = sp.coo_matrix((np.r_[jc.ravel(), jp.ravel()], (np.r_[rows_c, rows_p], np.r_[cols_c, cols_p])),
                      shape=(2 * n, 9 * nc + 3 * o.np_)).tocsr()
    return J, (J.T @ J).toarray()


def _dense_schur(o, H, lam):
    n = 9 * o.nc
    Hd = H + lam * np.diag(o.export(ob.DAMPING))
    S = Hd[:n, :n] - Hd[:n, n:] @ np.linalg.solve(Hd[n:, n:], Hd[:n, n:].T)
    return Hd, S


@pytest.fixture(scope="module")
def tiny(scene_cache):
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s)
    o.linearize()
    J, H = _dense_normal_matrix(o)
    return s, o, J, H


# ------------------------------------------------------------------ C15: breakdown branch
def test_pcg_reports_breakdown_when_the_operator_is_not_positive(scene_cache):
    """For lambda >= 0 the Schur complement is positive definite and p.Sp <= 0 cannot happen, so the C15 branch is
    pinned with an operator that is indefinite BY CONSTRUCTION: lambda I damping (damping_mode = 1) with
    lambda = -0.05.  Every U'_j and V'_k stays positive definite (their smallest eigenvalues are 0.087 and 380 on
    this scene, checked below on the dense matrix), but S(-0.05) has negative eigenvalues beyond the seven gauge
    directions of bundle adjustment (S(0) has its first non-gauge eigenvalue at 0.037), along which b is not zero:
    CG must meet p.Sp <= 0, return ENUMERIC and keep the last good iterate."""
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s, damping_mode=1)
    o.linearize()
    J, H = _dense_normal_matrix(o)
    lam = -0.05
    Hd, S = _dense_schur(o, H, lam)
    n = 9 * o.nc
    assert min(np.linalg.eigvalsh(Hd[9 * j:9 * j + 9, 9 * j:9 * j + 9]).min() for j in range(o.nc)) > 0
    assert min(np.linalg.eigvalsh(Hd[n + 3 * k:n + 3 * k + 3, n + 3 * k:n + 3 * k + 3]).min() for k in range(o.np_)) > 0
    ev, evec = np.linalg.eigh(0.5 * (S + S.T))
    assert (ev < 0).sum() >= 8                                # more than the 7 gauge directions
    with pytest.raises(ob.OracleError) as e:
        o.pcg_solve(lam, 0.0, 400)
    assert e.value.code == -4
    x = o.export(ob.DELTA)[:n]                                # the last good iterate
    b = o.export(ob.SCHUR_RHS)
    g = o.export(ob.G)
    want_b = -g[:n] + Hd[:n, n:] @ np.linalg.solve(Hd[n:, n:], g[n:])
    assert np.abs(b - want_b).max() <= 1e-11 * np.abs(want_b).max()
    assert np.abs(evec[:, :8].T @ b).max() > 1e-8 * np.linalg.norm(b)     # b does see a negative direction (rounding: 1e-16)
    assert np.isfinite(x).all()
    # every accepted CG step lowered the quadratic model phi(x) = 1/2 x.Sx - b.x, so phi(x_last) <= phi(0) = 0
    assert 0.5 * x @ S @ x - b @ x <= 0.0
    # a block that is not positive definite is caught before PCG starts (same code, other message)
    o2 = oracle.OracleBA.from_scene(s)
    o2.linearize()
    with pytest.raises(ob.OracleError) as e:
        o2.pcg_solve(-2.0, 1e-6, 10)
    assert e.value.code == -4


# ------------------------------------------------------------------ damping_mode = 1 through the dense operator
def test_schur_operator_matches_dense_with_identity_damping(scene_cache):
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s, damping_mode=1)
    o.linearize()
    J, H = _dense_normal_matrix(o)
    n = 9 * o.nc
    for lam in (1e-2, 3.0):
        Hd = H + lam * np.eye(H.shape[0])                    # lambda I, written without the oracle's D export
        S = Hd[:n, :n] - Hd[:n, n:] @ np.linalg.solve(Hd[n:, n:], Hd[:n, n:].T)
        p = np.random.default_rng(4).normal(size=n)
        want = S @ p
        assert np.abs(o.schur_matvec(lam, p) - want).max() <= 1e-12 * np.abs(want).max()
        info = o.pcg_solve(lam, 1e-13, 2000)
        assert info.converged
        want_d = -np.linalg.solve(Hd, o.export(ob.G))
        got = o.export(ob.DELTA)
        assert np.linalg.norm(got - want_d) <= 1e-7 * np.linalg.norm(want_d)


# ------------------------------------------------------------------ N1: full-system PCGNR
def test_pcgnr_converges_to_the_dense_solution(tiny):
    s, o, J, H = tiny
    Hd = H + LAM * np.diag(o.export(ob.DAMPING))
    g = o.export(ob.G)
    want = -np.linalg.solve(Hd, g)
    info = o.pcgnr_solve(LAM, 1e-13, 5000)
    assert info.converged
    got = o.export(ob.DELTA)
    n = 9 * o.nc
    assert np.linalg.norm(got[:n] - want[:n]) <= 1e-8 * np.linalg.norm(want[:n])
    assert np.linalg.norm(got[n:] - want[n:]) <= 1e-8 * np.linalg.norm(want[n:])
    # ... which is also what the Schur path converges to (exact solutions coincide)
    o.pcg_solve(LAM, 1e-13, 500)
    schur = o.export(ob.DELTA)
    assert np.linalg.norm(schur - got) <= 1e-8 * np.linalg.norm(got)


def test_pcgnr_first_iterate_and_invariants(tiny):
    """k = 1: x1 = alpha z, z = M^-1 (-g), M = blockdiag(U'_j, V'_k) (one block per node), alpha = (r.z)/(z.A z);
    the recursive residual equals -g - A x_k; the A-norm error decreases monotonically."""
    s, o, J, H = tiny
    Hd = H + LAM * np.diag(o.export(ob.DAMPING))
    g = o.export(ob.G)
    n, N = 9 * o.nc, H.shape[0]
    z = np.zeros(N)
    for j in range(o.nc):
        z[9 * j:9 * j + 9] = np.linalg.solve(Hd[9 * j:9 * j + 9, 9 * j:9 * j + 9], -g[9 * j:9 * j + 9])
    for k in range(o.np_):
        a = n + 3 * k
        z[a:a + 3] = np.linalg.solve(Hd[a:a + 3, a:a + 3], -g[a:a + 3])
    x1 = (-g @ z) / (z @ Hd @ z) * z
    info = o.pcgnr_solve(LAM, 0.0, 1)
    assert info.iterations == 1
    got = o.export(ob.DELTA)
    assert np.linalg.norm(got - x1) <= 1e-10 * np.linalg.norm(x1)
    assert abs(info.rz0 - (-g @ z)) <= 1e-10 * abs(g @ z)
    x_star = -np.linalg.solve(Hd, g)
    prev = np.inf
    for k in (1, 2, 5, 10, 20, 40):
        info = o.pcgnr_solve(LAM, 0.0, k)
        x = o.export(ob.DELTA)
        true_res = np.linalg.norm(-g - Hd @ x) / np.linalg.norm(g)
        assert abs(true_res - info.rel_residual) <= 1e-9 + 1e-6 * true_res
        e = x - x_star
        energy = float(e @ Hd @ e)
        assert energy < prev
        prev = energy


def test_lm_step_with_pcgnr_matches_the_schur_step_when_both_converge(scene_cache):
    s = scene_cache("tiny")
    a, b = oracle.OracleBA.from_scene(s), oracle.OracleBA.from_scene(s)
    b.set_linear_solver(1)
    sa = a.lm_step(LAM, 1e-13, 500, accept_mode=1)
    sb = b.lm_step(LAM, 1e-13, 5000, accept_mode=1)
    assert abs(sa.cost_after - sb.cost_after) <= 1e-9 * sa.cost_after
    assert abs(sa.model_decrease - sb.model_decrease) <= 1e-7 * sa.model_decrease
    assert np.abs(a.cameras - b.cameras).max() <= 1e-8 * np.abs(a.cameras).max()


# ------------------------------------------------------------------ N4: Schur-Jacobi preconditioner
def test_schur_jacobi_blocks_are_the_diagonal_blocks_of_the_dense_schur_complement(tiny):
    s, o, J, H = tiny
    for lam in (LAM, 1e-4):
        Hd, S = _dense_schur(o, H, lam)
        o.set_preconditioner(1)
        o.schur_matvec(lam, np.zeros(9 * o.nc))              # prepares the damped blocks at this lambda
        blocks = o.preconditioner_blocks()
        for j in range(o.nc):
            want = S[9 * j:9 * j + 9, 9 * j:9 * j + 9]
            assert np.abs(blocks[j] - want).max() <= 1e-11 * np.abs(want).max(), j
        o.set_preconditioner(0)
        o.schur_matvec(lam, np.zeros(9 * o.nc))
        blocks = o.preconditioner_blocks()
        for j in range(o.nc):
            want = Hd[9 * j:9 * j + 9, 9 * j:9 * j + 9]
            assert np.abs(blocks[j] - want).max() <= 1e-12 * np.abs(want).max(), j


def test_pcg_with_the_schur_jacobi_preconditioner(tiny):
    """Same solution as the dense solve; first iterate = preconditioned steepest descent with M = blockdiag(S_jj);
    the iteration counts of the two preconditioners are of the same order (on this fully coupled 16-camera scene
    blockdiag(S_jj) needs 21 against 19; on the banded scenes it saves 5-25 %: DESIGN.md N4)."""
    s, o, J, H = tiny
    n = 9 * o.nc
    Hd, S = _dense_schur(o, H, LAM)
    g = o.export(ob.G)
    o.set_preconditioner(1)
    info = o.pcg_solve(LAM, 1e-12, 500)
    assert info.converged
    want = -np.linalg.solve(Hd, g)
    got = o.export(ob.DELTA)
    assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want)
    b = o.export(ob.SCHUR_RHS)
    o.pcg_solve(LAM, 0.0, 1)
    z = np.concatenate([np.linalg.solve(S[9 * j:9 * j + 9, 9 * j:9 * j + 9], b[9 * j:9 * j + 9])
                        for j in range(o.nc)])
    x1 = (b @ z) / (z @ S @ z) * z
    assert np.linalg.norm(o.export(ob.DELTA)[:n] - x1) <= 1e-10 * np.linalg.norm(x1)
    it_sj = o.pcg_solve(LAM, 1e-6, 500).iterations
    o.set_preconditioner(0)
    it_u = o.pcg_solve(LAM, 1e-6, 500).iterations
    assert abs(it_sj - it_u) <= 5, (it_sj, it_u)


# ------------------------------------------------------------------ N3: Pose3 tangent-space camera and d_safe
def test_retraction_is_scipys_rotation_composition():
    rng = np.random.default_rng(9)
    for theta in (0.0, 1e-9, 1e-4, 0.3, 2.0, 3.1):
        for dth in (0.0, 1e-10, 1e-3, 0.5):
            w = rng.normal(size=3)
            w *= theta / max(np.linalg.norm(w), 1e-300)
            d = rng.normal(size=9)
            d[:3] *= dth / np.linalg.norm(d[:3])
            cam = np.r_[w, rng.normal(size=6)]
            out = oracle.retract_camera(1, cam, d)
            want = (Rotation.from_rotvec(w) * Rotation.from_rotvec(d[:3])).as_matrix()
            got = Rotation.from_rotvec(out[:3]).as_matrix()
            assert np.abs(got - want).max() <= 1e-14
            assert np.linalg.norm(out[:3]) <= np.pi + 1e-12
            assert np.array_equal(out[3:], cam[3:] + d[3:])
            assert np.array_equal(oracle.retract_camera(0, cam, d), cam + d)


def _random_observation(rng, theta):
    w = rng.normal(size=3)
    w *= theta / max(np.linalg.norm(w), 1e-300)
    X = rng.uniform(-2, 2, size=3)
    R = Rotation.from_rotvec(w).as_matrix()
    t = np.array([0.3, -0.2, -10.0]) - R @ X + rng.normal(size=3) * 0.5     # depth around -10
    cam = np.r_[w, t, 500.0, 0.01, -1e-4]
    return cam, X, rng.normal(size=2) * 50


@pytest.mark.parametrize("theta", [0.0, 1e-6, 1e-3, 0.1, 1.0, 3.0])
@pytest.mark.parametrize("eps", [0.0, 1e-3])
def test_pose3_jacobian_is_the_derivative_through_the_retraction(theta, eps):
    """d r / d delta of r(cam (+) delta) at delta = 0 by central differences, all nine tangent directions."""
    rng = np.random.default_rng(int(theta * 1e6) + 1)
    cam, X, m = _random_observation(rng, theta)
    r0, jc, jp = oracle.observation_model(1, eps, cam, X, m)
    h = 1e-6
    for a in range(9):
        d = np.zeros(9)
        d[a] = h * max(1.0, abs(cam[a])) if a >= 3 else h
        rp = oracle.observation_model(1, eps, oracle.retract_camera(1, cam, d), X, m, jacobians=False)
        rm = oracle.observation_model(1, eps, oracle.retract_camera(1, cam, -d), X, m, jacobians=False)
        fd = (rp - rm) / (2 * d[a])
        assert np.abs(fd - jc[:, a]).max() <= 1e-7 * max(1.0, np.abs(jc[:, a]).max()), (a, fd, jc[:, a])
    for a in range(3):
        d = np.zeros(3)
        d[a] = h
        fd = (oracle.observation_model(1, eps, cam, X + d, m, jacobians=False)
              - oracle.observation_model(1, eps, cam, X - d, m, jacobians=False)) / (2 * h)
        assert np.abs(fd - jp[:, a]).max() <= 1e-7 * max(1.0, np.abs(jp[:, a]).max())
    # the tangent-space rotation block is -J_p [X]x (J_p = A R, d(R Exp(d) X)/dd = -R [X]x)
    Xx = np.array([[0, -X[2], X[1]], [X[2], 0, -X[0]], [-X[1], X[0], 0]])
    assert np.abs(jc[:, :3] + jp @ Xx).max() <= 1e-12 * np.abs(jc[:, :3]).max()
    # everything but the rotation block is the angle-axis model's
    _, jc0, jp0 = oracle.observation_model(0, eps, cam, X, m)
    assert np.array_equal(jc0[:, 3:], jc[:, 3:]) and np.array_equal(jp0, jp)


def test_depth_guard_is_the_papers_d_safe():
    """p = -P_xy / (d + eps sign_no_zero(d)), written out by hand; eps = 0 is the unguarded model;
    a point at depth exactly 0 stays finite with eps > 0."""
    cam = np.r_[0.0, 0.0, 0.0, 0.1, -0.2, 0.0, 500.0, 0.01, -1e-4]
    for X, eps in ((np.array([0.5, 0.4, -8.0]), 0.05), (np.array([0.5, 0.4, 8.0]), 0.05),
                   (np.array([0.5, 0.4, 0.0]), 0.05), (np.array([0.5, 0.4, -8.0]), 0.0)):
        P = X + cam[3:6]
        d_safe = P[2] + eps * (1.0 if P[2] >= 0 else -1.0)
        p = -P[:2] / d_safe
        n = p @ p
        want = 500.0 * (1 + 0.01 * n - 1e-4 * n * n) * p - np.array([3.0, 4.0])
        got = oracle.observation_model(0, eps, cam, X, np.array([3.0, 4.0]), jacobians=False)
        assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    assert np.array_equal(oracle.observation_model(0, 0.0, cam, X, np.zeros(2), jacobians=False),
                          oracle.observation(cam, X, np.zeros(2), jacobians=False))


def test_pose3_lm_reaches_the_same_minimum_on_a_noise_free_scene(scene_cache):
    """Two parametrisations of the same problem: on the noise-free twin both drive the cost to ~0, and an accepted
    Pose3 step moves the cameras by the retraction (not by adding delta to the angle-axis vector)."""
    s = scene_cache("tiny", noise_free=True)
    o = oracle.OracleBA.from_scene(s, camera_model=1, depth_epsilon=1e-6)
    before = o.cameras.copy()
    st = o.lm_step(LAM, 1e-10, 200, accept_mode=1)
    d = o.export(ob.DELTA)[:9 * o.nc].reshape(-1, 9)
    for j in range(o.nc):
        assert np.array_equal(o.cameras[j], oracle.retract_camera(1, before[j], d[j]))
    assert abs(o.cost() - st.cost_after) <= 1e-12 * max(st.cost_after, 1e-30)
    steps = o.solve(s.lm_iterations, 1e-2, s.pcg_rel_tol, s.pcg_max_iter)
    assert min(x.cost_after for x in steps) <= 1e-10 * st.cost_before
