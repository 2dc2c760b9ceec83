"""Pins of the oracle's normal equations, Schur operator, PCG and LM (O4-O7) against
explicitly assembled matrices (scipy.sparse / numpy dense), dense Cholesky, and invariants."""
import numpy as np
import pytest
import scipy.sparse as sp

import oracle
from oracle import binding as ob

LAM = 1e-2


def _assemble_J(o):
    """Explicit sparse Jacobian [2N, 9Nc + 3Np] from the exported per-observation blocks."""
    jc, jp = o.export(ob.JC), o.export(ob.JP)
    n, nc = o.n, o.nc
    rows_c = (2 * np.arange(n)[:, None, None] + np.arange(2)[None, :, None] + np.zeros((1, 1, 9), int)).ravel()
    cols_c = (9 * o.camera_index[:, None, None] + np.zeros((1, 2, 1), int) + np.arange(9)[None, None, :]).ravel()
    rows_p = (2 * np.arange(n)[:, None, None] + np.arange(2)[None, :, None] + np.zeros((1, 1, 3), int)).ravel()
    cols_p = (9 * nc + 3 * o.point_index[:, None, None] + np.zeros((1, 2, 1), int)
              + np.arange(3)[None, None, :]).ravel()
    J = sp.coo_matrix((np.r_[jc.ravel(), jp.ravel()], (np.r_[rows_c, rows_p], np.r_[cols_c, cols_p])),
                      shape=(2 * n, 9 * nc + 3 * o.np_)).tocsr()
    return J


@pytest.fixture(scope="module")
def tiny(scene_cache):
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s)
    o.linearize()
    J = _assemble_J(o)
    H = (J.T @ J).toarray()
    return s, o, J, H


# ------------------------------------------------------------------ O4 normal equations
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_blocks_and_gradient_match_assembled_JtJ(scene_cache, name):
    s = scene_cache(name)
    o = oracle.OracleBA.from_scene(s)
    o.linearize()
    J = _assemble_J(o)
    r = o.export(ob.RESIDUALS).ravel()
    g = J.T @ r
    assert np.abs(o.export(ob.G) - g).max() <= 1e-12 * np.abs(g).max()
    H = (J.T @ J).tocsr()
    U, V = o.export(ob.U), o.export(ob.V)
    for j in range(0, o.nc, max(1, o.nc // 8)):
        blk = H[9 * j:9 * j + 9, 9 * j:9 * j + 9].toarray()
        assert np.abs(U[j] - blk).max() <= 1e-12 * np.abs(blk).max()
    off = 9 * o.nc
    for k in range(0, o.np_, max(1, o.np_ // 50)):
        blk = H[off + 3 * k:off + 3 * k + 3, off + 3 * k:off + 3 * k + 3].toarray()
        assert np.abs(V[k] - blk).max() <= 1e-12 * np.abs(blk).max()
    D = o.export(ob.DAMPING)
    assert np.abs(D - np.maximum(H.diagonal(), 1e-6)).max() <= 1e-12 * D.max()
    x = np.random.default_rng(0).normal(size=g.shape)
    want = H @ x + LAM * D * x
    assert np.abs(o.full_matvec(LAM, x) - want).max() <= 1e-12 * np.abs(want).max()


def test_damping_mode_identity(scene_cache):
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s, damping_mode=1)
    o.linearize()
    assert np.array_equal(o.export(ob.DAMPING), np.ones(9 * o.nc + 3 * o.np_))


# ------------------------------------------------------------------ O5 Schur complement
def _dense_schur(o, H, lam):
    n = 9 * o.nc
    Hd = H + lam * np.diag(o.export(ob.DAMPING))
    Ud, W, Vd = Hd[:n, :n], Hd[:n, n:], Hd[n:, n:]
    S = Ud - W @ np.linalg.solve(Vd, W.T)
    return Hd, S


def test_schur_operator_matches_dense(tiny):
    s, o, J, H = tiny
    Hd, S = _dense_schur(o, H, LAM)
    assert np.abs(S - S.T).max() <= 1e-12 * np.abs(S).max()
    np.linalg.cholesky(0.5 * (S + S.T))                      # positive definite
    rng = np.random.default_rng(1)
    for _ in range(3):
        p = rng.normal(size=9 * o.nc)
        want = S @ p
        assert np.abs(o.schur_matvec(LAM, p) - want).max() <= 1e-12 * np.abs(want).max()


def test_schur_rhs_and_solution_match_dense_cholesky(tiny):
    """PCG to 1e-12 + back-substitution == dense Cholesky of the full damped (9Nc+3Np)^2 system."""
    s, o, J, H = tiny
    n = 9 * o.nc
    Hd, S = _dense_schur(o, H, LAM)
    g = o.export(ob.G)
    info = o.pcg_solve(LAM, 1e-12, 500)
    assert info.converged and info.iterations <= n          # finite termination (loosely)
    b = -g[:n] + Hd[:n, n:] @ np.linalg.solve(Hd[n:, n:], g[n:])
    assert np.abs(o.export(ob.SCHUR_RHS) - b).max() <= 1e-11 * np.abs(b).max()
    L = np.linalg.cholesky(Hd)
    want = -np.linalg.solve(L.T, np.linalg.solve(L, g))
    got = o.export(ob.DELTA)
    assert np.linalg.norm(got[:n] - want[:n]) <= 1e-8 * np.linalg.norm(want[:n])
    assert np.linalg.norm(got[n:] - want[n:]) <= 1e-8 * np.linalg.norm(want[n:])


def test_spd_inverse_against_numpy():
    rng = np.random.default_rng(2)
    for n in (3, 9):
        a = rng.normal(size=(n, n))
        a = a @ a.T + n * np.eye(n)
        rc, inv = oracle.spd_inverse(a)
        assert rc == 0 and np.abs(inv - np.linalg.inv(a)).max() <= 1e-12 * np.abs(inv).max()
    rc, _ = oracle.spd_inverse(np.array([[1.0, 2.0], [2.0, 1.0]]))      # indefinite
    assert rc != 0


# ------------------------------------------------------------------ O6 PCG invariants
def test_pcg_recursive_residual_and_energy_norm(tiny):
    s, o, J, H = tiny
    n = 9 * o.nc
    Hd, S = _dense_schur(o, H, LAM)
    o.pcg_solve(LAM, 0.0, 1)
    b = o.export(ob.SCHUR_RHS)
    x_star = np.linalg.solve(S, b)
    prev = np.inf
    for k in (1, 2, 5, 10, 20, 30):
        info = o.pcg_solve(LAM, 0.0, k)
        assert info.iterations == k and not info.converged
        x = o.export(ob.DELTA)[:n]
        true_res = np.linalg.norm(b - S @ x) / np.linalg.norm(b)
        assert abs(true_res - info.rel_residual) <= 1e-9 + 1e-6 * true_res     # recursive == recomputed
        e = x - x_star
        energy = float(e @ S @ e)
        assert energy < prev                                                   # CG minimises the S-norm error
        prev = energy


def test_pcg_first_iterate_is_preconditioned_steepest_descent(tiny):
    """k = 1: x1 = alpha M^-1 b with alpha = (b.z)/(z.S z), z = M^-1 b, M = blockdiag(U'_j) (reading C9)."""
    s, o, J, H = tiny
    n = 9 * o.nc
    Hd, S = _dense_schur(o, H, LAM)
    info = o.pcg_solve(LAM, 0.0, 1)
    b = o.export(ob.SCHUR_RHS)
    z = np.concatenate([np.linalg.solve(Hd[9 * j:9 * j + 9, 9 * j:9 * j + 9], b[9 * j:9 * j + 9])
                        for j in range(o.nc)])
    x1 = (b @ z) / (z @ S @ z) * z
    got = o.export(ob.DELTA)[:n]
    assert np.linalg.norm(got - x1) <= 1e-10 * np.linalg.norm(x1)
    assert abs(info.rz0 - b @ z) <= 1e-10 * abs(b @ z)


def test_pcg_stops_on_relative_residual(tiny):
    s, o, J, H = tiny
    info = o.pcg_solve(LAM, 1e-6, 50)
    assert info.converged and info.rel_residual <= 1e-6
    fewer = o.pcg_solve(LAM, 1e-3, 50)
    assert fewer.converged and fewer.iterations < info.iterations


# ------------------------------------------------------------------ O7 LM
def test_model_decrease_identity_with_exact_solve(scene_cache):
    """With an exact solve, -delta^T g - 1/2 |J delta|^2 = 1/2 delta^T (lambda D delta - g) (Madsen eq. 3.14)."""
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s)
    step = o.lm_step(LAM, 1e-13, 500, accept_mode=2)
    d, g, D = o.export(ob.DELTA), o.export(ob.G), o.export(ob.DAMPING)
    want = 0.5 * d @ (LAM * D * d - g)
    assert abs(step.model_decrease - want) <= 1e-8 * abs(want)
    assert not step.accepted and step.cost_after < step.cost_before


def test_large_lambda_limit_is_scaled_gradient_step(scene_cache):
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s)
    lam = 1e9
    o.lm_step(lam, 1e-13, 200, accept_mode=2)
    d, g, D = o.export(ob.DELTA), o.export(ob.G), o.export(ob.DAMPING)
    want = -g / (lam * D)
    assert np.linalg.norm(d - want) <= 1e-6 * np.linalg.norm(want)


def test_accept_modes(scene_cache):
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s)
    before = o.cameras.copy()
    st = o.lm_step(LAM, 1e-6, 50, accept_mode=2)             # dry run: parameters untouched
    assert not st.accepted and np.array_equal(o.cameras, before)
    st = o.lm_step(LAM, 1e-6, 50, accept_mode=1)             # forced accept
    assert st.accepted and not np.array_equal(o.cameras, before)
    assert abs(o.cost() - st.cost_after) <= 1e-12 * st.cost_after


@pytest.mark.parametrize("name", ["tiny", "small"])
def test_noise_free_scene_converges_to_zero_cost(scene_cache, name):
    s = scene_cache(name, noise_free=True)
    o = oracle.OracleBA.from_scene(s)
    steps = o.solve(s.lm_iterations, 1e-2, s.pcg_rel_tol, s.pcg_max_iter)
    f0 = steps[0].cost_before
    assert min(st.cost_after for st in steps) <= 1e-10 * f0
    cost = f0
    for st in steps:                                          # accepted steps never increase the cost
        assert abs(st.cost_before - cost) <= 1e-12 * max(cost, 1e-30)
        if st.accepted:
            assert st.cost_after < st.cost_before or st.cost_before < 1e-12 * f0
            cost = st.cost_after


def test_nielsen_damping_schedule(scene_cache):
    """lambda_{t+1} = lambda_t max(1/3, 1 - (2 rho - 1)^3) after an accepted step, lambda nu (nu doubling)
    after a rejected one (Madsen et al. 2004, Alg. 3.16); lambda_0 = 1e-2 (reading C6)."""
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s)
    steps = o.solve(10, 1e-2, 1e-6, 50)
    assert steps[0].lam == 1e-2
    nu = 2.0
    for a, b in zip(steps[:-1], steps[1:]):
        if a.accepted:
            assert abs(b.lam - a.lam * max(1 / 3, 1 - (2 * a.rho - 1) ** 3)) <= 1e-15 * b.lam
            nu = 2.0
        else:
            assert abs(b.lam - a.lam * nu) <= 1e-15 * b.lam
            nu *= 2
    replay = oracle.OracleBA.from_scene(s)                     # replaying (lambda_t, accepted_t) reproduces F_t
    for st in steps:
        rp = replay.lm_step(st.lam, 1e-6, 50, accept_mode=1 if st.accepted else 2)
        assert abs(rp.cost_after - st.cost_after) <= 1e-12 * st.cost_after    # (OpenMP cost reduction: ulp-level order)


# ------------------------------------------------------------------ degenerate inputs
def test_unobserved_nodes_get_zero_step(scene_cache):
    s = scene_cache("tiny")
    cams = np.vstack([s.cameras, s.cameras[:1]])              # camera 16: no observations
    pts = np.vstack([s.points, s.points[:2]])                 # points 1000, 1001: no observations
    o = oracle.OracleBA(cams, pts, s.observations, s.camera_index, s.point_index)
    base = oracle.OracleBA.from_scene(s)
    st, sb = o.lm_step(LAM, 1e-10, 200, 2), base.lm_step(LAM, 1e-10, 200, 2)
    d, db = o.export(ob.DELTA), base.export(ob.DELTA)
    assert np.all(d[9 * 16:9 * 17] == 0.0) and np.all(d[9 * 17 + 3000:] == 0.0)
    assert np.linalg.norm(d[:144] - db[:144]) <= 1e-9 * np.linalg.norm(db[:144])
    assert abs(st.cost_after - sb.cost_after) <= 1e-9 * sb.cost_after


def test_empty_and_invalid_problems():
    z2, z9, z3 = np.zeros((0, 2)), np.zeros((0, 9)), np.zeros((0, 3))
    zi = np.zeros(0, np.int32)
    o = oracle.OracleBA(np.zeros((2, 9)), np.zeros((3, 3)), z2, zi, zi)
    assert o.linearize() == 0.0
    info = o.pcg_solve(LAM, 1e-6, 10)
    assert info.iterations == 0 and info.converged
    assert np.all(o.export(ob.DELTA) == 0.0)
    o = oracle.OracleBA(z9, z3, z2, zi, zi)
    assert o.linearize() == 0.0
    with pytest.raises(ob.OracleError):                        # index out of range
        oracle.OracleBA(np.zeros((1, 9)), np.zeros((1, 3)), np.zeros((1, 2)), np.array([1], np.int32),
                        np.array([0], np.int32))
    with pytest.raises(ob.OracleError):                        # pcg before linearize
        oracle.OracleBA(np.zeros((1, 9)), np.zeros((1, 3)), z2, zi, zi).pcg_solve(LAM, 1e-6, 1)


def test_point_behind_nothing_guards_depth_zero():
    """Reading C7: P_z = 0 is not guarded -> non-finite cost -> ENUMERIC."""
    cam = np.r_[0, 0, 0, 0, 0, 0, 500.0, 0, 0][None, :]
    pt = np.array([[1.0, 1.0, 0.0]])
    o = oracle.OracleBA(cam, pt, np.zeros((1, 2)), np.array([0], np.int32), np.array([0], np.int32))
    with pytest.raises(ob.OracleError) as e:
        o.linearize()
    assert e.value.code == -4
