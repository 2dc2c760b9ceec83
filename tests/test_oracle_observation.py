"""Pins of the oracle's per-observation arithmetic (O1-O3) against things other than itself:
library rotations, a hand-worked example, closed-form special cases, finite differences."""
import json
import os

import numpy as np
import pytest
from scipy.linalg import expm
from scipy.spatial.transform import Rotation

import oracle
from oracle import binding as ob

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
ANGLES = [0.0, 1e-9, 1e-6, 1e-3, 0.0099, 0.0101, 0.1, 1.0, 2.0, 3.0, np.pi - 1e-3, np.pi]


def _skew(v):
    return np.array([[0.0, -v[2], v[1]], [v[2], 0.0, -v[0]], [-v[1], v[0], 0.0]])


def _axis(seed):
    a = np.random.default_rng(seed).normal(size=3)
    return a / np.linalg.norm(a)


# ------------------------------------------------------------------ rotation R(w)
@pytest.mark.parametrize("theta", ANGLES)
def test_rotation_matches_library_routines(theta):
    w = theta * _axis(1)
    R = oracle.rotation(w)
    assert np.abs(R - Rotation.from_rotvec(w).as_matrix()).max() < 5e-15
    assert np.abs(R - expm(_skew(w))).max() < 5e-15
    assert np.abs(R.T @ R - np.eye(3)).max() < 5e-15
    assert abs(np.linalg.det(R) - 1.0) < 5e-15


def test_rotation_closed_forms():
    # quarter turn about z: x -> y, y -> -x
    R = oracle.rotation([0.0, 0.0, np.pi / 2])
    assert np.abs(R - np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])).max() < 1e-15
    # theta -> 0: R X = X + w x X + O(theta^2)
    w = 1e-7 * _axis(2)
    X = np.array([0.3, -1.2, 2.0])
    assert np.abs(oracle.rotation(w) @ X - (X + np.cross(w, X))).max() < 1e-13


# ------------------------------------------------------------------ projection
def test_hand_worked_example():
    """tests/golden/pinhole_worked_example.json: values derived by hand from PAPER.md:194-203."""
    with open(os.path.join(GOLDEN, "pinhole_worked_example.json")) as fh:
        g = json.load(fh)
    r, jc, jp = oracle.observation(g["camera"], g["point"], g["pixel"])
    assert np.abs(r - np.array(g["residual"])).max() < 1e-12
    assert np.abs(jc - np.array(g["jc"])).max() < 1e-11
    assert np.abs(jp - np.array(g["jp"])).max() < 1e-11


def test_pinhole_special_case():
    # w = 0, k1 = k2 = 0: uv = -f (X + t)_xy / (X + t)_z
    rng = np.random.default_rng(3)
    for _ in range(20):
        t = rng.normal(size=3) + np.array([0.0, 0.0, -8.0])
        X = rng.uniform(-2, 2, size=3)
        f = rng.uniform(400, 600)
        m = rng.normal(size=2)
        r = oracle.observation(np.r_[0, 0, 0, t, f, 0, 0], X, m, jacobians=False)
        P = X + t
        assert np.abs(r - (-f * P[:2] / P[2] - m)).max() < 1e-12


def test_radial_polynomial_identity():
    # uv(k1, k2) / uv(0, 0) = 1 + k1 n + k2 n^2 with n = |p|^2, for a general rotation
    rng = np.random.default_rng(4)
    for _ in range(20):
        w = rng.normal(size=3)
        t = rng.normal(size=3)
        X = rng.uniform(-2, 2, size=3)
        P = Rotation.from_rotvec(w).apply(X) + t
        n = (P[0] ** 2 + P[1] ** 2) / P[2] ** 2
        k1, k2 = rng.normal(0, 0.1), rng.normal(0, 0.01)
        uv0 = oracle.observation(np.r_[w, t, 500.0, 0, 0], X, [0, 0], jacobians=False)
        uv = oracle.observation(np.r_[w, t, 500.0, k1, k2], X, [0, 0], jacobians=False)
        assert np.abs(uv - uv0 * (1 + k1 * n + k2 * n * n)).max() < 1e-10 * max(1.0, np.abs(uv).max())


def test_residual_is_projection_minus_measurement():
    cam = np.r_[0.2, -0.1, 0.3, 0.1, 0.2, -9.0, 450.0, 0.01, 1e-4]
    X = np.array([0.5, -0.4, 1.0])
    uv = oracle.observation(cam, X, [0.0, 0.0], jacobians=False)
    r = oracle.observation(cam, X, [3.0, -7.0], jacobians=False)
    assert np.abs(r - (uv - np.array([3.0, -7.0]))).max() < 1e-12


# ------------------------------------------------------------------ Jacobians
def _fd(cam, X, m):
    """Central differences, h = 1e-6 max(1, |x|), on the 12 scalars."""
    x0 = np.r_[cam, X]
    J = np.empty((2, 12))
    for k in range(12):
        h = 1e-6 * max(1.0, abs(x0[k]))
        xp, xm = x0.copy(), x0.copy()
        xp[k] += h
        xm[k] -= h
        J[:, k] = (oracle.observation(xp[:9], xp[9:], m, jacobians=False)
                   - oracle.observation(xm[:9], xm[9:], m, jacobians=False)) / (2 * h)
    return J[:, :9], J[:, 9:]


@pytest.mark.parametrize("theta", ANGLES)
def test_jacobians_match_finite_differences(theta):
    rng = np.random.default_rng(int(theta * 1e6) % 9973 + 5)
    for trial in range(4):
        w = theta * _axis(10 + trial)
        X = rng.uniform(-2, 2, size=3)
        # translation that puts the point at depth ~ -8 in the camera frame
        t = -Rotation.from_rotvec(w).apply(X) + np.array([rng.normal(), rng.normal(), -8.0 + rng.normal()])
        cam = np.r_[w, t, rng.uniform(400, 600), rng.normal(0, 1e-2), rng.normal(0, 1e-4)]
        m = rng.normal(size=2) * 50
        _, jc, jp = oracle.observation(cam, X, m)
        fc, fp = _fd(cam, X, m)
        scale = max(np.abs(fc).max(), np.abs(fp).max())
        assert np.abs(jc - fc).max() <= 2e-8 * scale, (theta, trial)
        assert np.abs(jp - fp).max() <= 2e-8 * scale, (theta, trial)


@pytest.mark.parametrize("theta", [1e-3, 0.1, 1.0, 3.0])
def test_rotation_block_matches_gallego_yezzi(theta):
    """d(RX)/dw = -R [X]x (w w^T + (R^T - I) [w]x) / theta^2  (Gallego & Yezzi 2015, eq. III.7),
    evaluated with scipy's R; the oracle exposes A d(RX)/dw (first 3 columns) and A (next 3)."""
    rng = np.random.default_rng(7)
    w = theta * _axis(20)
    X = rng.uniform(-2, 2, size=3)
    cam = np.r_[w, 0.1, -0.2, -9.0, 500.0, 0.01, 1e-4]
    _, jc, _ = oracle.observation(cam, X, [0.0, 0.0])
    R = Rotation.from_rotvec(w).as_matrix()
    G = -R @ _skew(X) @ (np.outer(w, w) + (R.T - np.eye(3)) @ _skew(w)) / theta ** 2
    want = jc[:, 3:6] @ G
    assert np.abs(jc[:, 0:3] - want).max() <= 1e-6 * np.abs(want).max() / max(theta, 1e-2)


def test_series_and_closed_form_agree_across_the_switch():
    """theta^2 = 1e-4 is the series/closed-form switch (reading C3): both sides must give the same J."""
    X = np.array([0.7, -1.1, 0.4])
    ax = _axis(30)
    lo = np.r_[np.sqrt(1e-4) * (1 - 1e-9) * ax, 0.0, 0.0, -9.0, 500.0, 0.01, 1e-4]
    hi = np.r_[np.sqrt(1e-4) * (1 + 1e-9) * ax, 0.0, 0.0, -9.0, 500.0, 0.01, 1e-4]
    _, jl, pl = oracle.observation(lo, X, [0, 0])
    _, jh, ph = oracle.observation(hi, X, [0, 0])
    assert np.abs(jl - jh).max() <= 1e-6 * np.abs(jl).max() * 1e-2
    assert np.abs(pl - ph).max() <= 1e-8 * np.abs(pl).max()


# ------------------------------------------------------------------ cost, gradient, robust loss
def _tiny_problem(scene_cache, **kw):
    s = scene_cache("tiny")
    return s, oracle.OracleBA.from_scene(s, **kw)


def test_cost_is_half_sum_of_squares(scene_cache):
    s, o = _tiny_problem(scene_cache)
    f = o.linearize()
    r = o.export(ob.RESIDUALS)
    assert abs(f - 0.5 * np.sum(r * r)) <= 1e-12 * f
    assert abs(o.cost() - f) <= 1e-12 * f


@pytest.mark.parametrize("robust", [0, 1])
def test_gradient_matches_finite_difference_of_cost(scene_cache, robust):
    """grad F = J~^T r~, also under the Cauchy reweighting (d/dx 1/2 rho(s) = rho'(s) J^T r)."""
    s = scene_cache("tiny")
    o = oracle.OracleBA.from_scene(s, robust_loss=robust, robust_scale=2.0)
    o.linearize()
    g = o.export(ob.G)
    rng = np.random.default_rng(8)
    cams0, pts0 = o.cameras.copy(), o.points.copy()
    for _ in range(5):
        v = rng.normal(size=g.shape)
        v[: 9 * o.nc] *= 1e-3                       # camera parameters are stiff
        h = 1e-5
        vals = []
        for sgn in (+1, -1):
            o.cameras[:] = cams0 + sgn * h * v[: 9 * o.nc].reshape(-1, 9)
            o.points[:] = pts0 + sgn * h * v[9 * o.nc:].reshape(-1, 3)
            vals.append(o.cost())
        o.cameras[:], o.points[:] = cams0, pts0
        fd = (vals[0] - vals[1]) / (2 * h)
        assert abs(fd - g @ v) <= 1e-6 * abs(fd) + 1e-6


def test_cauchy_limits_and_bounds(scene_cache):
    s = scene_cache("tiny")
    plain = oracle.OracleBA.from_scene(s, robust_loss=0)
    huge = oracle.OracleBA.from_scene(s, robust_loss=1, robust_scale=1e9)     # c -> infinity: no reweighting
    cauchy = oracle.OracleBA.from_scene(s, robust_loss=1, robust_scale=2.0)
    f0, f1, f2 = plain.linearize(), huge.linearize(), cauchy.linearize()
    assert abs(f0 - f1) <= 1e-9 * f0
    assert np.abs(plain.export(ob.JC) - huge.export(ob.JC)).max() <= 1e-9 * np.abs(plain.export(ob.JC)).max()
    assert np.abs(plain.export(ob.RESIDUALS) - huge.export(ob.RESIDUALS)).max() <= 1e-9
    assert f2 < f0                                                           # rho(s) <= s
    r, rt = plain.export(ob.RESIDUALS), cauchy.export(ob.RESIDUALS)
    s2 = np.sum(r * r, axis=1)
    w = np.sum(rt * rt, axis=1) / s2                                         # = rho'(s)
    assert (w > 0).all() and (w <= 1 + 1e-15).all()
    assert np.abs(w - 1.0 / (1.0 + s2 / 4.0)).max() < 1e-12                  # w = 1 / (1 + s / c^2), c = 2
    assert abs(f2 - 0.5 * np.sum(4.0 * np.log1p(s2 / 4.0))) <= 1e-12 * f2    # F = 1/2 sum c^2 log(1 + s/c^2)
    jc, jct = plain.export(ob.JC), cauchy.export(ob.JC)
    assert np.abs(jct - np.sqrt(w)[:, None, None] * jc).max() <= 1e-12 * np.abs(jc).max()
