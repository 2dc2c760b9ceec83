"""GPU parity at BASELINE.json's FULL sizes against stored oracle results: configs[2] "mid" (5.0 M observations),
configs[3] "large" (28.8 M, the scene bench.py times) and configs[4] "skewed" (15.2 M, Cauchy loss, Zipf cameras: the
HOT instantiation of the pipelined Schur matvec), in the library's default launch configuration.

tests/golden/fullsize_<config>.npz was written by tests/golden/make_fullsize_golden.py, which calls ONLY `oracle/`
on the seeded scene of `ba_scenes/` (minutes of fp64 CPU work per config; nothing in it comes from the CUDA path).
Tolerances are north_star's (C12 / C13): blocks 1e-5, gradient / Schur right-hand side / Schur matvec /
PCG step 1e-4 in L2 -- taken PER PARAMETER CLASS (rotation, translation, f, k1, k2) as well as globally -- and the
cost after EVERY step of the config's own LM schedule (PCG cap 100, tol 1e-10: C16) to 1e-4, whether or not the
oracle's linear solve is resolved at that step (measured: <= 3e-7 on mid and large, <= 6e-5 on skewed, whose PCG
stalls at 0.1-3 |b| from step 10 on: DESIGN.md C17)."""
import hashlib
import json
import os

import numpy as np
import pytest

import paper_2605_30583_b200 as pkg
from parity_util import assert_per_class, per_class_rel_l2, rel_l2, scaled_block_rel

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
REPORT = os.path.join(os.path.dirname(GOLDEN), "..", "gpurun_out")

# DESIGN.md C17: the final cameras are compared where every linear solve of the schedule was resolved by the oracle
RESOLVED = 1e-2          # |r|/|b| <= 1e-2
COST_TOL = 1e-4          # north_star, every step of every config


def _sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


@pytest.fixture(scope="module", params=["mid", "large", "skewed"])
def full(request, scene_cache):
    import torch

    name = request.param
    path = os.path.join(GOLDEN, f"fullsize_{name}.npz")
    assert os.path.exists(path), f"{path} missing: run tests/golden/make_fullsize_golden.py {name}"
    gold = dict(np.load(path))
    s = scene_cache(name)
    # the scene must be the one the oracle saw
    assert list(gold["fp_counts"]) == [s.num_cameras, s.num_points, s.num_observations]
    from ba_scenes import FULL_OBSERVATIONS
    assert s.num_observations == FULL_OBSERVATIONS[name]
    assert str(gold["fp_sha_camera_index"]) == _sha(s.camera_index)
    assert str(gold["fp_sha_point_index"]) == _sha(s.point_index)
    sums = np.array([np.abs(s.cameras.astype(np.float64)).sum(), np.abs(s.points.astype(np.float64)).sum(),
                     np.abs(s.observations.astype(np.float64)).sum()])
    assert np.allclose(sums, gold["fp_sums"], rtol=1e-9, atol=0), (sums, gold["fp_sums"])
    g = pkg.CasparBA.from_scene(s)
    cost = g.linearize()
    report = {}
    yield dict(name=name, scene=s, gold=gold, gpu=g, cost=cost, torch=torch, report=report)
    g.close()
    try:
        os.makedirs(REPORT, exist_ok=True)
        with open(os.path.join(REPORT, f"golden_margins_{name}.json"), "w") as fh:
            json.dump(report, fh, indent=1)
    except OSError:
        pass


def test_launch_configuration(full):
    st = full["gpu"].stats()
    assert st.tile_slots == 256 and st.matvec_pipelined == 1 and st.linearize_pipelined == 1
    if full["name"] == "skewed":
        assert st.num_hot_cameras > 0          # the HOT instantiation of the pipelined matvec
    else:
        assert st.num_hot_cameras == 0


def test_linearize_against_the_golden(full):
    g, gold, s, torch = full["gpu"], full["gold"], full["scene"], full["torch"]
    nc9 = 9 * s.num_cameras
    assert abs(full["cost"] - gold["cost0"]) <= 1e-5 * gold["cost0"]
    grad = g.export_device(pkg.G)
    gc = grad[:nc9].cpu().numpy()
    rep = full["report"]
    rep["cost0"] = abs(full["cost"] - float(gold["cost0"])) / float(gold["cost0"])
    rep["gc"] = assert_per_class(gc, gold["gc"], 1e-4, "g_c")
    pt = torch.as_tensor(gold["pt_ids"], device=g.device)
    gp = grad[nc9:].reshape(-1, 3)[pt].cpu().numpy()
    rep["gp"] = rel_l2(gp, gold["gp"])
    assert rep["gp"] <= 1e-4
    del grad
    u_dev = g.export_device(pkg.U)
    diag = torch.diagonal(u_dev, dim1=1, dim2=2).reshape(-1).cpu().numpy()
    rep["Dc"] = assert_per_class(np.maximum(diag, 1e-6), gold["Dc"], 1e-5, "diag U")
    u = u_dev[torch.as_tensor(gold["cam_ids"], device=g.device)].cpu().numpy()
    del u_dev
    err = scaled_block_rel(u, gold["U_blocks"])
    rep["U_scaled_worst"] = float(err.max())
    assert err.max() <= 1e-5, float(err.max())
    v = g.export_device(pkg.V)[pt].cpu().numpy().reshape(-1, 9)
    assert np.array_equal(v[:, [1, 2, 5]], v[:, [3, 6, 7]])             # symmetric by construction
    v = v[:, [0, 1, 2, 4, 5, 8]]
    errv = np.linalg.norm(v - gold["V_upper"], axis=1) / np.linalg.norm(gold["V_upper"], axis=1)
    rep["V_worst_block"] = float(errv.max())
    rep["V"] = rel_l2(v, gold["V_upper"])
    assert rep["V"] <= 1e-5 and errv.max() <= 1e-4   # per block: short fp32 sums of <= 200 terms


def test_linearize_repeats_bit_for_bit_at_full_size(full):
    """Stress repeat of S2+S3 in the bench launch configuration: the cost (an fp64 sum in a fixed order over every
    observation) must come back with the same BITS on every call.  This is the test that catches a stage of the TMA
    ring being refilled while a lagging warp still reads it: before the proxy fence in linearize_pipelined_kernel
    22 of 400 calls on the skewed scene had one warp of wrong residuals, i.e. a miss probability of
    < 0.5 % at 100 calls."""
    g, torch = full["gpu"], full["torch"]
    calls = 100 if full["name"] == "skewed" else 40
    ref = g.export_device(pkg.RESIDUALS).clone()
    costs = {g.linearize() for _ in range(calls)}
    assert costs == {full["cost"]}, sorted(costs)
    assert torch.equal(g.export_device(pkg.RESIDUALS), ref)
    q0 = g.schur_matvec(float(full["gold"]["lam1"]), full["gold"]["p1"].astype(np.float64))
    worst = 0.0
    for _ in range(calls):            # q = S p: the order of the fp64 REDs is free (C14), a wrong warp is not
        q = g.schur_matvec(float(full["gold"]["lam1"]), full["gold"]["p1"].astype(np.float64))
        worst = max(worst, rel_l2(q, q0))
    full["report"]["matvec_repeat_worst"] = worst
    assert worst <= 1e-12, worst


def test_schur_matvec_against_the_golden(full):
    g, gold = full["gpu"], full["gold"]
    for tag in ("1", "2"):
        lam = float(gold["lam" + tag])
        p = gold["p" + tag].astype(np.float64)
        q = g.schur_matvec(lam, p)
        full["report"]["q" + tag] = assert_per_class(q, gold["q" + tag], 1e-4, f"S p (lambda {lam:g})")


def test_pcg_step_against_the_golden(full):
    g, gold, s, torch = full["gpu"], full["gold"], full["scene"], full["torch"]
    nc9 = 9 * s.num_cameras
    info = g.pcg_solve(float(gold["lam1"]), 0.0, 30)
    assert info.iterations == 30
    rep = full["report"]
    rep["b"] = assert_per_class(g.export_device(pkg.SCHUR_RHS).cpu().numpy(), gold["b"], 1e-4, "Schur rhs")
    d = g.export_device(pkg.DELTA)
    rep["delta_c"] = assert_per_class(d[:nc9].cpu().numpy(), gold["delta_c"], 1e-4, "delta_c")
    pt = torch.as_tensor(gold["pt_ids"], device=g.device)
    rep["delta_p"] = rel_l2(d[nc9:].reshape(-1, 3)[pt].cpu().numpy(), gold["delta_p"])
    assert rep["delta_p"] <= 1e-4
    res_o = float(gold["pcg30_rel_residual"])
    rep["pcg30_rel_residual"] = [info.rel_residual, res_o]
    assert abs(info.rel_residual - res_o) <= 1e-2 * res_o


def test_lm_schedule_against_the_golden(full):
    """Replay the oracle's own adaptive (lambda_t, accepted_t) sequence at the config's cap (100) on a fresh handle."""
    s, gold, torch = full["scene"], full["gold"], full["torch"]
    name = full["name"]
    g = pkg.CasparBA.from_scene(s)
    cap, tol = int(gold["sched_cap"]), float(gold["sched_tol"])
    rows, resolved_all = [], True
    try:
        for t in range(len(gold["sched_lambda"])):
            lam = float(np.float32(gold["sched_lambda"][t]))
            acc = bool(gold["sched_accepted"][t])
            got = g.lm_step(lam, tol, cap, accept_mode=1 if acc else 2)
            fb, fa = float(gold["sched_cost_before"][t]), float(gold["sched_cost_after"][t])
            res_o = float(gold["sched_pcg_rel_residual"][t])
            eb, ea = abs(got.cost_before - fb) / fb, abs(got.cost_after - fa) / fa
            rows.append(dict(t=t, lam=lam, accepted=acc, oracle_pcg_iters=int(gold["sched_pcg_iterations"][t]),
                             gpu_pcg_iters=got.pcg_iterations, oracle_pcg_res=res_o, gpu_pcg_res=got.pcg_rel_residual,
                             cost_before_err=eb, cost_after_err=ea, rho_gpu=got.rho, rho_oracle=float(gold["sched_rho"][t])))
            resolved = res_o <= RESOLVED
            resolved_all &= resolved
            assert eb <= COST_TOL and ea <= COST_TOL, rows[-1]
    finally:
        full["report"]["schedule"] = rows
    cams = g.cameras.cpu().numpy().astype(np.float64)
    errs = per_class_rel_l2(cams, gold["final_cameras"])
    full["report"]["final_cameras"] = errs
    full["report"]["all_solves_resolved"] = bool(resolved_all)
    if resolved_all:      # otherwise the end point of 20 unconverged solves is not unique to 1e-4 (recorded only)
        assert max(errs.values()) <= 1e-4, errs
    g.close()
