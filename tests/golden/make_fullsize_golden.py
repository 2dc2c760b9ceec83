#!/usr/bin/env python
"""Write the FULL-SIZE oracle goldens tests/golden/fullsize_<config>.npz (configs[2] mid, [3] large, [4] skewed).

    python tests/golden/make_fullsize_golden.py [mid large skewed]

Imports ONLY `oracle/` (the fp64 CPU oracle) and `ba_scenes/` (the seeded input generator): no value in these
files comes from the CUDA path.  The oracle needs minutes per config at these sizes (Large: 6 GB of fp64
Jacobians, ~2 s per Schur matvec on 8 threads, 1,000+ matvecs), which is why its results are stored instead of
recomputed inside `pytest -m gpu` (tests/test_gpu_golden.py compares the CUDA path with them).

What each file holds (all fp64 unless noted; PAPER.md:194-203 factor, :163-169 LM + PCG, through SURVEY.md
8(c) O1-O7 with DESIGN.md's readings):
  fingerprint of the scene (sha256 of the index arrays, sums of the float arrays) -- the test refuses a scene
      that is not the one the oracle saw;
  cost0                      F at the start point;
  gc, Dc                     camera gradient and diag(U) floored (the Marquardt scaling), full;
  cam_ids, U_blocks          U_j of sampled cameras (64 random + the 8 most observed);
  pt_ids, V_upper, gp        V_k (xx xy xz yy yz zz), g_p,k of 20,000 sampled points;
  p1 (fp32 values), q1       q = S p at lambda = 1e-2, p ~ N(0,1);
  p2 (fp32 values), q2       q = S p at lambda = 1e-4, p = N(0,1) / sqrt(Dc): a preconditioned direction;
  b, delta_c, delta_p        Schur right-hand side and the PCG step after 30 iterations at lambda = 1e-2, tol 0
                             (delta_p on pt_ids); pcg30_rel_residual;
  sched_*                    the oracle's adaptive LM run on the config's own schedule (lambda0 = 1e-2, the config's
                             iteration count and PCG cap, tol 1e-10 per DESIGN.md C16): lambda, accepted, cost before /
                             after, model decrease, rho, PCG iterations and final relative residual per step;
  final_cameras              cameras after that run, final_points on pt_ids.
"""
from __future__ import annotations

import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from ba_scenes import make_scene  # noqa: E402
from oracle import binding as ob  # noqa: E402

LAM1 = float(np.float32(1e-2))
LAM2 = float(np.float32(1e-4))
REPLAY_TOL = 1e-10          # DESIGN.md C16
SAMPLE_POINTS = 100_000    # drawn, of which every 5th is kept (20,000: the files stay a few MB)
POINT_STRIDE = 5
SAMPLE_CAMERAS = 64
TOP_CAMERAS = 8
SEED = 20260530


def fingerprint(scene) -> dict:
    """What identifies the scene: exact hashes of the integer structure, fp64 sums of the float arrays (a last-ulp
    difference of a libm routine between two hosts must not look like another scene; a different scene must)."""
    def sha(a):
        return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()
    return {
        "fp_counts": np.array([scene.num_cameras, scene.num_points, scene.num_observations], np.int64),
        "fp_sha_camera_index": sha(scene.camera_index),
        "fp_sha_point_index": sha(scene.point_index),
        "fp_sums": np.array([np.abs(scene.cameras.astype(np.float64)).sum(),
                             np.abs(scene.points.astype(np.float64)).sum(),
                             np.abs(scene.observations.astype(np.float64)).sum()]),
    }


def sample_ids(scene) -> tuple:
    rng = np.random.default_rng(SEED)
    per_cam = np.bincount(scene.camera_index, minlength=scene.num_cameras)
    top = np.argsort(-per_cam, kind="stable")[:TOP_CAMERAS]
    cams = np.unique(np.concatenate([rng.choice(scene.num_cameras, min(SAMPLE_CAMERAS, scene.num_cameras),
                                                replace=False), top]))
    pts = np.sort(rng.choice(scene.num_points, min(SAMPLE_POINTS, scene.num_points), replace=False))[::POINT_STRIDE]
    return cams.astype(np.int64), pts.astype(np.int64)


def directions(scene, dc: np.ndarray) -> tuple:
    rng = np.random.default_rng(SEED + 1)
    n = 9 * scene.num_cameras
    p1 = rng.normal(size=n).astype(np.float32)
    p2 = (rng.normal(size=n) / np.sqrt(dc)).astype(np.float32)
    return p1, p2


def make(name: str) -> str:
    t0 = time.time()

    def log(msg):
        print(f"[{name} {time.time() - t0:7.1f}s] {msg}", flush=True)

    scene = make_scene(name)
    log(f"scene: {scene.num_cameras} cameras, {scene.num_points} points, {scene.num_observations} observations")
    out = dict(fingerprint(scene))
    o = oracle.OracleBA.from_scene(scene)
    nc9 = 9 * scene.num_cameras
    out["cost0"] = np.float64(o.linearize())
    log(f"linearized, cost0 = {out['cost0']:.9g}")

    cam_ids, pt_ids = sample_ids(scene)
    out["cam_ids"], out["pt_ids"] = cam_ids, pt_ids
    g = o.export(ob.G)
    out["gc"] = g[:nc9].copy()
    out["gp"] = g[nc9:].reshape(-1, 3)[pt_ids].copy()
    del g
    out["Dc"] = o.export(ob.DAMPING)[:nc9].copy()
    out["U_blocks"] = o.export(ob.U)[cam_ids].copy()
    out["V_upper"] = o.export(ob.V)[pt_ids].reshape(-1, 9)[:, [0, 1, 2, 4, 5, 8]].copy()

    p1, p2 = directions(scene, out["Dc"])
    out["p1"], out["p2"] = p1, p2
    out["lam1"], out["lam2"] = np.float64(LAM1), np.float64(LAM2)
    out["q1"] = o.schur_matvec(LAM1, p1.astype(np.float64))
    out["q2"] = o.schur_matvec(LAM2, p2.astype(np.float64))
    log("Schur matvecs done")

    info = o.pcg_solve(LAM1, 0.0, 30)
    assert info.iterations == 30
    out["pcg30_rel_residual"] = np.float64(info.rel_residual)
    out["b"] = o.export(ob.SCHUR_RHS)
    d = o.export(ob.DELTA)
    out["delta_c"] = d[:nc9].copy()
    out["delta_p"] = d[nc9:].reshape(-1, 3)[pt_ids].copy()
    del d
    log(f"30 PCG iterations done, residual {info.rel_residual:.3e}")

    steps = o.solve(scene.lm_iterations, 1e-2, REPLAY_TOL, scene.pcg_max_iter)
    out["sched_tol"] = np.float64(REPLAY_TOL)
    out["sched_cap"] = np.int64(scene.pcg_max_iter)
    out["sched_lambda"] = np.array([s.lam for s in steps])
    out["sched_accepted"] = np.array([s.accepted for s in steps], np.int8)
    out["sched_cost_before"] = np.array([s.cost_before for s in steps])
    out["sched_cost_after"] = np.array([s.cost_after for s in steps])
    out["sched_model_decrease"] = np.array([s.model_decrease for s in steps])
    out["sched_rho"] = np.array([s.rho for s in steps])
    out["sched_pcg_iterations"] = np.array([s.pcg_iterations for s in steps], np.int32)
    out["sched_pcg_rel_residual"] = np.array([s.pcg_rel_residual for s in steps])
    out["final_cameras"] = o.cameras.copy()
    out["final_points"] = o.points[pt_ids].copy()
    for t, s in enumerate(steps):
        log(f"step {t:2d}: lambda {s.lam:.3e} accepted {int(s.accepted)} F {s.cost_before:.9g} -> {s.cost_after:.9g} "
            f"rho {s.rho:.4f} pcg {s.pcg_iterations} res {s.pcg_rel_residual:.2e}")
    o.close()

    path = os.path.join(HERE, f"fullsize_{name}.npz")
    np.savez_compressed(path, **out)
    log(f"wrote {path} ({os.path.getsize(path) / 1e6:.1f} MB), oracle threads {oracle.num_threads()}")
    return path


if __name__ == "__main__":
    for cfg in (sys.argv[1:] or ["mid", "large", "skewed"]):
        make(cfg)
