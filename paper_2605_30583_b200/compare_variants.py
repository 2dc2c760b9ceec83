#!/usr/bin/env python
"""The paper's variants beside the default path, on one GPU:

    python -m paper_2605_30583_b200.compare_variants [tiny small mid large skewed] [--cap 400]

For every config, at the start point and lambda = 1e-2, with the config's tolerance: iterations and time to tolerance
of (a) the Schur PCG with the U' block-Jacobi preconditioner (default), (b) the same with the Schur-Jacobi
preconditioner (N4), (c) the full-system PCG with normal residual, no Schur (N1: the paper's own solve); then LM
iterations/s of the config's adaptive schedule with fusion off / on (N2).  Prints a markdown table.  Every number
comes from the library's kernels; the oracle is not involved."""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def nielsen(lam, nu, st):
    if st.accepted:
        c = 2.0 * st.rho - 1.0
        return lam * max(1.0 / 3.0, 1.0 - c * c * c), 2.0
    return lam * nu, 2.0 * nu


def timed(fn):
    import torch
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    out = fn()
    torch.cuda.synchronize()
    return out, (time.perf_counter() - t0) * 1e3


def main():
    import torch

    import paper_2605_30583_b200 as pkg
    from ba_scenes import CONFIGS, make_scene

    ap = argparse.ArgumentParser()
    ap.add_argument("workloads", nargs="*", default=["tiny", "small", "mid", "large", "skewed"])
    ap.add_argument("--cap", type=int, default=400, help="iteration cap of the solver comparison")
    args = ap.parse_args()
    lam = float(np.float32(1e-2))
    print("| config | Schur PCG, U' blocks: iterations (converged), ms | Schur PCG, Schur-Jacobi blocks | full-system PCGNR (no Schur) "
          "| LM it/s, fusion off | LM it/s, fusion on |")
    print("|---|---|---|---|---|---|")
    for name in args.workloads:
        s, cfg = make_scene(name), CONFIGS[name]
        tol = cfg["pcg_rel_tol"]
        g = pkg.CasparBA.from_scene(s)
        g.linearize()
        cells = []
        for what in ("schur", "schur_jacobi", "pcgnr"):
            g.set_preconditioner(1 if what == "schur_jacobi" else 0)
            solve = g.pcgnr_solve if what == "pcgnr" else g.pcg_solve
            try:
                solve(lam, tol, args.cap)                                 # warm-up (graphs, caches)
                info, ms = timed(lambda: solve(lam, tol, args.cap))
                cells.append(f"{info.iterations} ({'yes' if info.converged else 'no: ' + format(info.rel_residual, '.1e')}), {ms:.2f}")
            except pkg.CasparError as e:                                  # a breakdown is a result, not a crash
                cells.append(f"stopped: {e}")
        g.close()
        rates = []
        for fusion in (0, 1):
            g = pkg.CasparBA.from_scene(s)
            g.set_fusion(fusion)
            cam_h = torch.from_numpy(s.cameras.copy()).pin_memory()
            pts_h = torch.from_numpy(s.points.copy()).pin_memory()

            def run():
                lm, nu = 1e-2, 2.0
                for _ in range(cfg["lm_iterations"]):
                    st = g.lm_step(float(np.float32(lm)), tol, cfg["pcg_max_iter"], 0)
                    lm, nu = nielsen(lm, nu, st)

            run()
            g.set_parameters_host(cam_h, pts_h)
            _, ms = timed(run)
            rates.append(cfg["lm_iterations"] / (ms * 1e-3))
            g.close()
        print(f"| {name} ({s.num_observations} obs) | {cells[0]} | {cells[1]} | {cells[2]} | {rates[0]:.1f} | {rates[1]:.1f} |", flush=True)


if __name__ == "__main__":
    main()
