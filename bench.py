#!/usr/bin/env python
"""bench.py — LM iterations/s (and Schur matvecs/s, HBM roofline fraction) of the B200 bundle-adjustment path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload large]

A "step" is ONE Levenberg-Marquardt iteration of the whole hot path (S1-S10: linearize, block assembly,
Schur PCG with the config's cap / tolerance, back-substitution, trial cost, accept / reject) on the seeded
synthetic scene of BASELINE.json configs[3] ("large": 13,700 cameras, 4.5 M points, ~28.8 M observations),
the scene the north_star's roofline target is quoted on.  The timed K steps are the first K iterations of
the adaptive LM schedule from the perturbed start (lambda0 = 1e-2); the W warm-up steps run first and the
parameters are then reset.  One JSON line is printed by rank 0.

N > 1 (torchrun): the path is single-GPU (north_star); by default ranks run independent replicas of the config with
different seeds and no data-path collective ("scaling": "weak"); time = max over ranks.  `--parallelism sharded` runs
ONE problem instead, its points split over the ranks (caspar_ba_set_shard with NCCL all-reduce /
broadcast through torch.distributed): "scaling": "strong".  That mode has only ever run on one GPU (world size 1 and
two emulated ranks in tests/test_gpu_sharding.py): no multi-GPU box was available to this build.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

LAMBDA0 = 1e-2
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
# bounded oracle sample: same recipe as the workload, shrunk (see cpu_baseline.sample)
SAMPLES = {"large": dict(grid=(24, 32), num_points=250_000), "mid": dict(grid=(15, 20), num_points=160_000),
           "skewed": dict(num_cameras=600, num_points=120_000), "small": {}, "tiny": {}}


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


TRAFFIC_FILE = os.path.join("profiles", "r02_traffic.csv")


def ncu_traffic(kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on the Large scene, from the committed
    `ncu --set full` summary (a builder run under ncu, not measured in this run: `traffic_source` says so)."""
    import csv
    try:
        with open(os.path.join(ROOT, TRAFFIC_FILE)) as fh:
            for row in csv.DictReader(fh):
                if row["kernel"] == kernel:
                    return float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
            except Exception:
                continue
            for name, cell in zip(names, r[5:9]):
                if cell.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def nielsen(lam: float, nu: float, step):
    if step.accepted:
        c = 2.0 * step.rho - 1.0
        return lam * max(1.0 / 3.0, 1.0 - c * c * c), 2.0
    return lam * nu, 2.0 * nu


# ---------------------------------------------------------------------------------------------------
# reference arm: the fp64 oracle, as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------
def time_oracle(workload: str, steps: int, warmup: int):
    """The oracle, as it stands, on the box's host cores, on a BOUNDED SAMPLE of `workload` (the same recipe shrunk:
    the full 'large' scene needs ~30 s per LM iteration and 6 GB of fp64 Jacobians).  Returns a description dict
    whose `sample_lm_iterations_per_s` is MEASURED and whose `value` is that rate scaled by the observation count to
    the full workload (`extrapolated`: the oracle is O(observations) per matvec; PCG iteration counts are the
    sample's own)."""
    import oracle
    from ba_scenes import CONFIGS, FULL_OBSERVATIONS, make_scene

    scene = make_scene(workload, **SAMPLES[workload])
    cfg = CONFIGS[workload]
    ref = oracle.OracleBA.from_scene(scene)
    lam, nu = LAMBDA0, 2.0
    matvecs = 0
    elapsed = 0.0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        st = ref.lm_step(lam, cfg["pcg_rel_tol"], cfg["pcg_max_iter"], 0)
        dt = time.perf_counter() - t0
        if it >= warmup:
            elapsed += dt
            matvecs += st.pcg_iterations
        lam, nu = nielsen(lam, nu, st)
    n_s, n_full = scene.num_observations, FULL_OBSERVATIONS[workload]
    per_it_sample = steps / elapsed
    factor = n_s / n_full
    return {"kind": "oracle", "cores": oracle.num_threads(), "unit": "LM iterations/s",
            "value": per_it_sample * factor, "extrapolated": factor != 1.0, "extrapolation_factor": factor,
            "sample": (f"{workload} recipe shrunk to {scene.num_cameras} cameras / {scene.num_points} points / "
                       f"{n_s} observations; {steps} LM iterations (PCG cap {cfg['pcg_max_iter']}, tol "
                       f"{cfg['pcg_rel_tol']:g}; {matvecs} matvecs) took {elapsed:.2f} s = {per_it_sample:.3f} it/s MEASURED "
                       f"on the sample; `value` scales it by observations ({n_s}/{n_full})"),
            "sample_lm_iterations_per_s": per_it_sample, "sample_observations": n_s, "sample_seconds": elapsed,
            "sample_matvecs_per_s": matvecs / elapsed}


def time_oracle_full(scene, workload: str, budget_s: float = 10.0, max_steps: int = 5):
    """The oracle, as it stands, on the box's host cores, on the ACTUAL bench scene (not shrunk, nothing extrapolated):
    the first LM iterations of the same adaptive schedule, stopped once `budget_s` of CPU work is spent (at least one
    iteration: 16-17 s with 42 PCG iterations on Large, 8 GB of fp64 Jacobians)."""
    import oracle
    from ba_scenes import CONFIGS

    cfg = CONFIGS[workload]
    t_create = time.perf_counter()
    ref = oracle.OracleBA.from_scene(scene)
    t_create = time.perf_counter() - t_create
    lam, nu, matvecs, elapsed, done = LAMBDA0, 2.0, 0, 0.0, 0
    per_step = []
    while done < max_steps and (done == 0 or elapsed < budget_s):
        t0 = time.perf_counter()
        st = ref.lm_step(lam, cfg["pcg_rel_tol"], cfg["pcg_max_iter"], 0)
        dt = time.perf_counter() - t0
        elapsed += dt
        matvecs += st.pcg_iterations
        per_step.append((dt, st.pcg_iterations))
        lam, nu = nielsen(lam, nu, st)
        done += 1
    ref.close()
    return {"kind": "oracle", "cores": oracle.num_threads(), "unit": "LM iterations/s", "value": done / elapsed,
            "extrapolated": False,
            "sample": (f"the first {done} LM iteration(s) of the bench workload itself ({scene.num_observations} observations, PCG cap "
                       f"{cfg['pcg_max_iter']}, tol {cfg['pcg_rel_tol']:g}): {matvecs} Schur matvecs in {elapsed:.2f} s MEASURED; the GPU's "
                       f"`value` averages over its K steps, whose later iterations run more PCG iterations: compare matvecs/s"),
            "sample_lm_iterations": done, "sample_seconds": elapsed, "sample_matvecs": matvecs,
            "sample_matvecs_per_s": matvecs / elapsed, "seconds_per_step": [round(a, 3) for a, _ in per_step],
            "pcg_iterations_per_step": [b for _, b in per_step], "oracle_create_seconds": t_create}


def time_oracle_single_thread(workload: str):
    """One LM iteration of the same sample with OMP_NUM_THREADS=1, in a child process (the thread count is fixed
    when the OpenMP runtime starts)."""
    code = ("import json,sys,time; sys.path.insert(0, %r); import bench, oracle; from ba_scenes import CONFIGS, make_scene;"
            "w=%r; s=make_scene(w, **bench.SAMPLES[w]); c=CONFIGS[w]; o=oracle.OracleBA.from_scene(s);"
            "t=time.perf_counter(); st=o.lm_step(bench.LAMBDA0, c['pcg_rel_tol'], c['pcg_max_iter'], 0);"
            "print(json.dumps({'seconds': time.perf_counter()-t, 'matvecs': st.pcg_iterations, 'cores': oracle.num_threads()}))"
            % (ROOT, workload))
    try:
        out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, OMP_NUM_THREADS="1"),
                             capture_output=True, text=True, timeout=600, check=True).stdout
        d = json.loads(out.strip().splitlines()[-1])
        return {"cores": d["cores"], "sample_lm_iterations_per_s": 1.0 / d["seconds"], "matvecs": d["matvecs"],
                "matvecs_per_s": d["matvecs"] / d["seconds"],
                "what": "first LM iteration of the SHRUNKEN sample of this workload (bench.SAMPLES: the full scene would "
                        "take minutes on one thread), OMP_NUM_THREADS=1"}
    except Exception as exc:  # reported, never fatal for the bench line
        return {"error": str(exc)[:200]}


def run_reference(args):
    """--impl reference: the oracle on the host cores.  `value` and `ms_per_step` are MEASURED on the bounded sample
    (not scaled); cpu_baseline carries the same number scaled to the full workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from ba_scenes import CONFIGS
    t0 = time.perf_counter()
    desc = time_oracle(args.workload, args.steps, args.warmup)
    wall = time.perf_counter() - t0
    cfg = CONFIGS[args.workload]
    value = desc["sample_lm_iterations_per_s"]
    line = {"impl": "reference", "metric": "lm_iterations_per_s", "value": value, "unit": "LM iterations/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BOUNDED SAMPLE of BASELINE.json configs '{args.workload}' (seed {cfg['seed']}): "
                                   f"{desc['sample_observations']} observations, not the full workload",
                       "pcg_max_iter": cfg["pcg_max_iter"], "pcg_rel_tol": cfg["pcg_rel_tol"], "lambda0": LAMBDA0},
            "cpu_baseline": desc, "gpu_launches": 0, "wall_s": wall,
            "e2e": {"value": value, "unit": "LM iterations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# N > 1: the path does not shard ("replicas only"): every rank runs an independent replica of the
# config on its own seed, there is no data-path collective; the only exchange is the timing reduction below
# ---------------------------------------------------------------------------------------------------
def replica_seed(config_seed: int, rank: int) -> int:
    return config_seed + 1000 * rank


def max_over_ranks(value: float, device=None) -> float:
    """MAX of a per-rank scalar over the process group (identity without one)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world: int, units_per_rank: float, ms_max: float) -> float:
    """Units all ranks processed / the slowest rank's time (weak scaling: per-rank work is fixed)."""
    return world * units_per_rank / (ms_max * 1e-3)


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2605_30583_b200 as pkg
    from ba_scenes import CONFIGS, make_scene

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = CONFIGS[args.workload]
    kw = {}
    if args.shrink:                                   # debugging only; the bench line says so
        kw = SAMPLES[args.workload]
    sharded = args.parallelism == "sharded"
    scene = make_scene(args.workload, seed=cfg["seed"] if sharded else replica_seed(cfg["seed"], rank), **kw)
    n_obs = scene.num_observations
    full_scene = scene
    if sharded:   # every rank builds the same scene and keeps its own range of points (whole tracks)
        import dataclasses
        from paper_2605_30583_b200 import sharding
        sh = sharding.make_shard(scene.num_points, scene.camera_index, scene.point_index, world, rank)
        pts_l, obs_l = sharding.shard_arrays(sh, scene.points, scene.observations)
        scene = dataclasses.replace(scene, points=np.ascontiguousarray(pts_l), observations=np.ascontiguousarray(obs_l),
                                    camera_index=sh.camera_index, point_index=sh.point_index)
    cams0 = torch.from_numpy(scene.cameras).to(dev)
    pts0 = torch.from_numpy(scene.points).to(dev)
    gpu = pkg.CasparBA(cams0.clone(), pts0.clone(), scene.observations, scene.camera_index, scene.point_index,
                       scene.robust_loss, scene.robust_scale, 0, device=dev)
    if sharded:
        if world == 1 and not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29655")
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
        gpu.set_shard(sharding.torch_exchange(), is_root=(rank == 0))
    tol, cap = cfg["pcg_rel_tol"], cfg["pcg_max_iter"]

    cam_h = torch.empty((scene.num_cameras, 9), dtype=torch.float32).pin_memory()
    pts_h = torch.empty((scene.num_points, 3), dtype=torch.float32).pin_memory()

    def reset():
        """Start parameters back into the borrowed device arrays; the handle's cached linearization is
        marked stale, so the first timed step linearizes like every other one."""
        cam_h.copy_(torch.from_numpy(scene.cameras))
        pts_h.copy_(torch.from_numpy(scene.points))
        gpu.set_parameters_host(cam_h, pts_h)
        torch.cuda.synchronize()

    def run_steps(k, e2e_buffers=None):
        lam, nu, out = LAMBDA0, 2.0, []
        for _ in range(k):
            if e2e_buffers is not None:
                gpu.set_parameters_host(*e2e_buffers)
            st = gpu.lm_step(float(np.float32(lam)), tol, cap, 0)
            if e2e_buffers is not None:
                gpu.get_parameters_host(*e2e_buffers)
            lam, nu = nielsen(lam, nu, st)
            out.append(st)
        return out

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident: warm-up, reset, K timed steps in the library's DEFAULT mode (profiling off: the PCG loop
    # goes out as CUDA-graph chunks) -> `value`
    create_stats = gpu.stats()
    run_steps(args.warmup)
    reset()
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches_before = int(gpu.stats().kernels_launched)
    with ClockSampler(local) as clocks:
        start.record()
        steps = run_steps(args.steps)
        stop.record()
        barrier()
    ms = start.elapsed_time(stop)
    launches_default = int(gpu.stats().kernels_launched) - launches_before
    ms_max = max_over_ranks(ms, dev)
    matvecs = sum(s.pcg_iterations for s in steps)

    # ---- the same K steps again with CUDA events around every linearize / Schur-matvec launch (this switches the
    # graph chunks off): only the per-kernel averages of the roofline fields come from this pass
    reset()
    gpu.set_profiling(True)
    barrier()
    start2, stop2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    start2.record()
    steps_prof = run_steps(args.steps)
    stop2.record()
    barrier()
    ms_prof = start2.elapsed_time(stop2)
    st = gpu.stats()
    gpu.set_profiling(False)
    matvecs_prof = sum(s.pcg_iterations for s in steps_prof)
    lin_count = int(st.linearize_count)

    # ---- end to end: host buffers, H2D + lm_step + D2H every step ------------------------------------
    e2e_s = float("nan")
    if not args.no_e2e:
        reset()
        run_steps(1, (cam_h, pts_h))
        reset()
        barrier()
        t0 = time.perf_counter()
        run_steps(args.steps, (cam_h, pts_h))
        barrier()
        e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dev)
    param_bytes = 4 * (9 * scene.num_cameras + 3 * scene.num_points)

    if rank != 0:
        if dist.is_initialized():
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (Schur matvec) and of linearize -----------------------------
    peak, peak_src = hbm_peak()
    observed_points = int(np.unique(scene.point_index).size)
    # algorithmic bytes:
    #   matvec   : J_c 72 + J_p 24 + camera id 4 per observation, V'^-1 24 per observed point
    #   linearize: pixel 8 + camera id 4 + r 8 + J_c 72 + J_p 24 per observation, X 12 + V,g_p 36 per point
    n_local = scene.num_observations          # = n_obs unless the problem is sharded (then: this rank's share)
    mv_bytes = 100.0 * n_local + 24.0 * observed_points
    lin_bytes = 116.0 * n_local + 48.0 * observed_points
    # launches enqueued after the device-side convergence flag was set return at once (a few us each):
    # their time is kept in the total, but the average is over the matvecs that ran
    mv_ms = st.matvec_ms_total / max(1, matvecs_prof)
    lin_ms = st.linearize_ms_total / max(1, st.linearize_count)
    mv_gbs = mv_bytes / (mv_ms * 1e-3) / 1e9 if mv_ms > 0 else 0.0
    lin_gbs = lin_bytes / (lin_ms * 1e-3) / 1e9 if lin_ms > 0 else 0.0

    # replicas: every rank did K steps of its own problem; sharded: the ranks did K steps of ONE problem together
    value = args.steps / (ms_max * 1e-3) if sharded else whole_job_rate(world, args.steps, ms_max)
    line = {
        "metric": "lm_iterations_per_s", "value": value, "unit": "LM iterations/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{['tiny', 'small', 'mid', 'large', 'skewed'].index(args.workload)}] '{args.workload}' (seed {cfg['seed']})" + (" SHRUNK (debug)" if args.shrink else ""),
                   "cameras": full_scene.num_cameras, "points": full_scene.num_points, "observations": n_obs,
                   "pcg_max_iter": cap, "pcg_rel_tol": tol, "lambda0": LAMBDA0, "tile_slots": int(st.tile_slots),
                   "l2": "inputs larger than L2 (stored Jacobians %.2f GB per pass)" % (96.0 * n_obs / 1e9),
                   "replicas": 1 if sharded else world,
                   "parallelism": (f"points sharded over {world} rank(s): all-reduce of U/g_c, b, every q (9 Nc doubles) and "
                                   f"the step scalars, broadcast of the PCG scalars; {int(st.shard_exchanges)} collectives in the profiled pass")
                   if sharded else "independent replicas, no collective"},
        "schur_matvecs_per_s": (matvecs / (ms_max * 1e-3)) if sharded else whole_job_rate(world, matvecs, ms_max),
        "matvecs_in_timed_region": matvecs,
        "linearizations_per_s": world * n_local / (lin_ms * 1e-3) if lin_ms > 0 else None,
        "lm_costs": [s.cost_after for s in steps], "lm_accepted": [bool(s.accepted) for s in steps],
        "pcg_iterations": [s.pcg_iterations for s in steps],
        "roofline": {"kernel": "schur_matvec_pipelined_kernel<T>" if st.matvec_pipelined else "schur_pass_kernel<T,MATVEC>", "bound": "hbm", "achieved": mv_gbs, "peak": peak,
                     "unit": "GB/s", "frac": mv_gbs / peak, "traffic": ncu_traffic("schur_matvec") if args.workload == "large" and not args.shrink else None,
                     "traffic_source": TRAFFIC_FILE + " (ncu --set full, builder run; not measured in this run)",
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": mv_bytes, "avg_launch_ms": mv_ms,
                     "launches_timed": int(matvecs_prof), "launches_enqueued": int(st.matvec_count), "frac_of_nominal_8TBs": mv_gbs / 8000.0,
                     "timed_in": "second pass of the same K steps with per-launch CUDA events (graph chunks off)"},
        "roofline_linearize": {"kernel": "linearize_pipelined_kernel<T,NG>" if st.linearize_pipelined else "linearize_kernel<T,true>", "bound": "hbm", "achieved": lin_gbs, "peak": peak,
                               "unit": "GB/s", "frac": lin_gbs / peak, "traffic": ncu_traffic("linearize") if args.workload == "large" and not args.shrink else None,
                               "algorithmic_bytes_per_launch": lin_bytes, "avg_launch_ms": lin_ms,
                               "launches_timed": lin_count, "frac_of_nominal_8TBs": lin_gbs / 8000.0},
        "e2e": {"value": (1 if sharded else world) * args.steps / e2e_s, "unit": "LM iterations/s", "h2d_bytes_per_step": param_bytes,
                "d2h_bytes_per_step": param_bytes + 88,
                "what": "pinned host parameters -> caspar_ba_set_parameters_host, caspar_ba_lm_step, "
                        "caspar_ba_get_parameters_host + step_info, every step; wall clock"},
        "gpu_launches": launches_default,
        "value_mode": "library default (profiling off, PCG iterations launched as CUDA-graph chunks of 8)",
        "profiled_pass": {"ms_per_step": ms_prof / args.steps, "lm_iterations_per_s": args.steps / (ms_prof * 1e-3),
                          "gpu_launches": int(st.kernels_launched)},
        "create": {"seconds": create_stats.create_seconds, "reorder_seconds": create_stats.reorder_seconds,
                   "arena_bytes": int(create_stats.arena_bytes),
                   "what": "caspar_ba_create on this scene (host reordering S0 + uploads), once, untimed"},
        "clocks": clocks.summary(),
    }
    if world == 1 and not args.no_cpu_baseline:
        gpu.close()                                                # the oracle needs the host, not the GPU arena
        if args.shrink:
            desc = time_oracle(args.workload, 5, 0)
        else:
            desc = time_oracle_full(full_scene, args.workload)     # 10-20 s of oracle work on the ACTUAL workload
            desc["gpu_matvecs_per_s_same_run"] = line["schur_matvecs_per_s"]
        desc["single_thread"] = time_oracle_single_thread(args.workload)
        line["cpu_baseline"] = desc
    print(json.dumps(line), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="large", choices=list(SAMPLES))
    ap.add_argument("--shrink", action="store_true", help="debug: run the shrunken sample scene on the GPU")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "sharded"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE problem with its points sharded "
                         "over the ranks (strong scaling; caspar_ba_set_shard over NCCL)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="profiling runs: skip the host-buffer end-to-end leg")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
