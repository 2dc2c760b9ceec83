"""Thin ctypes binding of libcaspar_ba.so (include/caspar_ba.h): argument marshalling only.

PyTorch is used for device memory and streams, nothing else; every step of the path runs in the
library's sm_100a kernels.  There is NO fallback: if the library is missing or no CUDA device is
present, construction raises.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
from typing import List, Optional

import numpy as np
import torch

from . import build as _build

OK, EINVAL, ECUDA, ENOMEM, ENUMERIC, ESTATE = 0, -1, -2, -3, -4, -5
RESIDUALS, JC, JP, U, V, G, SCHUR_RHS, DELTA, PRECONDITIONER = range(9)

EXPORTED_SYMBOLS = [
    "caspar_ba_create", "caspar_ba_linearize", "caspar_ba_pcg_solve", "caspar_ba_lm_step", "caspar_ba_solve",
    "caspar_ba_cost", "caspar_ba_destroy", "caspar_ba_set_parameters_host", "caspar_ba_get_parameters_host",
    "caspar_ba_export", "caspar_ba_schur_matvec", "caspar_ba_get_stats", "caspar_ba_set_profiling",
    "caspar_ba_last_error", "caspar_ba_layout_create", "caspar_ba_layout_get_info", "caspar_ba_layout_copy",
    "caspar_ba_layout_destroy", "caspar_ba_set_preconditioner", "caspar_ba_pcgnr_solve", "caspar_ba_set_linear_solver",
    "caspar_ba_set_fusion", "caspar_ba_set_shard", "caspar_ba_cost_static",
]

STATIC_MAX_CAMERAS = 16384  # CASPAR_BA_STATIC_MAX_CAMERAS


class Problem(C.Structure):
    _fields_ = [("num_cameras", C.c_int32), ("num_points", C.c_int32), ("num_observations", C.c_int64),
                ("cameras", C.c_void_p), ("points", C.c_void_p), ("observations", C.c_void_p),
                ("camera_index", C.c_void_p), ("point_index", C.c_void_p),
                ("robust_loss", C.c_int32), ("robust_scale", C.c_float), ("damping_mode", C.c_int32),
                ("camera_model", C.c_int32), ("depth_epsilon", C.c_float)]


class PcgInfo(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("converged", C.c_int32), ("rel_residual", C.c_double),
                ("rz0", C.c_double), ("rz", C.c_double)]


class StepInfo(C.Structure):
    _fields_ = [("cost_before", C.c_double), ("cost_after", C.c_double), ("model_decrease", C.c_double),
                ("rho", C.c_double), ("accepted", C.c_int32), ("pcg", PcgInfo)]


class Stats(C.Structure):
    _fields_ = [("tile_slots", C.c_int32), ("num_tiles", C.c_int32), ("padded_slots", C.c_int64),
                ("camera_runs", C.c_int64), ("arena_bytes", C.c_int64), ("kernels_launched", C.c_int64),
                ("linearize_ms_total", C.c_double), ("matvec_ms_total", C.c_double),
                ("linearize_count", C.c_int64), ("matvec_count", C.c_int64),
                ("matvec_pipelined", C.c_int32), ("pipeline_stages", C.c_int32),
                ("num_hot_cameras", C.c_int32), ("device", C.c_int32),
                ("create_seconds", C.c_double), ("reorder_seconds", C.c_double),
                ("linearize_pipelined", C.c_int32), ("reserved", C.c_int32),
                ("speculative_hits", C.c_int64), ("speculative_misses", C.c_int64), ("arena2_bytes", C.c_int64),
                ("shard_exchanges", C.c_int64)]


# int fn(void* ctx, size_t count, void* cuda_stream)
EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_size_t, C.c_void_p)


class LayoutInfo(C.Structure):
    _fields_ = [("tile_slots", C.c_int32), ("num_tiles", C.c_int32), ("observed_points", C.c_int32),
                ("num_chunks", C.c_int32), ("padded_slots", C.c_int64), ("camera_runs", C.c_int64)]


@dataclasses.dataclass
class Step:
    lam: float
    cost_before: float
    cost_after: float
    model_decrease: float
    rho: float
    accepted: bool
    pcg_iterations: int
    pcg_converged: bool
    pcg_rel_residual: float


def _step(info: StepInfo, lam: float) -> Step:
    return Step(lam, info.cost_before, info.cost_after, info.model_decrease, info.rho, bool(info.accepted),
                info.pcg.iterations, bool(info.pcg.converged), info.pcg.rel_residual)


class CasparError(RuntimeError):
    def __init__(self, code: int, where: str, text: str = ""):
        super().__init__(f"caspar_ba: {where} returned {code}" + (f" ({text})" if text else ""))
        self.code = code


_lib: Optional[C.CDLL] = None


def library_path() -> str:
    return _build.LIBRARY


def load_library() -> C.CDLL:
    """dlopen the in-tree library (building it first if the sources are newer).  Loading needs no GPU."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    if not os.path.exists(path):
        raise RuntimeError(f"CUDA library missing: {path} (run __graft_entry__.build())")
    L = C.CDLL(path)
    vp = C.c_void_p
    L.caspar_ba_create.argtypes = [C.POINTER(Problem), vp, C.POINTER(vp)]
    L.caspar_ba_linearize.argtypes = [vp, vp, C.POINTER(C.c_double)]
    L.caspar_ba_pcg_solve.argtypes = [vp, C.c_float, C.c_float, C.c_int32, vp, C.POINTER(PcgInfo)]
    L.caspar_ba_lm_step.argtypes = [vp, C.c_float, C.c_float, C.c_int32, C.c_int32, vp, C.POINTER(StepInfo)]
    L.caspar_ba_solve.argtypes = [vp, C.c_int32, C.c_float, C.c_float, C.c_int32, vp, C.POINTER(StepInfo),
                                  C.POINTER(C.c_float)]
    L.caspar_ba_cost.argtypes = [vp, vp, C.POINTER(C.c_double)]
    L.caspar_ba_destroy.argtypes = [vp]
    L.caspar_ba_destroy.restype = None
    L.caspar_ba_set_parameters_host.argtypes = [vp, vp, vp, vp]
    L.caspar_ba_get_parameters_host.argtypes = [vp, vp, vp, vp]
    L.caspar_ba_export.argtypes = [vp, C.c_int32, vp, C.c_size_t, vp]
    L.caspar_ba_schur_matvec.argtypes = [vp, C.c_float, vp, vp, vp]
    L.caspar_ba_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.caspar_ba_set_profiling.argtypes = [vp, C.c_int32]
    L.caspar_ba_last_error.argtypes = [vp]
    L.caspar_ba_last_error.restype = C.c_char_p
    L.caspar_ba_layout_create.argtypes = [C.c_int32, C.c_int32, C.c_int64, vp, vp, C.c_int32, C.POINTER(vp)]
    L.caspar_ba_layout_get_info.argtypes = [vp, C.POINTER(LayoutInfo)]
    L.caspar_ba_layout_copy.argtypes = [vp, C.c_int32, vp, C.c_size_t]
    L.caspar_ba_layout_destroy.argtypes = [vp]
    L.caspar_ba_layout_destroy.restype = None
    L.caspar_ba_set_preconditioner.argtypes = [vp, C.c_int32]
    L.caspar_ba_set_fusion.argtypes = [vp, C.c_int32]
    L.caspar_ba_set_shard.argtypes = [vp, EXCHANGE_FN, vp, vp, C.c_size_t, C.c_int32]
    L.caspar_ba_set_linear_solver.argtypes = [vp, C.c_int32]
    L.caspar_ba_cost_static.argtypes = [C.POINTER(Problem), vp, vp]
    L.caspar_ba_pcgnr_solve.argtypes = [vp, C.c_float, C.c_float, C.c_int32, vp, C.POINTER(PcgInfo)]
    _lib = L
    return L


def plan_layout(num_cameras: int, num_points: int, camera_index, point_index, tile: int = 0) -> dict:
    """Step S0 on its own (host only, needs no GPU): the reordering `caspar_ba_create` performs."""
    L = load_library()
    ci = np.ascontiguousarray(np.asarray(camera_index, dtype=np.int32))
    pi = np.ascontiguousarray(np.asarray(point_index, dtype=np.int32))
    h = C.c_void_p()
    rc = L.caspar_ba_layout_create(num_cameras, num_points, ci.shape[0], ci.ctypes.data, pi.ctypes.data, tile,
                                   C.byref(h))
    if rc:
        raise CasparError(rc, "layout_create", L.caspar_ba_last_error(None).decode())
    try:
        info = LayoutInfo()
        L.caspar_ba_layout_get_info(h, C.byref(info))
        slots, tiles, runs = info.padded_slots, info.num_tiles, info.camera_runs
        spec = [("obs_of_slot", np.int32, slots), ("cam", np.int32, slots), ("rank", np.uint16, slots),
                ("tile_pt", np.int32, tiles + 1), ("run_begin", np.int32, tiles + 1),
                ("run_cam", np.int32, runs + tiles + 1), ("run_slot", np.uint16, runs + tiles + 1),
                ("pt_ptr", np.int32, info.observed_points + 1), ("pt_perm", np.int32, num_points),
                ("cslot", np.int32, ci.shape[0]), ("chunk_cam", np.int32, info.num_chunks),
                ("chunk_begin", np.int32, info.num_chunks + 1)]
        out = dict(T=info.tile_slots, num_tiles=tiles, observed_points=info.observed_points,
                   num_chunks=info.num_chunks, padded_slots=slots, camera_runs=runs)
        for which, (name, dtype, count) in enumerate(spec):
            a = np.empty(int(count), dtype=dtype)
            rc = L.caspar_ba_layout_copy(h, which, a.ctypes.data, a.nbytes)
            if rc:
                raise CasparError(rc, f"layout_copy({name})")
            out[name] = a
        return out
    finally:
        L.caspar_ba_layout_destroy(h)


def _stream_ptr(stream: Optional[torch.cuda.Stream], device=None) -> int:
    """cudaStream_t of `stream`, default: the current stream OF `device` (not of whatever device is current)."""
    return (stream or torch.cuda.current_stream(device)).cuda_stream


def cost_static(cameras: torch.Tensor, points: torch.Tensor, observations: torch.Tensor, camera_index: torch.Tensor,
                point_index: torch.Tensor, cost_out: torch.Tensor, robust_loss: int = 0, robust_scale: float = 0.0,
                depth_epsilon: float = 0.0, stream=None) -> None:
    """caspar_ba_cost_static: F at the given parameters into `cost_out[0]` (CUDA float64), no handle, no allocation
    (the library's fixed scratch array; at most STATIC_MAX_CAMERAS cameras).  Asynchronous on `stream`.  Every tensor
    must already be a contiguous CUDA tensor of the right dtype: nothing is converted or copied here."""
    if not torch.cuda.is_available():
        raise RuntimeError("caspar_ba needs a CUDA device; there is no CPU fallback")
    for name, t, dtype in (("cameras", cameras, torch.float32), ("points", points, torch.float32),
                           ("observations", observations, torch.float32), ("camera_index", camera_index, torch.int32),
                           ("point_index", point_index, torch.int32), ("cost_out", cost_out, torch.float64)):
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    if cost_out.numel() < 1 or camera_index.numel() != point_index.numel() or observations.numel() != 2 * camera_index.numel():
        raise ValueError("cost_out needs one element; the index arrays one entry per observation")
    L = load_library()
    dev = cameras.device
    pb = Problem(cameras.numel() // 9, points.numel() // 3, camera_index.numel(), cameras.data_ptr(),
                 points.data_ptr(), observations.data_ptr(), camera_index.data_ptr(), point_index.data_ptr(),
                 int(robust_loss), float(robust_scale), 0, 0, float(depth_epsilon))
    with torch.cuda.device(dev):   # the entry point runs on the CURRENT device
        rc = L.caspar_ba_cost_static(C.byref(pb), cost_out.data_ptr(), _stream_ptr(stream, dev))
    if rc:
        raise CasparError(rc, "cost_static", L.caspar_ba_last_error(None).decode())


class CasparBA:
    """One bundle-adjustment problem on the current CUDA device.

    `cameras` [Nc, 9] and `points` [Np, 3] are float32 CUDA tensors that the library borrows and
    updates in place on an accepted step; numpy arrays are copied to new device tensors
    (available as `.cameras` / `.points`)."""

    def __init__(self, cameras, points, observations, camera_index, point_index, robust_loss: int = 0,
                 robust_scale: float = 0.0, damping_mode: int = 0, device: Optional[torch.device] = None,
                 camera_model: int = 0, depth_epsilon: float = 0.0):
        if not torch.cuda.is_available():
            raise RuntimeError("caspar_ba needs a CUDA device; there is no CPU fallback")
        self._lib = load_library()
        self._h = None
        dev = torch.device(device) if device is not None else torch.device("cuda", torch.cuda.current_device())
        self.device = dev

        def dev_tensor(x, dtype, shape):
            t = torch.as_tensor(x)
            t = t.to(device=dev, dtype=dtype).contiguous()
            return t.reshape(shape)

        self.cameras = dev_tensor(cameras, torch.float32, (-1, 9))
        self.points = dev_tensor(points, torch.float32, (-1, 3))
        obs = dev_tensor(observations, torch.float32, (-1, 2))
        ci = dev_tensor(camera_index, torch.int32, (-1,))
        pi = dev_tensor(point_index, torch.int32, (-1,))
        self.nc, self.np_, self.n = self.cameras.shape[0], self.points.shape[0], obs.shape[0]
        if ci.shape[0] != self.n or pi.shape[0] != self.n:
            raise ValueError("index arrays must have one entry per observation")
        pb = Problem(self.nc, self.np_, self.n, self.cameras.data_ptr(), self.points.data_ptr(), obs.data_ptr(),
                     ci.data_ptr(), pi.data_ptr(), int(robust_loss), float(robust_scale), int(damping_mode),
                     int(camera_model), float(depth_epsilon))
        h = C.c_void_p()
        with torch.cuda.device(dev):   # create binds the handle to the CURRENT device; later calls switch to it
            rc = self._lib.caspar_ba_create(C.byref(pb), _stream_ptr(None, dev), C.byref(h))
        if rc:
            raise CasparError(rc, "create", self._lib.caspar_ba_last_error(None).decode())
        self._h = h

    @classmethod
    def from_scene(cls, scene, damping_mode: int = 0, **kw) -> "CasparBA":
        return cls(scene.cameras, scene.points, scene.observations, scene.camera_index, scene.point_index,
                   kw.pop("robust_loss", scene.robust_loss), kw.pop("robust_scale", scene.robust_scale),
                   damping_mode, **kw)

    def close(self):
        if getattr(self, "_h", None) and self._lib is not None and self._lib.caspar_ba_destroy is not None:
            self._lib.caspar_ba_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, rc: int, where: str):
        if rc:
            raise CasparError(rc, where, self._lib.caspar_ba_last_error(self._h).decode())

    # ---- the path ------------------------------------------------------------------------------
    def linearize(self, stream=None) -> float:
        cost = C.c_double()
        self._check(self._lib.caspar_ba_linearize(self._h, _stream_ptr(stream, self.device), C.byref(cost)), "linearize")
        return cost.value

    def cost(self, stream=None) -> float:
        cost = C.c_double()
        self._check(self._lib.caspar_ba_cost(self._h, _stream_ptr(stream, self.device), C.byref(cost)), "cost")
        return cost.value

    def pcg_solve(self, lam: float, rel_tol: float, max_iter: int, stream=None) -> PcgInfo:
        info = PcgInfo()
        self._check(self._lib.caspar_ba_pcg_solve(self._h, lam, rel_tol, max_iter, _stream_ptr(stream, self.device),
                                                  C.byref(info)), "pcg_solve")
        return info

    def pcgnr_solve(self, lam: float, rel_tol: float, max_iter: int, stream=None) -> PcgInfo:
        info = PcgInfo()
        self._check(self._lib.caspar_ba_pcgnr_solve(self._h, lam, rel_tol, max_iter, _stream_ptr(stream, self.device),
                                                    C.byref(info)), "pcgnr_solve")
        return info

    def set_linear_solver(self, mode: int):
        self._check(self._lib.caspar_ba_set_linear_solver(self._h, int(mode)), "set_linear_solver")

    def lm_step(self, lam: float, rel_tol: float, max_iter: int, accept_mode: int = 0, stream=None) -> Step:
        info = StepInfo()
        self._check(self._lib.caspar_ba_lm_step(self._h, lam, rel_tol, max_iter, accept_mode, _stream_ptr(stream, self.device),
                                                C.byref(info)), "lm_step")
        return _step(info, lam)

    def solve(self, iterations: int, lambda0: float, rel_tol: float, max_iter: int, stream=None) -> List[Step]:
        infos = (StepInfo * max(1, iterations))()
        lams = (C.c_float * max(1, iterations))()
        self._check(self._lib.caspar_ba_solve(self._h, iterations, lambda0, rel_tol, max_iter, _stream_ptr(stream, self.device),
                                              infos, lams), "solve")
        return [_step(infos[i], float(lams[i])) for i in range(iterations)]

    def set_parameters_host(self, cameras: torch.Tensor, points: torch.Tensor, stream=None):
        assert cameras.dtype == torch.float32 and points.dtype == torch.float32 and not cameras.is_cuda
        self._check(self._lib.caspar_ba_set_parameters_host(self._h, cameras.data_ptr(), points.data_ptr(),
                                                            _stream_ptr(stream, self.device)), "set_parameters_host")

    def get_parameters_host(self, cameras: torch.Tensor, points: torch.Tensor, stream=None):
        assert cameras.dtype == torch.float32 and points.dtype == torch.float32 and not cameras.is_cuda
        self._check(self._lib.caspar_ba_get_parameters_host(self._h, cameras.data_ptr(), points.data_ptr(),
                                                            _stream_ptr(stream, self.device)), "get_parameters_host")

    # ---- test-only exports ---------------------------------------------------------------------
    def export(self, what: int, stream=None) -> np.ndarray:
        nc, np_, n = self.nc, self.np_, self.n
        shape = {RESIDUALS: (n, 2), JC: (n, 2, 9), JP: (n, 2, 3), U: (nc, 9, 9), V: (np_, 3, 3),
                 G: (9 * nc + 3 * np_,), SCHUR_RHS: (9 * nc,), DELTA: (9 * nc + 3 * np_,),
                 PRECONDITIONER: (nc, 9, 9)}[what]
        return self.export_device(what, stream).cpu().numpy()

    def export_device(self, what: int, stream=None) -> torch.Tensor:
        """The same export left on the device (fp64, caller's order): full-size tests sample it there."""
        nc, np_, n = self.nc, self.np_, self.n
        shape = {RESIDUALS: (n, 2), JC: (n, 2, 9), JP: (n, 2, 3), U: (nc, 9, 9), V: (np_, 3, 3),
                 G: (9 * nc + 3 * np_,), SCHUR_RHS: (9 * nc,), DELTA: (9 * nc + 3 * np_,),
                 PRECONDITIONER: (nc, 9, 9)}[what]
        count = int(np.prod(shape))
        out = torch.zeros(max(count, 1), dtype=torch.float64, device=self.device)
        self._check(self._lib.caspar_ba_export(self._h, what, out.data_ptr(), count, _stream_ptr(stream, self.device)),
                    f"export({what})")
        return out[:count].reshape(shape)

    def schur_matvec(self, lam: float, p, stream=None) -> np.ndarray:
        p_dev = torch.as_tensor(np.asarray(p, dtype=np.float64)).to(self.device).contiguous()
        q_dev = torch.empty_like(p_dev)
        self._check(self._lib.caspar_ba_schur_matvec(self._h, lam, p_dev.data_ptr(), q_dev.data_ptr(),
                                                     _stream_ptr(stream, self.device)), "schur_matvec")
        return q_dev.cpu().numpy()

    def schur_matvec_device(self, lam: float, p_dev: torch.Tensor, q_dev: torch.Tensor, stream=None):
        self._check(self._lib.caspar_ba_schur_matvec(self._h, lam, p_dev.data_ptr(), q_dev.data_ptr(),
                                                     _stream_ptr(stream, self.device)), "schur_matvec")

    # ---- introspection -------------------------------------------------------------------------
    def stats(self) -> Stats:
        st = Stats()
        self._check(self._lib.caspar_ba_get_stats(self._h, C.byref(st)), "get_stats")
        return st

    def set_shard(self, exchange, is_root: bool):
        """Make this handle ONE SHARD of a point-sharded problem (include/caspar_ba.h: caspar_ba_set_shard).
        `exchange(buffer, count)` is called with the handle's exchange buffer (a float64 CUDA tensor), on the current
        stream: it sums buffer[:count] over the shards in place (an all-reduce).  `exchange=None` returns to a
        single-GPU problem.  See `sharding.torch_exchange`."""
        if exchange is None:
            self._check(self._lib.caspar_ba_set_shard(self._h, EXCHANGE_FN(0), None, None, 0, 1), "set_shard")
            self._exchange_cb = self._xchg = None
            return
        self._xchg = torch.zeros(54 * self.nc + 8, dtype=torch.float64, device=self.device)
        buf = self._xchg

        def _cb(_ctx, count, _stream):
            try:
                exchange(buf, int(count))
                return 0
            except Exception:  # never let an exception cross the C ABI
                import traceback
                traceback.print_exc()
                return 1

        self._exchange_cb = EXCHANGE_FN(_cb)      # keep the trampoline alive as long as the handle uses it
        self._check(self._lib.caspar_ba_set_shard(self._h, self._exchange_cb, None, buf.data_ptr(), buf.numel(),
                                                  1 if is_root else 0), "set_shard")

    def set_fusion(self, mode: int):
        self._check(self._lib.caspar_ba_set_fusion(self._h, int(mode)), "set_fusion")

    def set_preconditioner(self, mode: int):
        self._check(self._lib.caspar_ba_set_preconditioner(self._h, int(mode)), "set_preconditioner")

    def set_profiling(self, enable: bool):
        self._check(self._lib.caspar_ba_set_profiling(self._h, int(enable)), "set_profiling")
