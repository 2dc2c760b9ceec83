"""ctypes binding of oracle/liboracle_ba.so (TEST INFRASTRUCTURE ONLY; see oracle_ba.h)."""
from __future__ import annotations

import ctypes as C
import dataclasses
from typing import List, Optional, Tuple

import numpy as np

from . import build as _build

_lib = None

RESIDUALS, JC, JP, U, V, G, SCHUR_RHS, DELTA, DAMPING = range(9)


class _Problem(C.Structure):
    _fields_ = [("num_cameras", C.c_int32), ("num_points", C.c_int32), ("num_observations", C.c_int64),
                ("cameras", C.c_void_p), ("points", C.c_void_p), ("observations", C.c_void_p),
                ("camera_index", C.c_void_p), ("point_index", C.c_void_p),
                ("robust_loss", C.c_int32), ("robust_scale", C.c_double), ("damping_mode", C.c_int32),
                ("camera_model", C.c_int32), ("depth_epsilon", C.c_double)]


class PcgInfo(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("converged", C.c_int32), ("rel_residual", C.c_double),
                ("rz0", C.c_double), ("rz", C.c_double)]


class StepInfo(C.Structure):
    _fields_ = [("cost_before", C.c_double), ("cost_after", C.c_double), ("model_decrease", C.c_double),
                ("rho", C.c_double), ("accepted", C.c_int32), ("pcg", PcgInfo)]


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


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        L.oracle_ba_observation.argtypes = [vp] * 6
        L.oracle_ba_observation.restype = None
        L.oracle_ba_rotation.argtypes = [vp, vp]
        L.oracle_ba_rotation.restype = None
        L.oracle_ba_spd_inverse.argtypes = [C.c_int, vp, vp]
        L.oracle_ba_create.argtypes = [C.POINTER(_Problem), C.POINTER(vp)]
        L.oracle_ba_destroy.argtypes = [vp]
        L.oracle_ba_destroy.restype = None
        L.oracle_ba_linearize.argtypes = [vp, dp]
        L.oracle_ba_cost.argtypes = [vp, dp]
        L.oracle_ba_pcg_solve.argtypes = [vp, C.c_double, C.c_double, C.c_int32, C.POINTER(PcgInfo)]
        L.oracle_ba_lm_step.argtypes = [vp, C.c_double, C.c_double, C.c_int32, C.c_int32, C.POINTER(StepInfo)]
        L.oracle_ba_solve.argtypes = [vp, C.c_int32, C.c_double, C.c_double, C.c_int32, C.POINTER(StepInfo), dp]
        L.oracle_ba_export.argtypes = [vp, C.c_int32, vp, C.c_size_t]
        L.oracle_ba_schur_matvec.argtypes = [vp, C.c_double, vp, vp]
        L.oracle_ba_full_matvec.argtypes = [vp, C.c_double, vp, vp]
        L.oracle_ba_num_threads.restype = C.c_int
        L.oracle_ba_observation_model.argtypes = [C.c_int32, C.c_double] + [vp] * 6
        L.oracle_ba_observation_model.restype = None
        L.oracle_ba_retract_camera.argtypes = [C.c_int32, vp, vp, vp]
        L.oracle_ba_retract_camera.restype = None
        L.oracle_ba_pcgnr_solve.argtypes = [vp, C.c_double, C.c_double, C.c_int32, C.POINTER(PcgInfo)]
        L.oracle_ba_set_preconditioner.argtypes = [vp, C.c_int32]
        L.oracle_ba_set_linear_solver.argtypes = [vp, C.c_int32]
        L.oracle_ba_export_preconditioner_blocks.argtypes = [vp, vp, C.c_size_t]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_ba_num_threads())


def _f64(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def rotation(w) -> np.ndarray:
    w = _f64(w)
    out = np.empty(9)
    lib().oracle_ba_rotation(w.ctypes.data, out.ctypes.data)
    return out.reshape(3, 3)


def observation(cam, pt, pixel, jacobians: bool = True):
    cam, pt, pixel = _f64(cam), _f64(pt), _f64(pixel)
    r, jc, jp = np.empty(2), np.empty(18), np.empty(6)
    lib().oracle_ba_observation(cam.ctypes.data, pt.ctypes.data, pixel.ctypes.data, r.ctypes.data,
                                jc.ctypes.data if jacobians else None, jp.ctypes.data if jacobians else None)
    return (r, jc.reshape(2, 9), jp.reshape(2, 3)) if jacobians else r


def observation_model(camera_model: int, depth_epsilon: float, cam, pt, pixel, jacobians: bool = True):
    cam, pt, pixel = _f64(cam), _f64(pt), _f64(pixel)
    r, jc, jp = np.empty(2), np.empty(18), np.empty(6)
    lib().oracle_ba_observation_model(int(camera_model), float(depth_epsilon), cam.ctypes.data, pt.ctypes.data,
                                      pixel.ctypes.data, r.ctypes.data, jc.ctypes.data if jacobians else None,
                                      jp.ctypes.data if jacobians else None)
    return (r, jc.reshape(2, 9), jp.reshape(2, 3)) if jacobians else r


def retract_camera(camera_model: int, cam, delta) -> np.ndarray:
    cam, delta = _f64(cam), _f64(delta)
    out = np.empty(9)
    lib().oracle_ba_retract_camera(int(camera_model), cam.ctypes.data, delta.ctypes.data, out.ctypes.data)
    return out


def spd_inverse(a) -> Tuple[int, np.ndarray]:
    a = _f64(a)
    n = a.shape[0]
    inv = np.empty((n, n))
    rc = lib().oracle_ba_spd_inverse(n, a.ctypes.data, inv.ctypes.data)
    return rc, inv


class OracleError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"oracle_ba: {where} returned {code}")
        self.code = code


class OracleBA:
    """fp64 oracle handle.  Takes the (float32) scene arrays, up-casts them to float64 copies it owns."""

    def __init__(self, cameras, points, observations, camera_index, point_index, robust_loss: int = 0,
                 robust_scale: float = 0.0, damping_mode: int = 0, camera_model: int = 0, depth_epsilon: float = 0.0):
        self.cameras = _f64(cameras).copy().reshape(-1, 9)
        self.points = _f64(points).copy().reshape(-1, 3)
        self.observations = _f64(observations).copy().reshape(-1, 2)
        self.camera_index = np.ascontiguousarray(np.asarray(camera_index, dtype=np.int32))
        self.point_index = np.ascontiguousarray(np.asarray(point_index, dtype=np.int32))
        self.nc, self.np_, self.n = self.cameras.shape[0], self.points.shape[0], self.observations.shape[0]
        pb = _Problem(self.nc, self.np_, self.n, self.cameras.ctypes.data, self.points.ctypes.data,
                      self.observations.ctypes.data, self.camera_index.ctypes.data, self.point_index.ctypes.data,
                      int(robust_loss), float(robust_scale), int(damping_mode), int(camera_model), float(depth_epsilon))
        self._h = C.c_void_p()
        rc = lib().oracle_ba_create(C.byref(pb), C.byref(self._h))
        if rc:
            self._h = None
            raise OracleError(rc, "create")

    @classmethod
    def from_scene(cls, scene, damping_mode: int = 0, robust_loss: Optional[int] = None,
                   robust_scale: Optional[float] = None, camera_model: int = 0, depth_epsilon: float = 0.0) -> "OracleBA":
        return cls(scene.cameras, scene.points, scene.observations, scene.camera_index, scene.point_index,
                   scene.robust_loss if robust_loss is None else robust_loss,
                   scene.robust_scale if robust_scale is None else robust_scale, damping_mode, camera_model,
                   depth_epsilon)

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:   # (_lib is gone at interpreter shutdown)
            _lib.oracle_ba_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, rc: int, where: str):
        if rc:
            raise OracleError(rc, where)

    def linearize(self) -> float:
        cost = C.c_double()
        self._check(lib().oracle_ba_linearize(self._h, C.byref(cost)), "linearize")
        return cost.value

    def cost(self) -> float:
        cost = C.c_double()
        self._check(lib().oracle_ba_cost(self._h, C.byref(cost)), "cost")
        return cost.value

    def pcg_solve(self, lam: float, rel_tol: float, max_iter: int) -> PcgInfo:
        info = PcgInfo()
        self._check(lib().oracle_ba_pcg_solve(self._h, lam, rel_tol, max_iter, C.byref(info)), "pcg_solve")
        return info

    def pcgnr_solve(self, lam: float, rel_tol: float, max_iter: int) -> PcgInfo:
        info = PcgInfo()
        self._check(lib().oracle_ba_pcgnr_solve(self._h, lam, rel_tol, max_iter, C.byref(info)), "pcgnr_solve")
        return info

    def set_preconditioner(self, mode: int):
        self._check(lib().oracle_ba_set_preconditioner(self._h, int(mode)), "set_preconditioner")

    def set_linear_solver(self, mode: int):
        self._check(lib().oracle_ba_set_linear_solver(self._h, int(mode)), "set_linear_solver")

    def preconditioner_blocks(self) -> np.ndarray:
        out = np.empty((self.nc, 9, 9))
        self._check(lib().oracle_ba_export_preconditioner_blocks(self._h, out.ctypes.data, out.size),
                    "export_preconditioner_blocks")
        return out

    def lm_step(self, lam: float, rel_tol: float, max_iter: int, accept_mode: int = 0) -> Step:
        info = StepInfo()
        self._check(lib().oracle_ba_lm_step(self._h, lam, rel_tol, max_iter, accept_mode, C.byref(info)), "lm_step")
        return _step(info, lam)

    def solve(self, iterations: int, lambda0: float, rel_tol: float, max_iter: int) -> List[Step]:
        infos = (StepInfo * max(1, iterations))()
        lams = np.zeros(max(1, iterations))
        self._check(lib().oracle_ba_solve(self._h, iterations, lambda0, rel_tol, max_iter, infos,
                                          lams.ctypes.data_as(C.POINTER(C.c_double))), "solve")
        return [_step(infos[i], float(lams[i])) for i in range(iterations)]

    def export(self, what: int) -> np.ndarray:
        nc, np_, n = self.nc, self.np_, self.n
        shape = {RESIDUALS: (n, 2), JC: (n, 2, 9), JP: (n, 2, 3), U: (nc, 9, 9), V: (np_, 3, 3),
                 G: (9 * nc + 3 * np_,), SCHUR_RHS: (9 * nc,), DELTA: (9 * nc + 3 * np_,),
                 DAMPING: (9 * nc + 3 * np_,)}[what]
        out = np.empty(shape)
        self._check(lib().oracle_ba_export(self._h, what, out.ctypes.data, out.size), f"export({what})")
        return out

    def schur_matvec(self, lam: float, p) -> np.ndarray:
        p = _f64(p)
        q = np.empty_like(p)
        self._check(lib().oracle_ba_schur_matvec(self._h, lam, p.ctypes.data, q.ctypes.data), "schur_matvec")
        return q

    def full_matvec(self, lam: float, x) -> np.ndarray:
        x = _f64(x)
        y = np.empty_like(x)
        self._check(lib().oracle_ba_full_matvec(self._h, lam, x.ctypes.data, y.ctypes.data), "full_matvec")
        return y
