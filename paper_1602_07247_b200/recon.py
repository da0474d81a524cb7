"""Thin ctypes binding of include/ants_recon.h (argument marshalling only).

Every reconstruction step runs in the CUDA kernels behind the C ABI; this
module never computes anything itself and there is no CPU fallback: a missing
library or a missing GPU raises.  torch is used for device memory and streams.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libants_recon.so")

POISSON_ML, CHI_SQUARE, CHI_SQUARE_SUMRATIO = 0, 1, 2


class AntsError(RuntimeError):
    def __init__(self, status: int, what: str):
        super().__init__(f"{what}: {strerror(status)} (status {status})")
        self.status = status


class LrfDims(C.Structure):
    _fields_ = [("n_sensors", C.c_int32), ("n_lrf", C.c_int32), ("lrf_dim", C.c_int32),
                ("n_int_r", C.c_int32), ("n_int_z", C.c_int32)]


class GridParams(C.Structure):
    _fields_ = [("dim", C.c_int32), ("nodes_per_axis", C.c_int32), ("step0_xy", C.c_float),
                ("step0_z", C.c_float), ("factor", C.c_float), ("n_iter", C.c_int32),
                ("seed_mode", C.c_int32), ("z_seed", C.c_float)]


class FilterCriteria(C.Structure):
    _fields_ = [("score_max", C.c_float), ("energy_min", C.c_float), ("energy_max", C.c_float),
                ("radius_max", C.c_float)]


_lib = None


def load():
    """dlopen the in-tree library (building it if nvcc is there and it is missing)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from . import build as _build
        _build.build()
    lib = C.CDLL(LIB_PATH)
    vp, i32p = C.c_void_p, C.POINTER(C.c_int32)
    lib.ants_lrf_create.restype = C.c_int
    lib.ants_lrf_create.argtypes = [vp, vp, vp, vp, C.POINTER(LrfDims), C.POINTER(vp)]
    lib.ants_reconstruct.restype = C.c_int
    lib.ants_reconstruct.argtypes = [vp, vp, C.c_int64, C.POINTER(GridParams), C.c_int32, vp, vp, vp]
    lib.ants_reconstruct_trace.restype = C.c_int
    lib.ants_reconstruct_trace.argtypes = [vp, vp, C.c_int64, C.POINTER(GridParams), C.c_int32, vp, vp, vp, vp]
    lib.ants_reconstruct_host.restype = C.c_int
    lib.ants_reconstruct_host.argtypes = [vp, vp, C.c_int64, C.POINTER(GridParams), C.c_int32, vp, vp, C.c_int64]
    lib.ants_lrf_set_selection.restype = C.c_int
    lib.ants_lrf_set_selection.argtypes = [vp, vp, C.c_float, C.c_float]
    lib.ants_lrf_fit_axial.restype = C.c_int
    lib.ants_lrf_fit_axial.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, vp, vp, C.c_int64, vp, vp, vp]
    lib.ants_lrf_fit_gains.restype = C.c_int
    lib.ants_lrf_fit_gains.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, vp, vp, C.c_int64, vp, vp, vp]
    lib.ants_lrf_fit_axial_grouped.restype = C.c_int
    lib.ants_lrf_fit_axial_grouped.argtypes = [vp, vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, vp, vp, C.c_int64, vp, vp, vp]
    lib.ants_lrf_fit_axial_z.restype = C.c_int
    lib.ants_lrf_fit_axial_z.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, vp, vp, C.c_int64, vp, vp, vp]
    lib.ants_filter_events.restype = C.c_int
    lib.ants_filter_events.argtypes = [vp, vp, C.c_int64, C.POINTER(FilterCriteria), C.POINTER(C.c_int64), vp]
    lib.ants_destroy.restype = None
    lib.ants_destroy.argtypes = [vp]
    lib.ants_strerror.restype = C.c_char_p
    lib.ants_strerror.argtypes = [C.c_int]
    lib.ants_launch_count.restype = C.c_int64
    lib.ants_launch_count.argtypes = []
    lib.ants_plan_info.restype = C.c_int
    lib.ants_plan_info.argtypes = [vp, C.POINTER(GridParams), C.c_int32, i32p, i32p, i32p, i32p, i32p]
    _lib = lib
    return lib


def strerror(status: int) -> str:
    return load().ants_strerror(int(status)).decode()


def launch_count() -> int:
    return int(load().ants_launch_count())


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def ants_lrf_create(sensor_xy, gains, knots, coeffs, dims: LrfDims) -> int:
    """-> opaque handle (int).  Arrays are host float32; gains may be None."""
    xy, kn, co = _f32(sensor_xy), _f32(knots), _f32(coeffs)
    g = None if gains is None else _f32(gains)
    out = C.c_void_p()
    rc = load().ants_lrf_create(xy.ctypes.data, None if g is None else g.ctypes.data, kn.ctypes.data,
                                co.ctypes.data, C.byref(dims), C.byref(out))
    if rc != 0:
        raise AntsError(rc, "ants_lrf_create")
    return out.value


def ants_lrf_set_selection(handle, passive=None, signal_min=float("nan"), dist_max=float("nan")) -> None:
    """passive: host bool/uint8 [N] or None; signal_min / dist_max: NaN = off (include/ants_recon.h)."""
    pm = None if passive is None else np.ascontiguousarray(np.asarray(passive) != 0, dtype=np.uint8)
    rc = load().ants_lrf_set_selection(handle, None if pm is None else pm.ctypes.data, float(signal_min),
                                       float(dist_max))
    if rc != 0:
        raise AntsError(rc, "ants_lrf_set_selection")


def ants_filter_events(xyzA, score, score_max=float("nan"), energy_min=float("nan"), energy_max=float("nan"),
                       radius_max=float("nan"), stream=None) -> int:
    """Event filters (include/ants_recon.h): rejected rows of the CUDA tensor xyzA become NaN in place.
    -> number of passing events."""
    import torch
    for t in (xyzA, score):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_filter_events needs contiguous float32 CUDA tensors")
    E = int(score.shape[0])
    if tuple(xyzA.shape) != (E, 4):
        raise ValueError("ants_filter_events: shape mismatch")
    crit = FilterCriteria(score_max, energy_min, energy_max, radius_max)
    n_pass = C.c_int64(0)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_filter_events(xyzA.data_ptr(), score.data_ptr(), E, C.byref(crit), C.byref(n_pass), st)
    if rc != 0:
        raise AntsError(rc, "ants_filter_events")
    return int(n_pass.value)


def ants_lrf_fit_axial(sensor_xy, gains, knots, n_lrf: int, n_int_r: int, signals, xyzA, stream=None, group=None):
    """LRF calculation (include/ants_recon.h): signals [E][N] and xyzA [E][4] are CUDA float32 tensors.
    -> (coeffs float32 [n_lrf][n_int_r + 3], pairs used per table float64 [n_lrf])."""
    import torch
    xy, kn = _f32(sensor_xy).reshape(-1, 2), _f32(knots)
    N = xy.shape[0]
    g = None if gains is None else _f32(gains)
    for t in (signals, xyzA):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_lrf_fit_axial needs contiguous float32 CUDA tensors")
    E = int(signals.shape[0])
    if signals.shape[1] != N or tuple(xyzA.shape) != (E, 4):
        raise ValueError("ants_lrf_fit_axial: shape mismatch")
    coeffs = np.zeros((int(n_lrf), int(n_int_r) + 3), np.float32)
    used = np.zeros(int(n_lrf), np.float64)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    if group is None:
        rc = load().ants_lrf_fit_axial(xy.ctypes.data, None if g is None else g.ctypes.data, kn.ctypes.data, N,
                                       int(n_lrf), int(n_int_r), signals.data_ptr(), xyzA.data_ptr(), E,
                                       coeffs.ctypes.data, used.ctypes.data, st)
    else:       # explicit grouping (R28): n_lrf = number of groups
        gr = np.ascontiguousarray(np.asarray(group, dtype=np.int32))
        rc = load().ants_lrf_fit_axial_grouped(xy.ctypes.data, None if g is None else g.ctypes.data, gr.ctypes.data,
                                               kn.ctypes.data, N, int(n_lrf), int(n_int_r), signals.data_ptr(),
                                               xyzA.data_ptr(), E, coeffs.ctypes.data, used.ctypes.data, st)
    if rc != 0:
        raise AntsError(rc, "ants_lrf_fit_axial")
    return coeffs, used


def ants_lrf_fit_axial_z(sensor_xy, gains, knots, n_int_r: int, n_int_z: int, signals, xyzA, stream=None):
    """Axial+z tensor LRF calculation (include/ants_recon.h).  -> (coeffs float32 [n_int_z+3][n_int_r+3], pairs used)."""
    import torch
    xy, kn = _f32(sensor_xy).reshape(-1, 2), _f32(knots)
    N, E = xy.shape[0], int(signals.shape[0])
    g = None if gains is None else _f32(gains)
    for t in (signals, xyzA):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_lrf_fit_axial_z needs contiguous float32 CUDA tensors")
    if signals.shape[1] != N or tuple(xyzA.shape) != (E, 4) or kn.size < 4:
        raise ValueError("ants_lrf_fit_axial_z: shape mismatch")
    coeffs = np.zeros((int(n_int_z) + 3, int(n_int_r) + 3), np.float32)
    used = C.c_double(0.0)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_lrf_fit_axial_z(xy.ctypes.data, None if g is None else g.ctypes.data, kn.ctypes.data, N,
                                     int(n_int_r), int(n_int_z), signals.data_ptr(), xyzA.data_ptr(), E,
                                     coeffs.ctypes.data, C.addressof(used), st)
    if rc != 0:
        raise AntsError(rc, "ants_lrf_fit_axial_z")
    return coeffs, used.value


def ants_lrf_fit_gains(sensor_xy, knots, coeffs, signals, xyzA, stream=None):
    """Relative gains for a fixed shared profile (include/ants_recon.h).  -> (gains float32 [N], pairs [N])."""
    import torch
    xy, kn, co = _f32(sensor_xy).reshape(-1, 2), _f32(knots), _f32(coeffs).reshape(-1)
    N, E = xy.shape[0], int(signals.shape[0])
    for t in (signals, xyzA):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_lrf_fit_gains needs contiguous float32 CUDA tensors")
    if signals.shape[1] != N or tuple(xyzA.shape) != (E, 4):
        raise ValueError("ants_lrf_fit_gains: shape mismatch")
    gains, used = np.zeros(N, np.float32), np.zeros(N, np.float64)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_lrf_fit_gains(xy.ctypes.data, kn.ctypes.data, co.ctypes.data, N, co.size - 3, signals.data_ptr(),
                                   xyzA.data_ptr(), E, gains.ctypes.data, used.ctypes.data, st)
    if rc != 0:
        raise AntsError(rc, "ants_lrf_fit_gains")
    return gains, used


def group_by_radius(sensor_xy, tol: float = 1e-3):
    """Sensor groups "according to the distance from the sensor center to the detector center":
    sensors are sorted by their distance from the origin and a new group starts wherever the distance exceeds
    the group's first one by more than tol (mm).  -> (group int32 [N], n_groups), for ants_lrf_fit_axial(group=)."""
    xy = _f32(sensor_xy).reshape(-1, 2).astype(np.float64)
    dist = np.sqrt((xy * xy).sum(axis=1))
    order = np.argsort(dist, kind="stable")
    group = np.empty(len(dist), np.int32)
    current, anchor = -1, -np.inf
    for i in order:
        if dist[i] - anchor > tol:
            current, anchor = current + 1, dist[i]
        group[i] = current
    return group, current + 1


def expand_groups(coeffs, group, gains):
    """A grouped response as one table per sensor (what ants_lrf_create takes with n_lrf = N): the table of
    sensor i is its group's profile times its relative gain.  -> float32 [N][1][n_int_r + 3]."""
    c = np.asarray(coeffs, np.float64)[np.asarray(group)] * np.asarray(gains, np.float64)[:, None]
    return c.astype(np.float32)[:, None, :]


def ants_destroy(handle) -> None:
    load().ants_destroy(handle)


def ants_reconstruct(handle, signals, grid: GridParams, method: int, out_xyzA, out_score,
                     stream=None, out_path=None) -> None:
    """signals/out_*: CUDA torch tensors (float32, contiguous; out_path int16/uint16 [E][K])."""
    import torch
    E = int(signals.shape[0]) if signals.dim() == 2 else 0
    for t in (signals, out_xyzA, out_score) + (() if out_path is None else (out_path,)):
        if not (t.is_cuda and t.is_contiguous()):
            raise ValueError("ants_reconstruct needs contiguous CUDA tensors")
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    if out_path is None:
        rc = load().ants_reconstruct(handle, signals.data_ptr(), E, C.byref(grid), int(method),
                                     out_xyzA.data_ptr(), out_score.data_ptr(), st)
    else:
        rc = load().ants_reconstruct_trace(handle, signals.data_ptr(), E, C.byref(grid), int(method),
                                           out_xyzA.data_ptr(), out_score.data_ptr(), out_path.data_ptr(), st)
    if rc != 0:
        raise AntsError(rc, "ants_reconstruct")


def ants_reconstruct_host(handle, signals, grid: GridParams, method: int, out_xyzA, out_score,
                          chunk_events: int = 0) -> None:
    """signals/out_*: host buffers (numpy arrays or CPU torch tensors, pinned for async copies)."""
    def ptr(a):
        return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
    rc = load().ants_reconstruct_host(handle, ptr(signals), int(signals.shape[0]), C.byref(grid), int(method),
                                      ptr(out_xyzA), ptr(out_score), int(chunk_events))
    if rc != 0:
        raise AntsError(rc, "ants_reconstruct_host")


def plan_info(handle, grid: GridParams, method: int) -> dict:
    v = [C.c_int32() for _ in range(5)]
    rc = load().ants_plan_info(handle, C.byref(grid), int(method), *[C.byref(x) for x in v])
    if rc != 0:
        raise AntsError(rc, "ants_plan_info")
    keys = ("first_diff_iter", "nodes_per_lane", "warps_per_cta", "ctas_per_sm", "smem_bytes")
    return dict(zip(keys, (x.value for x in v)))


class Reconstructor:
    """Convenience owner of one LRF handle built from a synth.Config-like record."""

    def __init__(self, cfg):
        self.cfg = cfg
        self.dims = LrfDims(cfg.n_sensors, cfg.n_lrf, cfg.lrf_dim, cfg.n_int_r, cfg.n_int_z)
        self.grid = GridParams(cfg.dim, cfg.nodes_per_axis, cfg.step0_xy, cfg.step0_z, cfg.factor,
                               cfg.n_iter, int(getattr(cfg, "seed_mode", 0)), cfg.z_seed)
        self.method = int(cfg.method)
        self.handle = ants_lrf_create(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.coeffs, self.dims)
        passive = getattr(cfg, "passive", None)
        smin, dmax = getattr(cfg, "signal_min", float("nan")), getattr(cfg, "dist_max", float("nan"))
        if passive is not None or smin == smin or dmax == dmax:
            ants_lrf_set_selection(self.handle, passive, smin, dmax)

    def __call__(self, signals, trace: bool = False, stream=None):
        import torch
        E = signals.shape[0]
        xyzA = torch.empty((E, 4), dtype=torch.float32, device=signals.device)
        score = torch.empty((E,), dtype=torch.float32, device=signals.device)
        path = torch.empty((E, self.grid.n_iter), dtype=torch.int16, device=signals.device) if trace else None
        ants_reconstruct(self.handle, signals, self.grid, self.method, xyzA, score, stream, path)
        return (xyzA, score, path) if trace else (xyzA, score)

    def plan(self) -> dict:
        return plan_info(self.handle, self.grid, self.method)

    def close(self):
        if self.handle:
            ants_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
