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


class LrfXY(C.Structure):
    _fields_ = [("n_int_x", C.c_int32), ("n_int_y", C.c_int32), ("n_planes", C.c_int32),
                ("knots_xy", C.c_void_p), ("coeffs_xy", C.c_void_p), ("xform", C.c_void_p), ("group", C.c_void_p)]


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
    lib.ants_lrf_create_grouped.restype = C.c_int
    lib.ants_lrf_create_grouped.argtypes = [vp, vp, vp, vp, vp, C.POINTER(LrfDims), C.POINTER(vp)]
    lib.ants_lrf_create_xy.restype = C.c_int
    lib.ants_lrf_create_xy.argtypes = [vp, vp, vp, vp, C.POINTER(LrfDims), C.POINTER(LrfXY), C.POINTER(vp)]
    lib.ants_group_by_symmetry.restype = C.c_int
    lib.ants_group_by_symmetry.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_float, vp, vp, i32p]
    lib.ants_group_by_radius.restype = C.c_int
    lib.ants_group_by_radius.argtypes = [vp, C.c_int32, C.c_float, vp, i32p]
    lib.ants_gains_renormalise.restype = C.c_int
    lib.ants_gains_renormalise.argtypes = [vp, vp, C.c_int32, vp]
    lib.ants_lrf_n_sensors.restype = C.c_int32
    lib.ants_lrf_n_sensors.argtypes = [vp]
    lib.ants_plan_kernel_name.restype = C.c_int
    lib.ants_plan_kernel_name.argtypes = [vp, C.POINTER(GridParams), C.c_int32, C.c_char_p, C.c_int32]
    lib.ants_probe_throughput.restype = C.c_int
    lib.ants_probe_throughput.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.ants_lrf_fit_sliced.restype = C.c_int
    lib.ants_lrf_fit_sliced.argtypes = [vp, vp, vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp,
                                        C.c_int64, vp, vp, vp]
    lib.ants_lrf_fit_xy.restype = C.c_int
    lib.ants_lrf_fit_xy.argtypes = [vp, vp, vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, C.c_int32,
                                    vp, vp, C.c_int64, vp, vp, vp]
    lib.ants_refine.restype = C.c_int
    lib.ants_refine.argtypes = [vp, vp, C.c_int64, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp]
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
    lib.ants_lrf_fit_gains_static.restype = C.c_int
    lib.ants_lrf_fit_gains_static.argtypes = lib.ants_lrf_fit_gains.argtypes
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


def ants_lrf_create_grouped(sensor_xy, gains, group, knots, coeffs, dims: LrfDims) -> int:
    """Grouped model (include/ants_recon.h): dims.n_lrf = number of groups, group int32 [N],
    coeffs [n_groups][n_int_r + 3].  -> opaque handle (int)."""
    xy, kn, co = _f32(sensor_xy), _f32(knots), _f32(coeffs)
    g = None if gains is None else _f32(gains)
    gr = np.ascontiguousarray(np.asarray(group, dtype=np.int32))
    out = C.c_void_p()
    rc = load().ants_lrf_create_grouped(xy.ctypes.data, None if g is None else g.ctypes.data, gr.ctypes.data,
                                        kn.ctypes.data, co.ctypes.data, C.byref(dims), C.byref(out))
    if rc != 0:
        raise AntsError(rc, "ants_lrf_create_grouped")
    return out.value


def ants_lrf_create_xy(sensor_xy, gains, knots, coeffs, dims: LrfDims, n_int_x: int, n_int_y: int, n_planes: int,
                       knots_xy, coeffs_xy, xform=None, group=None) -> int:
    """XY / Composite / Sliced model (include/ants_recon.h, dims.lrf_dim = 3 / 4 / 5).  knots and coeffs describe
    the axial component of a Composite model (None otherwise).  -> opaque handle (int)."""
    xy, kxy, cxy = _f32(sensor_xy), _f32(knots_xy), _f32(coeffs_xy)
    g = None if gains is None else _f32(gains)
    kn = None if knots is None else _f32(knots)
    co = None if coeffs is None or np.size(coeffs) == 0 else _f32(coeffs)
    xf = None if xform is None else _f32(xform)
    gr = None if group is None else np.ascontiguousarray(np.asarray(group, dtype=np.int32))
    n_tab = int(dims.n_lrf)
    if cxy.size != n_tab * max(int(n_planes), 1) * (int(n_int_x) + 3) * (int(n_int_y) + 3) or kxy.size < (6 if dims.lrf_dim == 5 else 4):
        raise ValueError("ants_lrf_create_xy: coeffs_xy / knots_xy size mismatch")
    if xf is not None and xf.size != 4 * xy.size // 2:
        raise ValueError("ants_lrf_create_xy: xform must be [N][4]")
    desc = LrfXY(int(n_int_x), int(n_int_y), int(n_planes), kxy.ctypes.data, cxy.ctypes.data,
                 None if xf is None else xf.ctypes.data, None if gr is None else gr.ctypes.data)
    out = C.c_void_p()
    rc = load().ants_lrf_create_xy(xy.ctypes.data, None if g is None else g.ctypes.data,
                                   None if kn is None else kn.ctypes.data, None if co is None else co.ctypes.data,
                                   C.byref(dims), C.byref(desc), C.byref(out))
    if rc != 0:
        raise AntsError(rc, "ants_lrf_create_xy")
    return out.value


def ants_group_by_symmetry(sensor_xy, n_fold: int, reflect: bool = True, tol: float = 1e-3):
    """Symmetry groups and per-sensor frames (include/ants_recon.h).  -> (group int32 [N], xform float32 [N][4], n_groups)."""
    xy = _f32(sensor_xy).reshape(-1, 2)
    group = np.zeros(xy.shape[0], np.int32)
    xform = np.zeros((xy.shape[0], 4), np.float32)
    n = C.c_int32(0)
    rc = load().ants_group_by_symmetry(xy.ctypes.data, xy.shape[0], int(n_fold), int(bool(reflect)), float(tol),
                                       group.ctypes.data, xform.ctypes.data, C.byref(n))
    if rc != 0:
        raise AntsError(rc, "ants_group_by_symmetry")
    return group, xform, int(n.value)


def ants_group_by_radius(sensor_xy, tol: float = 1e-3):
    """Distance-from-centre sensor groups (include/ants_recon.h).  -> (group int32 [N], n_groups)."""
    xy = _f32(sensor_xy).reshape(-1, 2)
    group = np.zeros(xy.shape[0], np.int32)
    n = C.c_int32(0)
    rc = load().ants_group_by_radius(xy.ctypes.data, xy.shape[0], float(tol), group.ctypes.data, C.byref(n))
    if rc != 0:
        raise AntsError(rc, "ants_group_by_radius")
    return group, int(n.value)


def ants_gains_renormalise(gains_new, gains_prev):
    """Relative gains carried on at the scale of the previous set (include/ants_recon.h).  -> float32 [N]."""
    gn, gp = _f32(gains_new).reshape(-1), _f32(gains_prev).reshape(-1)
    if gn.size != gp.size:
        raise ValueError("ants_gains_renormalise: size mismatch")
    out = np.zeros(gn.size, np.float32)
    rc = load().ants_gains_renormalise(gn.ctypes.data, gp.ctypes.data, gn.size, out.ctypes.data)
    if rc != 0:
        raise AntsError(rc, "ants_gains_renormalise")
    return out


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


def ants_lrf_fit_xy(sensor_xy, gains, knots_xy, n_lrf: int, n_int_x: int, n_int_y: int, signals, xyzA, group=None,
                    xform=None, axial=None, stream=None):
    """XY / Composite-residual LRF calculation (include/ants_recon.h).  axial = (knots_ax, coeffs_ax [n_lrf][n_r+3])
    for the Composite residual fit.  -> (coeffs float32 [n_lrf][n_int_y+3][n_int_x+3], pairs used float64 [n_lrf])."""
    import torch
    xy, kn = _f32(sensor_xy).reshape(-1, 2), _f32(knots_xy)
    N, E = xy.shape[0], int(signals.shape[0])
    g = None if gains is None else _f32(gains)
    gr = None if group is None else np.ascontiguousarray(np.asarray(group, dtype=np.int32))
    xf = None if xform is None else _f32(xform).reshape(N, 4)
    for t in (signals, xyzA):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_lrf_fit_xy needs contiguous float32 CUDA tensors")
    if signals.shape[1] != N or tuple(xyzA.shape) != (E, 4) or kn.size < 4:
        raise ValueError("ants_lrf_fit_xy: shape mismatch")
    ka = ca = None
    n_r = 0
    if axial is not None:
        ka, ca = _f32(axial[0]), _f32(axial[1]).reshape(int(n_lrf), -1)
        n_r = ca.shape[1] - 3
    coeffs = np.zeros((int(n_lrf), int(n_int_y) + 3, int(n_int_x) + 3), np.float32)
    used = np.zeros(int(n_lrf), np.float64)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_lrf_fit_xy(xy.ctypes.data, None if g is None else g.ctypes.data, None if gr is None else gr.ctypes.data,
                                None if xf is None else xf.ctypes.data, kn.ctypes.data, N, int(n_lrf), int(n_int_x),
                                int(n_int_y), None if ka is None else ka.ctypes.data, None if ca is None else ca.ctypes.data,
                                int(n_r), signals.data_ptr(), xyzA.data_ptr(), E, coeffs.ctypes.data, used.ctypes.data, st)
    if rc != 0:
        raise AntsError(rc, "ants_lrf_fit_xy")
    return coeffs, used


def ants_lrf_fit_sliced(sensor_xy, gains, knots_xy, n_lrf: int, n_int_x: int, n_int_y: int, n_planes: int, signals, xyzA,
                        group=None, xform=None, stream=None):
    """Sliced LRF calculation, all planes of a table jointly (include/ants_recon.h).
    -> (coeffs float32 [n_lrf][n_planes][n_int_y+3][n_int_x+3], pairs used float64 [n_lrf])."""
    import torch
    xy, kn = _f32(sensor_xy).reshape(-1, 2), _f32(knots_xy)
    N, E = xy.shape[0], int(signals.shape[0])
    g = None if gains is None else _f32(gains)
    gr = None if group is None else np.ascontiguousarray(np.asarray(group, dtype=np.int32))
    xf = None if xform is None else _f32(xform).reshape(N, 4)
    for t in (signals, xyzA):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_lrf_fit_sliced needs contiguous float32 CUDA tensors")
    if signals.shape[1] != N or tuple(xyzA.shape) != (E, 4) or kn.size < 6:
        raise ValueError("ants_lrf_fit_sliced: shape mismatch")
    coeffs = np.zeros((int(n_lrf), int(n_planes), int(n_int_y) + 3, int(n_int_x) + 3), np.float32)
    used = np.zeros(int(n_lrf), np.float64)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_lrf_fit_sliced(xy.ctypes.data, None if g is None else g.ctypes.data,
                                    None if gr is None else gr.ctypes.data, None if xf is None else xf.ctypes.data,
                                    kn.ctypes.data, N, int(n_lrf), int(n_int_x), int(n_int_y), int(n_planes),
                                    signals.data_ptr(), xyzA.data_ptr(), E, coeffs.ctypes.data, used.ctypes.data, st)
    if rc != 0:
        raise AntsError(rc, "ants_lrf_fit_sliced")
    return coeffs, used


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



def ants_lrf_fit_gains_static(sensor_xy, knots, coeffs, signals, xyzA, stream=None):
    """ants_lrf_fit_gains without any allocation inside the library (include/ants_recon.h): scratch in a fixed 8 KB
    device array, N <= 128, len(coeffs) <= 1024.  -> (gains float32 [N], pairs [N])."""
    import torch
    xy, kn, co = _f32(sensor_xy).reshape(-1, 2), _f32(knots), _f32(coeffs).reshape(-1)
    N, E = xy.shape[0], int(signals.shape[0])
    for t in (signals, xyzA):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_lrf_fit_gains_static needs contiguous float32 CUDA tensors")
    if signals.shape[1] != N or tuple(xyzA.shape) != (E, 4):
        raise ValueError("ants_lrf_fit_gains_static: shape mismatch")
    gains, used = np.zeros(N, np.float32), np.zeros(N, np.float64)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_lrf_fit_gains_static(xy.ctypes.data, kn.ctypes.data, co.ctypes.data, N, co.size - 3,
                                          signals.data_ptr(), xyzA.data_ptr(), E, gains.ctypes.data, used.ctypes.data, st)
    if rc != 0:
        raise AntsError(rc, "ants_lrf_fit_gains_static")
    return gains, used

def ants_destroy(handle) -> None:
    load().ants_destroy(handle)


def ants_reconstruct(handle, signals, grid: GridParams, method: int, out_xyzA, out_score,
                     stream=None, out_path=None) -> None:
    """signals [E][N], out_xyzA [E][4], out_score [E]: contiguous float32 CUDA tensors;
    out_path (optional) [E][K] int16/uint16.  Shapes and dtypes are checked here: the C side only sees pointers."""
    import torch
    N = int(load().ants_lrf_n_sensors(handle))
    if signals.dim() != 2 or int(signals.shape[1]) != N:
        raise ValueError(f"ants_reconstruct: signals must be [E][{N}]")
    E = int(signals.shape[0])
    for t in (signals, out_xyzA, out_score):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_reconstruct needs contiguous float32 CUDA tensors")
    if tuple(out_xyzA.shape) != (E, 4) or tuple(out_score.shape) != (E,):
        raise ValueError("ants_reconstruct: out_xyzA must be [E][4] and out_score [E]")
    if out_path is not None:
        if not (out_path.is_cuda and out_path.is_contiguous() and out_path.element_size() == 2 and
                not out_path.dtype.is_floating_point and tuple(out_path.shape) == (E, int(grid.n_iter))):
            raise ValueError("ants_reconstruct: out_path must be a contiguous 16-bit integer CUDA tensor [E][K]")
    if len({t.device for t in (signals, out_xyzA, out_score)}) != 1:
        raise ValueError("ants_reconstruct: tensors on different devices")
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    if out_path is None:
        rc = load().ants_reconstruct(handle, signals.data_ptr(), E, C.byref(grid), int(method),
                                     out_xyzA.data_ptr(), out_score.data_ptr(), st)
    else:
        rc = load().ants_reconstruct_trace(handle, signals.data_ptr(), E, C.byref(grid), int(method),
                                           out_xyzA.data_ptr(), out_score.data_ptr(), out_path.data_ptr(), st)
    if rc != 0:
        raise AntsError(rc, "ants_reconstruct")


def ants_refine(handle, signals, method: int, xyzA, score, n_steps: int, dim: int = 2, seed_mode: int = 0,
                stream=None) -> None:
    """Continuous refinement in place (include/ants_recon.h): xyzA [E][4] holds the start positions on entry and the
    refined positions and energies on return; score [E] receives the scores.  Contiguous float32 CUDA tensors."""
    import torch
    N = int(load().ants_lrf_n_sensors(handle))
    if signals.dim() != 2 or int(signals.shape[1]) != N:
        raise ValueError(f"ants_refine: signals must be [E][{N}]")
    E = int(signals.shape[0])
    for t in (signals, xyzA, score):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
            raise ValueError("ants_refine needs contiguous float32 CUDA tensors")
    if tuple(xyzA.shape) != (E, 4) or tuple(score.shape) != (E,):
        raise ValueError("ants_refine: xyzA must be [E][4] and score [E]")
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = load().ants_refine(handle, signals.data_ptr(), E, int(method), int(dim), int(seed_mode), int(n_steps),
                            xyzA.data_ptr(), score.data_ptr(), st)
    if rc != 0:
        raise AntsError(rc, "ants_refine")


def _host_f32(a, shape, what):
    """pointer of a C-contiguous float32 host buffer (numpy array or CPU torch tensor) of the given shape"""
    if hasattr(a, "data_ptr"):
        import torch
        ok = (not a.is_cuda) and a.is_contiguous() and a.dtype == torch.float32 and tuple(a.shape) == shape
        ptr = a.data_ptr()
    else:
        ok = isinstance(a, np.ndarray) and a.flags["C_CONTIGUOUS"] and a.dtype == np.float32 and a.shape == shape
        ptr = a.ctypes.data if ok else 0
    if not ok:
        raise ValueError(f"ants_reconstruct_host: {what} must be a C-contiguous float32 host buffer of shape {shape}")
    return ptr


def ants_reconstruct_host(handle, signals, grid: GridParams, method: int, out_xyzA, out_score,
                          chunk_events: int = 0) -> None:
    """signals [E][N], out_xyzA [E][4], out_score [E]: host buffers (numpy arrays or CPU torch tensors,
    pinned for asynchronous copies)."""
    N = int(load().ants_lrf_n_sensors(handle))
    E = int(signals.shape[0])
    ps = _host_f32(signals, (E, N), "signals")
    px = _host_f32(out_xyzA, (E, 4), "out_xyzA")
    pc = _host_f32(out_score, (E,), "out_score")
    rc = load().ants_reconstruct_host(handle, ps, E, C.byref(grid), int(method), px, pc, int(chunk_events))
    if rc != 0:
        raise AntsError(rc, "ants_reconstruct_host")


def ants_probe_throughput(kind: int, iters: int = 4096):
    """Throughput micro-benchmark (include/ants_recon.h).  -> (scalar results per second, milliseconds)."""
    ops, ms = C.c_double(0.0), C.c_double(0.0)
    rc = load().ants_probe_throughput(int(kind), int(iters), C.byref(ops), C.byref(ms))
    if rc != 0:
        raise AntsError(rc, "ants_probe_throughput")
    return ops.value, ms.value


def plan_info(handle, grid: GridParams, method: int) -> dict:
    v = [C.c_int32() for _ in range(5)]
    rc = load().ants_plan_info(handle, C.byref(grid), int(method), *[C.byref(x) for x in v])
    if rc != 0:
        raise AntsError(rc, "ants_plan_info")
    keys = ("first_diff_iter", "nodes_per_lane", "warps_per_cta", "ctas_per_sm", "smem_bytes")
    out = dict(zip(keys, (x.value for x in v)))
    name = C.create_string_buffer(96)
    if load().ants_plan_kernel_name(handle, C.byref(grid), int(method), name, 96) == 0:
        out["kernel"] = name.value.decode()
    return out


class Reconstructor:
    """Convenience owner of one LRF handle built from a synth.Config-like record."""

    def __init__(self, cfg):
        self.cfg = cfg
        self.dims = LrfDims(cfg.n_sensors, cfg.n_lrf, cfg.lrf_dim, cfg.n_int_r, cfg.n_int_z)
        self.grid = GridParams(cfg.dim, cfg.nodes_per_axis, cfg.step0_xy, cfg.step0_z, cfg.factor,
                               cfg.n_iter, int(getattr(cfg, "seed_mode", 0)), cfg.z_seed)
        self.method = int(cfg.method)
        group = getattr(cfg, "group", None)
        if cfg.lrf_dim >= 3:
            self.handle = ants_lrf_create_xy(cfg.sensor_xy, cfg.gains, cfg.knots if cfg.lrf_dim == 4 else None,
                                             cfg.coeffs if cfg.lrf_dim == 4 else None, self.dims, cfg.n_int_x, cfg.n_int_y,
                                             cfg.n_planes, cfg.knots_xy, cfg.coeffs_xy, getattr(cfg, "xform", None), group)
        elif group is None:
            self.handle = ants_lrf_create(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.coeffs, self.dims)
        else:
            self.handle = ants_lrf_create_grouped(cfg.sensor_xy, cfg.gains, group, cfg.knots, cfg.coeffs, self.dims)
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
