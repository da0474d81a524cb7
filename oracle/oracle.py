"""ctypes wrapper of the CPU oracle (oracle/ants_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_1602_07247_b200 and shares no code with the CUDA
path.  The arithmetic lives in the C file; this file only marshals arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ants_oracle.c")
_LIB = os.path.join(_HERE, "libants_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (plain C99 + OpenMP over events)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
                               "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Model(C.Structure):
    _fields_ = [("n_sensors", C.c_int32), ("n_lrf", C.c_int32), ("lrf_dim", C.c_int32),
                ("n_int_r", C.c_int32), ("n_int_z", C.c_int32),
                ("sensor_xy", C.c_void_p), ("gains", C.c_void_p),
                ("knots", C.c_void_p), ("coeffs", C.c_void_p),
                ("passive", C.c_void_p), ("signal_min", C.c_float), ("dist_max", C.c_float),
                ("group", C.c_void_p),
                ("n_int_x", C.c_int32), ("n_int_y", C.c_int32), ("n_planes", C.c_int32),
                ("knots_xy", C.c_void_p), ("coeffs_xy", C.c_void_p), ("xform", C.c_void_p)]


class _Grid(C.Structure):
    _fields_ = [("dim", C.c_int32), ("nodes_per_axis", C.c_int32),
                ("step0_xy", C.c_float), ("step0_z", C.c_float), ("factor", C.c_float),
                ("n_iter", C.c_int32), ("seed_mode", C.c_int32), ("z_seed", C.c_float)]


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.oracle_spline1.restype = C.c_double
        lib.oracle_spline1.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double]
        lib.oracle_spline2.restype = C.c_double
        lib.oracle_spline2.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.c_double] * 6
        lib.oracle_lrf.restype = C.c_double
        lib.oracle_lrf.argtypes = [C.POINTER(_Model), C.c_int, C.c_double, C.c_double, C.c_double]
        lib.oracle_centroid.restype = C.c_int
        lib.oracle_centroid.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int, C.c_void_p]
        lib.oracle_score_at.restype = C.c_int
        lib.oracle_start.restype = C.c_int
        lib.oracle_start.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        lib.oracle_score_at.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double,
                                        C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.oracle_score_at_many.restype = C.c_int
        lib.oracle_score_at_many.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int64, C.c_int, C.c_int,
                                             C.c_void_p, C.c_void_p, C.c_void_p]
        lib.oracle_threads.restype = C.c_int
        lib.oracle_threads.argtypes = [C.c_int]
        lib.oracle_reconstruct.restype = C.c_int
        lib.oracle_reconstruct.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int64, C.POINTER(_Grid),
                                           C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_int]
        lib.oracle_lrf_grad.restype = C.c_double
        lib.oracle_lrf_grad.argtypes = [C.POINTER(_Model), C.c_int, C.c_double, C.c_double, C.c_double, C.c_void_p]
        lib.oracle_score_grad.restype = C.c_int
        lib.oracle_score_grad.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                          C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p, C.c_void_p]
        lib.oracle_refine.restype = C.c_int
        lib.oracle_refine.argtypes = [C.POINTER(_Model), C.c_void_p, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int,
                                      C.c_void_p, C.c_void_p, C.c_int]
        _lib = lib
    return _lib


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def spline1(coeffs, lo, hi, x):
    """Uniform cubic B-spline with len(coeffs)-3 intervals on [lo,hi] at scalar/array x."""
    lib = _load()
    c = _f32(coeffs)
    xs = np.atleast_1d(np.asarray(x, dtype=np.float64))
    out = np.array([lib.oracle_spline1(c.ctypes.data, c.size - 3, float(lo), float(hi), float(v))
                    for v in xs.ravel()]).reshape(xs.shape)
    return out if np.ndim(x) else float(out[0])


def spline2(coeffs, r_rng, z_rng, r, z):
    """Tensor-product spline, coeffs [nz+3][nr+3], at scalar (r,z)."""
    lib = _load()
    c = _f32(coeffs)
    return lib.oracle_spline2(c.ctypes.data, c.shape[1] - 3, c.shape[0] - 3, float(r_rng[0]),
                              float(r_rng[1]), float(z_rng[0]), float(z_rng[1]), float(r), float(z))


class Model:
    """The LRF model: the float32 arrays handed to ants_lrf_create, kept alive here."""

    def __init__(self, sensor_xy, gains, knots, coeffs, n_lrf, lrf_dim, n_int_r, n_int_z,
                 passive=None, signal_min=float("nan"), dist_max=float("nan"), group=None,
                 n_int_x=0, n_int_y=0, n_planes=0, knots_xy=None, coeffs_xy=None, xform=None):
        self.sensor_xy = _f32(sensor_xy).reshape(-1, 2)
        N = self.sensor_xy.shape[0]
        self.gains = _f32(np.ones(N) if gains is None else gains)
        self.knots = _f32(knots if knots is not None else [0.0, 1.0])
        self.coeffs = _f32(coeffs if coeffs is not None else np.zeros(0))
        if lrf_dim in (1, 2, 4):
            assert self.coeffs.size == n_lrf * (n_int_r + 3) * ((n_int_z + 3) if lrf_dim == 2 else 1)
        self.knots_xy = self.coeffs_xy = self.xform = None
        if lrf_dim >= 3:
            self.knots_xy = _f32(knots_xy)
            self.coeffs_xy = _f32(coeffs_xy)
            assert self.knots_xy.size == (6 if lrf_dim == 5 else 4)
            assert (n_planes >= 2) if lrf_dim == 5 else (n_planes == 0)
            assert self.coeffs_xy.size == n_lrf * max(n_planes, 1) * (n_int_x + 3) * (n_int_y + 3)
            if xform is not None:
                self.xform = _f32(xform).reshape(N, 4)
        self.n_sensors = N
        self.passive = None if passive is None else np.ascontiguousarray(np.asarray(passive) != 0, dtype=np.uint8)
        assert self.passive is None or self.passive.size == N
        self.group = None if group is None else np.ascontiguousarray(np.asarray(group, dtype=np.int32))
        assert self.group is None or (self.group.size == N and self.group.min() >= 0 and self.group.max() < n_lrf)
        self.c = _Model(N, n_lrf, lrf_dim, n_int_r, n_int_z, self.sensor_xy.ctypes.data,
                        self.gains.ctypes.data, self.knots.ctypes.data, self.coeffs.ctypes.data,
                        None if self.passive is None else self.passive.ctypes.data,
                        float(signal_min), float(dist_max),
                        None if self.group is None else self.group.ctypes.data,
                        int(n_int_x), int(n_int_y), int(n_planes),
                        None if self.knots_xy is None else self.knots_xy.ctypes.data,
                        None if self.coeffs_xy is None else self.coeffs_xy.ctypes.data,
                        None if self.xform is None else self.xform.ctypes.data)

    @classmethod
    def from_config(cls, cfg):
        return cls(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.coeffs, cfg.n_lrf, cfg.lrf_dim,
                   cfg.n_int_r, cfg.n_int_z, getattr(cfg, "passive", None),
                   getattr(cfg, "signal_min", float("nan")), getattr(cfg, "dist_max", float("nan")),
                   getattr(cfg, "group", None), getattr(cfg, "n_int_x", 0), getattr(cfg, "n_int_y", 0),
                   getattr(cfg, "n_planes", 0), getattr(cfg, "knots_xy", None), getattr(cfg, "coeffs_xy", None),
                   getattr(cfg, "xform", None))

    def lrf(self, i, x, y, z=0.0):
        return _load().oracle_lrf(C.byref(self.c), int(i), float(x), float(y), float(z))

    def centroid(self, signals, method=0):
        s = _f32(signals)
        xy = np.zeros(2)
        rc = _load().oracle_centroid(C.byref(self.c), s.ctypes.data, int(method), xy.ctypes.data)
        return xy, rc

    def start(self, signals, method=0, seed_mode=0):
        """Start search position (centroid or strongest sensor) and the unusable-event flag."""
        s = _f32(signals)
        xy = np.zeros(2)
        rc = _load().oracle_start(C.byref(self.c), s.ctypes.data, int(method), int(seed_mode), xy.ctypes.data)
        return xy, rc

    def score_at(self, signals, method, x, y, z=0.0, seed_mode=0):
        """(A, score) of one event's signals at a position; invalid node -> (nan, inf)."""
        s = _f32(signals)
        A, sc = C.c_double(), C.c_double()
        _load().oracle_score_at(C.byref(self.c), s.ctypes.data, int(method), int(seed_mode), float(x), float(y),
                                float(z), C.byref(A), C.byref(sc))
        return A.value, sc.value


def lrf_grad(model: Model, i, x, y, z=0.0):
    """(L_i, dL_i/d(x, y, z)) at a position."""
    g = np.zeros(3)
    v = _load().oracle_lrf_grad(C.byref(model.c), int(i), float(x), float(y), float(z), g.ctypes.data)
    return v, g


def score_grad(model: Model, signals, method, x, y, z=0.0, dim=2, seed_mode=0):
    """(A, F, gradient [3], Gauss-Newton matrix [3][3], rc) of one event at a position (R34)."""
    s = _f32(signals)
    A, F, g, H = C.c_double(), C.c_double(), np.zeros(3), np.zeros((3, 3))
    rc = _load().oracle_score_grad(C.byref(model.c), s.ctypes.data, int(method), int(seed_mode), int(dim), float(x),
                                   float(y), float(z), C.byref(A), C.byref(F), g.ctypes.data, H.ctypes.data)
    return A.value, F.value, g, H, rc


def refine(model: Model, signals, method, xyz_start, n_steps, dim=2, seed_mode=0, threads=0):
    """Levenberg-Marquardt refinement (R34) from xyz_start [E][3].  -> dict xyzA [E][4], score [E] (float64)."""
    s = _f32(signals).reshape(-1, model.n_sensors)
    E = s.shape[0]
    xyzA = np.zeros((E, 4))
    xyzA[:, :3] = np.asarray(xyz_start, np.float64).reshape(E, 3)
    score = np.full(E, np.inf)
    rc = _load().oracle_refine(C.byref(model.c), s.ctypes.data, E, int(method), int(seed_mode), int(dim), int(n_steps),
                               xyzA.ctypes.data, score.ctypes.data, int(threads))
    if rc != 0:
        raise ValueError("oracle_refine: invalid argument")
    return {"xyzA": xyzA, "score": score}


def score_at_many(model: Model, signals, method: int, pos, seed_mode: int = 0):
    """(A [E], score [E]) of each event's signals at its own position pos [E][3]."""
    s = _f32(signals).reshape(-1, model.n_sensors)
    p = np.ascontiguousarray(np.asarray(pos, dtype=np.float64)).reshape(-1, 3)
    assert p.shape[0] == s.shape[0]
    A, sc = np.zeros(s.shape[0]), np.zeros(s.shape[0])
    rc = _load().oracle_score_at_many(C.byref(model.c), s.ctypes.data, s.shape[0], int(method), int(seed_mode),
                                      p.ctypes.data, A.ctypes.data, sc.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_score_at_many: invalid argument")
    return A, sc


def grid_params(dim, nodes_per_axis, step0_xy, step0_z, factor, n_iter, z_seed=float("nan"), seed_mode=0):
    return _Grid(int(dim), int(nodes_per_axis), float(step0_xy), float(step0_z), float(factor),
                 int(n_iter), int(seed_mode), float(z_seed))


def grid_from_config(cfg):
    return grid_params(cfg.dim, cfg.nodes_per_axis, cfg.step0_xy, cfg.step0_z, cfg.factor,
                       cfg.n_iter, cfg.z_seed, getattr(cfg, "seed_mode", 0))


def n_threads(requested: int = 0) -> int:
    return _load().oracle_threads(int(requested))


def reconstruct(model: Model, signals, grid: _Grid, method: int, threads: int = 0, trace: bool = False):
    """Contracting-grid reconstruction of signals [E][N].

    Returns dict: xyzA [E][4] float64, score [E] float64 and, with trace=True,
    idx [E][K] int32 (winning linear node index per iteration, -1 = none valid),
    best [E][K], second [E][K] (best and second-best node score per iteration)."""
    s = _f32(signals).reshape(-1, model.n_sensors)
    E, K = s.shape[0], grid.n_iter
    xyzA = np.zeros((E, 4))
    score = np.zeros(E)
    idx = np.zeros((E, K), np.int32) if trace else None
    best = np.zeros((E, K)) if trace else None
    second = np.zeros((E, K)) if trace else None
    rc = _load().oracle_reconstruct(C.byref(model.c), s.ctypes.data, E, C.byref(grid), int(method),
                                    xyzA.ctypes.data, score.ctypes.data,
                                    idx.ctypes.data if trace else None,
                                    best.ctypes.data if trace else None,
                                    second.ctypes.data if trace else None, int(threads))
    if rc != 0:
        raise ValueError("oracle_reconstruct: invalid argument")
    out = {"xyzA": xyzA, "score": score}
    if trace:
        out.update(idx=idx, best=best, second=second)
    return out
