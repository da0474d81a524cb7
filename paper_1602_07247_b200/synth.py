"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module only *makes inputs*: sensor arrays, B-spline LRF coefficients and
flood-field event signals.  It serves the CPU oracle, the CUDA path, the tests
and bench.py alike and therefore holds none of the reconstruction arithmetic
(no centroid, no grid search, no score) and imports neither `oracle/` nor the
CUDA binding.  Spline fitting and spline evaluation go through
`scipy.interpolate.BSpline` (a library routine); bulk signal generation reads
a dense lookup table of that library evaluation so that it can run on the GPU
with torch's seeded generators (the XY-type LRFs, whose tables would be large,
are evaluated from the B-spline basis directly in torch float64; a test checks
that evaluation against scipy's).

Recipe:
  * sensors: hexagonal packing in axial coordinates, or a square grid
    (section 3.3 "regular ... square or hexagonal packing");
  * LRFs: uniform cubic B-splines, least-squares fitted to bell-shaped
    profiles (section 6, "Axial", PAPER.md:394
    "Axial+Z");
  * events: flood field (section 4.1.1) with Poisson photon
    statistics and Gaussian electronic noise (section 4.2.5).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
import torch
from scipy.interpolate import BSpline

# purpose ids of the seeded sub-streams
_STREAM_GAINS, _STREAM_FACTORS, _STREAM_EVENTS = 1, 2, 3


# --------------------------------------------------------------------------
# sensor arrays
# --------------------------------------------------------------------------
def hex_array(rings: int, pitch: float) -> np.ndarray:
    """Hexagonal packing: axial coordinates (q, r), P = pitch*(q + r/2, r*sqrt(3)/2),
    all cells with max(|q|,|r|,|q+r|) <= rings, enumerated r-major then q."""
    pts = []
    for r in range(-rings, rings + 1):
        for q in range(-rings, rings + 1):
            if max(abs(q), abs(r), abs(q + r)) <= rings:
                pts.append((pitch * (q + 0.5 * r), pitch * r * math.sqrt(3.0) / 2.0))
    return np.asarray(pts, dtype=np.float64).astype(np.float32)


def square_array(n_side: int, pitch: float) -> np.ndarray:
    """Square grid centred at the origin, y-major."""
    off = 0.5 * (n_side - 1)
    pts = [((i - off) * pitch, (j - off) * pitch) for j in range(n_side) for i in range(n_side)]
    return np.asarray(pts, dtype=np.float64).astype(np.float32)


# --------------------------------------------------------------------------
# B-spline fits (library routine: scipy BSpline design matrices + lstsq)
# --------------------------------------------------------------------------
def uniform_knot_vector(lo: float, hi: float, n_int: int) -> np.ndarray:
    """Extended uniform knot vector t_j = lo + (j-3)h, j = 0..n_int+6."""
    h = (hi - lo) / n_int
    return lo + (np.arange(n_int + 7) - 3) * h


def _design(x: np.ndarray, lo: float, hi: float, n_int: int) -> np.ndarray:
    t = uniform_knot_vector(lo, hi, n_int)
    return BSpline.design_matrix(np.clip(x, lo, hi), t, 3, extrapolate=True).toarray()


def fit_axial(profile, lo: float, hi: float, n_int: int, n_samples: int = 1000) -> np.ndarray:
    """Unweighted least-squares fit of n_int+3 uniform cubic B-spline coefficients
    to profile(r) on `n_samples` inclusive uniform samples; returns float32."""
    x = np.linspace(lo, hi, n_samples)
    c, *_ = np.linalg.lstsq(_design(x, lo, hi, n_int), profile(x), rcond=None)
    return c.astype(np.float32)


def fit_axial_z(profile, r_rng, z_rng, n_int_r: int, n_int_z: int,
                n_r: int = 200, n_z: int = 50) -> np.ndarray:
    """Separable LS fit of a tensor-product (r,z) spline; returns [n_int_z+3][n_int_r+3] float32."""
    r = np.linspace(r_rng[0], r_rng[1], n_r)
    z = np.linspace(z_rng[0], z_rng[1], n_z)
    F = profile(r[None, :], z[:, None])                      # [n_z][n_r]
    Br = _design(r, r_rng[0], r_rng[1], n_int_r)
    Bz = _design(z, z_rng[0], z_rng[1], n_int_z)
    C = np.linalg.pinv(Bz) @ F @ np.linalg.pinv(Br).T
    return C.astype(np.float32)


def fit_xy(profile, u_rng, v_rng, n_int_x: int, n_int_y: int, n_u: int = 120, n_v: int = 120) -> np.ndarray:
    """Separable LS fit of a tensor-product (u,v) spline to profile(u, v); returns [n_int_y+3][n_int_x+3] float32."""
    return fit_axial_z(lambda u, v: profile(u, v), u_rng, v_rng, n_int_x, n_int_y, n_u, n_v)


def eval_xy_points(coeffs: np.ndarray, u_rng, v_rng, u: np.ndarray, v: np.ndarray) -> np.ndarray:
    """Library evaluation (scipy design matrices) of the tensor-product spline at paired points (u_k, v_k),
    coordinates clamped into the tabulated ranges."""
    Bu = _design(np.asarray(u, dtype=np.float64).ravel(), u_rng[0], u_rng[1], coeffs.shape[1] - 3)
    Bv = _design(np.asarray(v, dtype=np.float64).ravel(), v_rng[0], v_rng[1], coeffs.shape[0] - 3)
    return np.einsum("kb,ba,ka->k", Bv, coeffs.astype(np.float64), Bu).reshape(np.shape(u))


def eval_axial(coeffs: np.ndarray, lo: float, hi: float, r: np.ndarray) -> np.ndarray:
    """Library evaluation (scipy BSpline) of a uniform cubic spline, r clamped to [lo,hi]."""
    n_int = coeffs.shape[-1] - 3
    spl = BSpline(uniform_knot_vector(lo, hi, n_int), coeffs.astype(np.float64), 3, extrapolate=True)
    return spl(np.clip(r, lo, hi))


def eval_axial_z(coeffs: np.ndarray, r_rng, z_rng, r: np.ndarray, z: np.ndarray) -> np.ndarray:
    """Library evaluation of the tensor-product spline on the outer grid z x r."""
    Br = _design(np.asarray(r, dtype=np.float64), r_rng[0], r_rng[1], coeffs.shape[1] - 3)
    Bz = _design(np.asarray(z, dtype=np.float64), z_rng[0], z_rng[1], coeffs.shape[0] - 3)
    return Bz @ coeffs.astype(np.float64) @ Br.T


# --------------------------------------------------------------------------
# configuration record
# --------------------------------------------------------------------------
@dataclasses.dataclass
class Config:
    """Everything ants_lrf_create / ants_reconstruct need, plus the event recipe."""
    name: str
    sensor_xy: np.ndarray            # [N][2] float32, mm
    gains: np.ndarray                # [N] float32
    knots: np.ndarray                # {r_lo,r_hi} or {r_lo,r_hi,z_lo,z_hi} float32
    coeffs: np.ndarray               # [n_lrf][n_int_z+3 or 1][n_int_r+3] float32
    n_lrf: int
    lrf_dim: int
    n_int_r: int
    n_int_z: int
    # search
    dim: int
    nodes_per_axis: int
    step0_xy: float
    step0_z: float
    factor: float
    n_iter: int
    method: int                      # 0 Poisson ML, 1 weighted chi-square
    z_seed: float = float("nan")
    # events
    n_events: int = 0
    region: str = "disk"             # "disk" (radius) or "square" (half-side)
    extent: float = 0.0
    z_range: Optional[tuple] = None
    nph: tuple = ("const", 0.0)      # ("const",v) | ("uniform",a,b) | ("lognormal",median,sigma_log)
    noise_sigma: float = 0.0         # Gaussian electronic noise, result clipped at 0
    n_batches: int = 1
    seed: int = 0
    # sensor selection (PAPER.md:358 passive photosensors; PAPER.md:318 signal threshold / distance from start)
    passive: Optional[np.ndarray] = None     # [N] bool/uint8, non-zero = passive
    signal_min: float = float("nan")         # NaN = off
    dist_max: float = float("nan")           # NaN = off
    seed_mode: int = 0                       # 0 centroid, 1 strongest sensor
    # photosensor grouping: table index of every sensor, n_lrf = number of groups; None = off
    group: Optional[np.ndarray] = None
    # XY-type parameterisations (lrf_dim 3 XY, 4 Composite = Axial + XY, 5 Sliced)
    n_int_x: int = 0
    n_int_y: int = 0
    n_planes: int = 0                        # Sliced: z planes, uniform from z_lo to z_hi
    knots_xy: Optional[np.ndarray] = None    # {u_lo,u_hi,v_lo,v_hi} (+ {z_lo,z_hi} for Sliced) float32
    coeffs_xy: Optional[np.ndarray] = None   # [n_lrf][n_planes or 1][n_int_y+3][n_int_x+3] float32
    xform: Optional[np.ndarray] = None       # [N][4] per-sensor local frame (symmetry groups), or None

    @property
    def n_sensors(self) -> int:
        return int(self.sensor_xy.shape[0])

    @property
    def nodes(self) -> int:
        return self.nodes_per_axis ** self.dim

    @property
    def pairs_per_event(self) -> int:
        return self.n_iter * self.nodes * self.n_sensors

    def final_step(self):
        return (self.step0_xy * self.factor ** (self.n_iter - 1),
                self.step0_z * self.factor ** (self.n_iter - 1))


def _bell(scale):
    return lambda r: (1.0 + (r / scale) ** 2) ** -1.5


def _rng(seed: int, purpose: int) -> np.random.Generator:
    return np.random.default_rng([seed, purpose])


def make_config(idx: int, seed: int = 0, n_events: Optional[int] = None) -> Config:
    """BASELINE.json configs[idx-1], idx = 1..5."""
    if idx == 1:
        xy = hex_array(1, 30.0)
        c = fit_axial(_bell(20.0), 0.0, 90.0, 16)[None, None, :]
        cfg = Config("cfg1_tiny2d_hex7", xy, np.ones(len(xy), np.float32),
                     np.array([0, 90], np.float32), c, 1, 1, 16, 0,
                     2, 9, 5.0, 0.0, 0.5, 8, 0,
                     n_events=10_000, region="disk", extent=30.0, nph=("const", 2000.0))
    elif idx == 2:
        xy = hex_array(2, 30.0)
        g = _rng(seed, _STREAM_GAINS).uniform(0.8, 1.2, len(xy)).astype(np.float32)
        c = fit_axial(_bell(20.0), 0.0, 90.0, 16)[None, None, :]
        cfg = Config("cfg2_pmt2d_hex19", xy, g, np.array([0, 90], np.float32), c, 1, 1, 16, 0,
                     2, 9, 5.0, 0.0, 0.5, 10, 0,
                     n_events=1_000_000, region="disk", extent=60.0,
                     nph=("uniform", 1000.0, 5000.0), noise_sigma=1.0)
    elif idx == 3:
        xy = square_array(8, 6.0)
        base = fit_axial(_bell(4.0), 0.0, 40.0, 12).astype(np.float64)
        fac = _rng(seed, _STREAM_FACTORS).normal(1.0, 0.05, len(xy))
        c = (base[None, :] * fac[:, None]).astype(np.float32)[:, None, :]
        cfg = Config("cfg3_sipm_chi2_sq64", xy, np.ones(len(xy), np.float32),
                     np.array([0, 40], np.float32), c, len(xy), 1, 12, 0,
                     2, 11, 2.0, 0.0, 0.5, 10, 1,
                     n_events=4_000_000, region="square", extent=24.0, nph=("const", 3000.0))
    elif idx == 4:
        xy = hex_array(3, 30.0)
        f = lambda r, z: 125.0 * (z + 5.0) / (r * r + (z + 5.0) ** 2) ** 1.5
        c = fit_axial_z(f, (0.0, 120.0), (0.0, 20.0), 16, 8)[None, :, :]
        cfg = Config("cfg4_axialz3d_hex37", xy, np.ones(len(xy), np.float32),
                     np.array([0, 120, 0, 20], np.float32), c, 1, 2, 16, 8,
                     3, 7, 8.0, 3.0, 0.5, 10, 0,
                     n_events=1_000_000, region="disk", extent=90.0, z_range=(0.0, 20.0),
                     nph=("const", 4000.0))
    elif idx == 5:
        xy = hex_array(6, 25.0)
        g = _rng(seed, _STREAM_GAINS).uniform(0.8, 1.2, len(xy)).astype(np.float32)
        c = fit_axial(_bell(20.0), 0.0, 150.0, 20)[None, None, :]
        cfg = Config("cfg5_flood_hex127", xy, g, np.array([0, 150], np.float32), c, 1, 1, 20, 0,
                     2, 9, 5.0, 0.0, 0.5, 12, 0,
                     n_events=16_000_000, region="disk", extent=140.0,
                     nph=("lognormal", 3000.0, 0.3), noise_sigma=1.5, n_batches=8)
    elif idx == 6:
        # XY LRFs shared by the symmetry of a square array: config 3's SiPM array with a
        # response that is not axial (elliptical bell in the sensor's own frame); 10 symmetry groups, D4
        xy = square_array(8, 6.0)
        group, xform, n_groups = symmetry_groups(xy, 4, True)
        base = fit_xy(lambda u, v: (1.0 + (u / 5.0) ** 2 + (v / 7.0) ** 2) ** -1.5, (-32.0, 32.0), (-32.0, 32.0),
                      16, 16).astype(np.float64)
        fac = _rng(seed, _STREAM_FACTORS).normal(1.0, 0.05, n_groups)
        cxy = (base[None, :, :] * fac[:, None, None]).astype(np.float32)[:, None, :, :]
        cfg = Config("cfg6_xy_sq64_sym", xy, np.ones(len(xy), np.float32), np.array([0, 1], np.float32),
                     np.zeros((n_groups, 1, 0), np.float32), n_groups, 3, 0, 0,
                     2, 11, 2.0, 0.0, 0.5, 10, 1,
                     n_events=1_000_000, region="square", extent=24.0, nph=("const", 3000.0),
                     group=group, xform=xform, n_int_x=16, n_int_y=16,
                     knots_xy=np.array([-32, 32, -32, 32], np.float32), coeffs_xy=cxy)
    elif idx == 7:
        # Sliced LRF: config 4's PMT array, one shared set of XY LRFs on 5 z planes
        xy = hex_array(3, 30.0)
        planes = np.linspace(0.0, 20.0, 5)
        cxy = np.stack([fit_xy(lambda u, v, zp=zp: 1000.0 * (zp + 15.0) / (u * u + v * v + (zp + 15.0) ** 2) ** 1.5,
                               (-120.0, 120.0), (-120.0, 120.0), 20, 20) for zp in planes])[None, :, :, :]
        cfg = Config("cfg7_sliced_hex37", xy, np.ones(len(xy), np.float32), np.array([0, 1], np.float32),
                     np.zeros((1, 1, 0), np.float32), 1, 5, 0, 0,
                     3, 7, 8.0, 3.0, 0.5, 10, 0,
                     n_events=1_000_000, region="disk", extent=90.0, z_range=(0.0, 20.0), nph=("const", 4000.0),
                     n_int_x=20, n_int_y=20, n_planes=5,
                     knots_xy=np.array([-120, 120, -120, 120, 0, 20], np.float32), coeffs_xy=cxy.astype(np.float32))
    elif idx == 8:
        # Composite LRF: config 2's axial response plus a small non-axial XY component
        xy = hex_array(2, 30.0)
        g = _rng(seed, _STREAM_GAINS).uniform(0.8, 1.2, len(xy)).astype(np.float32)
        c = fit_axial(_bell(20.0), 0.0, 90.0, 16)[None, None, :]
        cxy = fit_xy(lambda u, v: 0.03 * np.exp(-(u * u + v * v) / 1250.0) * (u / 25.0), (-90.0, 90.0), (-90.0, 90.0),
                     12, 12)[None, None, :, :]
        cfg = Config("cfg8_composite_hex19", xy, g, np.array([0, 90], np.float32), c, 1, 4, 16, 0,
                     2, 9, 5.0, 0.0, 0.5, 10, 0,
                     n_events=1_000_000, region="disk", extent=60.0, nph=("uniform", 1000.0, 5000.0), noise_sigma=1.0,
                     n_int_x=12, n_int_y=12, knots_xy=np.array([-90, 90, -90, 90], np.float32), coeffs_xy=cxy)
    else:
        raise ValueError("config index must be 1..8")
    cfg.seed = seed
    if n_events is not None:
        cfg.n_events = int(n_events)
    return cfg


def symmetry_groups(sensor_xy: np.ndarray, n_fold: int, reflect: bool, tol: float = 1e-3):
    """Input helper: orbits of the sensors under the rotations by 2 pi k / n_fold about the origin (and the mirror
    y -> -y first, with reflect), each sensor with the transposed operation that maps its group's first sensor
    onto it as its local frame.  -> (group int32 [N], xform float32 [N][4], n_groups).  Pure geometry of the
    input array; the library's own version is ants_group_by_symmetry."""
    P = sensor_xy.astype(np.float64)
    ops = []
    for mirror in ((False, True) if reflect else (False,)):
        for k in range(n_fold):
            a = 2.0 * math.pi * k / n_fold
            R = np.array([[math.cos(a), -math.sin(a)], [math.sin(a), math.cos(a)]])
            ops.append(R @ np.diag([1.0, -1.0]) if mirror else R)
    group = np.full(len(P), -1, np.int32)
    xform = np.zeros((len(P), 4), np.float32)
    n = 0
    for ref in range(len(P)):
        if group[ref] >= 0:
            continue
        for Q in ops:
            d = np.hypot(*(P - Q @ P[ref]).T)
            free = np.flatnonzero((group < 0) & (d <= tol))
            if free.size:
                group[free[0]] = n
                xform[free[0]] = Q.T.reshape(4)
        n += 1
    return group, xform, n


# --------------------------------------------------------------------------
# flood-field events
# --------------------------------------------------------------------------
def _basis4_t(t: torch.Tensor):
    o = 1.0 - t
    return (o * o * o / 6.0, (3.0 * t ** 3 - 6.0 * t * t + 4.0) / 6.0,
            (-3.0 * t ** 3 + 3.0 * t * t + 3.0 * t + 1.0) / 6.0, t ** 3 / 6.0)


def _xy_profile_t(cfg: Config, coef_flat: torch.Tensor, tabs: torch.Tensor, plane, u: torch.Tensor, v: torch.Tensor):
    """Tensor-product uniform cubic B-spline of the XY-type LRFs at (u, v) [m][N] (float64 torch; coordinates
    clamped into the tabulated range), table tabs[i] of sensor i, z plane index `plane` ([m][1] long or 0).
    tests/test_oracle_xy.py checks it against the scipy evaluation (eval_xy_points)."""
    nu3, nv3, P = cfg.n_int_x + 3, cfg.n_int_y + 3, max(cfg.n_planes, 1)
    kx = [float(k) for k in cfg.knots_xy[:4]]

    def locate(x, lo, hi, n):
        t = (x.clamp(lo, hi) - lo) * (n / (hi - lo))
        k = t.floor().clamp(max=n - 1).long()
        return k, t - k
    ku, tu = locate(u, kx[0], kx[1], cfg.n_int_x)
    kv, tv = locate(v, kx[2], kx[3], cfg.n_int_y)
    bu, bv = _basis4_t(tu), _basis4_t(tv)
    base = ((tabs[None, :] * P + plane) * nv3 + kv) * nu3 + ku
    s = torch.zeros_like(u)
    for b in range(4):
        for a in range(4):
            s = s + coef_flat[base + b * nu3 + a] * bu[a] * bv[b]
    return s

_TABLE_R, _TABLE_Z = 1 << 15, 257


def _mean_table(cfg: Config) -> np.ndarray:
    """Dense table of the *library-evaluated* LRF profile(s) over the clamped range.

    Returns [n_lrf][_TABLE_R] (axial) or [_TABLE_Z][_TABLE_R] (axial+z, n_lrf == 1)."""
    r = np.linspace(float(cfg.knots[0]), float(cfg.knots[1]), _TABLE_R)
    if cfg.lrf_dim in (1, 4):
        return np.stack([eval_axial(cfg.coeffs[m, 0], float(cfg.knots[0]), float(cfg.knots[1]), r)
                         for m in range(cfg.n_lrf)])
    z = np.linspace(float(cfg.knots[2]), float(cfg.knots[3]), _TABLE_Z)
    return eval_axial_z(cfg.coeffs[0], cfg.knots[0:2], cfg.knots[2:4], r, z)


def _lerp_table(tab: torch.Tensor, t: torch.Tensor) -> torch.Tensor:
    """tab[..., T] sampled at fractional index t in [0, T-1] (last axis), linear."""
    T = tab.shape[-1]
    t = t.clamp(0.0, T - 1.0)
    i0 = t.floor().clamp(max=T - 2).long()
    w = t - i0
    return tab[i0] * (1 - w) + tab[i0 + 1] * w


def generate_events(cfg: Config, n_events: Optional[int] = None, device="cpu",
                    batch: int = 0, chunk: int = 1 << 18, noise_free: bool = False):
    """Seeded flood-field events.  Returns dict of torch tensors on `device`:
    signals [E][N] float32, true_xyz [E][3] float32, n_ph [E] float32.

    mean_i = 0.1 * N_ph * g_i * profile_i(clamp(|p_xy - P_i|)[, z]); signals are
    Poisson(mean) (+ N(0, noise_sigma), clipped at 0).  `batch` selects an
    independent sub-stream (config 5 streams 8 batches)."""
    E = cfg.n_events // cfg.n_batches if n_events is None else int(n_events)
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed((cfg.seed * 1_000_003 + _STREAM_EVENTS) * 1009 + batch)
    tab = torch.from_numpy(_mean_table(cfg)).to(dev, torch.float64) if cfg.lrf_dim in (1, 2, 4) else None
    if cfg.lrf_dim >= 3:
        cxy_flat = torch.from_numpy(cfg.coeffs_xy.astype(np.float64).ravel()).to(dev)
        T = (torch.from_numpy(cfg.xform.astype(np.float64)).to(dev) if cfg.xform is not None
             else torch.tensor([1.0, 0.0, 0.0, 1.0], dtype=torch.float64, device=dev).repeat(cfg.n_sensors, 1))
    sx = torch.from_numpy(cfg.sensor_xy[:, 0].astype(np.float64)).to(dev)
    sy = torch.from_numpy(cfg.sensor_xy[:, 1].astype(np.float64)).to(dev)
    g = torch.from_numpy(cfg.gains.astype(np.float64)).to(dev)
    r_lo, r_hi = float(cfg.knots[0]), float(cfg.knots[1])
    N = cfg.n_sensors
    sig = torch.empty((E, N), dtype=torch.float32, device=dev)
    pos = torch.zeros((E, 3), dtype=torch.float32, device=dev)
    nph = torch.empty((E,), dtype=torch.float32, device=dev)
    for a in range(0, E, chunk):
        b = min(E, a + chunk)
        m = b - a
        u = torch.rand((m, 5), generator=gen, device=dev, dtype=torch.float64)
        if cfg.region == "disk":
            rho = cfg.extent * u[:, 0].sqrt()
            phi = 2.0 * math.pi * u[:, 1]
            x, y = rho * phi.cos(), rho * phi.sin()
        else:
            x = (2.0 * u[:, 0] - 1.0) * cfg.extent
            y = (2.0 * u[:, 1] - 1.0) * cfg.extent
        z = torch.zeros_like(x)
        if cfg.z_range is not None:
            z = cfg.z_range[0] + (cfg.z_range[1] - cfg.z_range[0]) * u[:, 2]
        kind = cfg.nph[0]
        if kind == "const":
            n = torch.full_like(x, cfg.nph[1])
        elif kind == "uniform":
            n = cfg.nph[1] + (cfg.nph[2] - cfg.nph[1]) * u[:, 3]
        else:  # lognormal(median, sigma_log)
            nrm = torch.randn((m,), generator=gen, device=dev, dtype=torch.float64)
            n = cfg.nph[1] * torch.exp(cfg.nph[2] * nrm)
        r = torch.sqrt((x[:, None] - sx[None, :]) ** 2 + (y[:, None] - sy[None, :]) ** 2)
        t = (r.clamp(r_lo, r_hi) - r_lo) * ((_TABLE_R - 1) / (r_hi - r_lo))
        if cfg.lrf_dim >= 3:
            tables = (torch.from_numpy(np.asarray(cfg.group, np.int64)).to(dev) if cfg.group is not None
                      else (torch.zeros(N, dtype=torch.long, device=dev) if cfg.n_lrf == 1 else torch.arange(N, device=dev)))
            dxs, dys = x[:, None] - sx[None, :], y[:, None] - sy[None, :]
            uu = T[None, :, 0] * dxs + T[None, :, 1] * dys
            vv = T[None, :, 2] * dxs + T[None, :, 3] * dys
            if cfg.lrf_dim == 5:
                z_lo, z_hi = float(cfg.knots_xy[4]), float(cfg.knots_xy[5])
                dzp = (z_hi - z_lo) / (cfg.n_planes - 1)
                pz = ((z.clamp(z_lo, z_hi) - z_lo) / dzp).floor().clamp(max=cfg.n_planes - 2).long()
                wz = ((z.clamp(z_lo, z_hi) - (z_lo + pz * dzp)) / dzp)[:, None]
                prof = ((1.0 - wz) * _xy_profile_t(cfg, cxy_flat, tables, pz[:, None], uu, vv)
                        + wz * _xy_profile_t(cfg, cxy_flat, tables, pz[:, None] + 1, uu, vv))
            else:
                prof = _xy_profile_t(cfg, cxy_flat, tables, 0, uu, vv)
                if cfg.lrf_dim == 4:
                    prof = prof + _lerp_table(tab[0], t)
        elif cfg.lrf_dim == 1:
            if cfg.n_lrf == 1:
                prof = _lerp_table(tab[0], t)
            else:
                i0 = t.floor().clamp(max=_TABLE_R - 2).long()
                w = t - i0
                tables = (torch.arange(N, device=dev) if cfg.group is None
                          else torch.from_numpy(np.asarray(cfg.group, np.int64)).to(dev))
                rows = tables[None, :].expand(m, N)
                prof = tab[rows, i0] * (1 - w) + tab[rows, i0 + 1] * w
        else:
            z_lo, z_hi = float(cfg.knots[2]), float(cfg.knots[3])
            tz = (z.clamp(z_lo, z_hi) - z_lo) * ((_TABLE_Z - 1) / (z_hi - z_lo))
            j0 = tz.floor().clamp(max=_TABLE_Z - 2).long()
            wz = (tz - j0)[:, None]
            i0 = t.floor().clamp(max=_TABLE_R - 2).long()
            w = t - i0
            j0 = j0[:, None].expand(m, N)
            prof = ((tab[j0, i0] * (1 - w) + tab[j0, i0 + 1] * w) * (1 - wz)
                    + (tab[j0 + 1, i0] * (1 - w) + tab[j0 + 1, i0 + 1] * w) * wz)
        mean = (0.1 * n)[:, None] * g[None, :] * prof
        mean = mean.clamp_min(0.0)
        if noise_free:
            s = mean
        else:
            s = torch.poisson(mean.to(torch.float32), generator=gen).to(torch.float64)
            if cfg.noise_sigma > 0.0:
                s = s + cfg.noise_sigma * torch.randn((m, N), generator=gen, device=dev,
                                                       dtype=torch.float64)
                s = s.clamp_min(0.0)
        sig[a:b] = s.to(torch.float32)
        pos[a:b, 0], pos[a:b, 1], pos[a:b, 2] = x.float(), y.float(), z.float()
        nph[a:b] = n.float()
    return {"signals": sig, "true_xyz": pos, "n_ph": nph}
