"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module only *makes inputs*: sensor arrays, B-spline LRF coefficients and
flood-field event signals.  It serves the CPU oracle, the CUDA path, the tests
and bench.py alike and therefore holds none of the reconstruction arithmetic
(no centroid, no grid search, no score) and imports neither `oracle/` nor the
CUDA binding.  Spline fitting and spline evaluation go through
`scipy.interpolate.BSpline` (a library routine); bulk signal generation reads
a dense lookup table of that library evaluation so that it can run on the GPU
with torch's seeded generators.

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
    else:
        raise ValueError("config index must be 1..5")
    cfg.seed = seed
    if n_events is not None:
        cfg.n_events = int(n_events)
    return cfg


# --------------------------------------------------------------------------
# flood-field events
# --------------------------------------------------------------------------
_TABLE_R, _TABLE_Z = 1 << 15, 257


def _mean_table(cfg: Config) -> np.ndarray:
    """Dense table of the *library-evaluated* LRF profile(s) over the clamped range.

    Returns [n_lrf][_TABLE_R] (axial) or [_TABLE_Z][_TABLE_R] (axial+z, n_lrf == 1)."""
    r = np.linspace(float(cfg.knots[0]), float(cfg.knots[1]), _TABLE_R)
    if cfg.lrf_dim == 1:
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
    tab = torch.from_numpy(_mean_table(cfg)).to(dev, torch.float64)
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
        if cfg.lrf_dim == 1:
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
