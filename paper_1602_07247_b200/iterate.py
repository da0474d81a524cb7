"""The iterative response reconstruction of PAPER.md:428-442 (section 8) as a thin driver:
reconstruct all flood events with the current LRFs -> filter -> recalculate the LRFs -> repeat.
Every step runs in the library's kernels (ants_reconstruct, ants_filter_events, ants_lrf_fit_*);
this module only chains the calls and swaps the coefficient arrays."""
from __future__ import annotations

import copy

import numpy as np

from . import recon


def iterate_response(cfg, signals, n_cycles: int, score_max: float = float("nan"),
                     energy_min: float = float("nan"), energy_max: float = float("nan"),
                     radius_max: float = float("nan"), refit_gains: bool = False):
    """cfg: a synth.Config-like record with the starting LRFs (axial, shared or per-sensor tables, axial+z,
    XY or Composite); signals: CUDA float32 [E][N].  Yields (cycle, cfg_k, n_events_used) after every cycle, cfg_k
    carrying the refitted coefficients (and gains when refit_gains, shared axial profile only).  A table that the
    passing events do not cover (an interval or cell without data: typical for per-sensor tables fitted over their full
    range from a small flood batch) ends the iteration with recon.AntsError (ANTS_ERR_SINGULAR): give cfg the knot range
    the data cover."""
    cur = copy.copy(cfg)
    for cycle in range(n_cycles):
        r = recon.Reconstructor(cur)
        try:
            xyzA, score = r(signals)
        finally:
            r.close()
        n_pass = recon.ants_filter_events(xyzA, score, score_max, energy_min, energy_max, radius_max)
        nxt = copy.copy(cur)
        if cur.lrf_dim in (3, 4):
            # XY tables; for a Composite LRF the axial component first, then the XY component on the residual
            axial = None
            if cur.lrf_dim == 4:
                ca, _ = recon.ants_lrf_fit_axial(cur.sensor_xy, cur.gains, cur.knots, cur.n_lrf, cur.n_int_r, signals, xyzA,
                                                 group=getattr(cur, "group", None))
                nxt.coeffs = ca[:, None, :].astype(np.float32)
                axial = (cur.knots, ca)
            c, _ = recon.ants_lrf_fit_xy(cur.sensor_xy, cur.gains, cur.knots_xy, cur.n_lrf, cur.n_int_x, cur.n_int_y, signals,
                                         xyzA, group=getattr(cur, "group", None), xform=getattr(cur, "xform", None), axial=axial)
            nxt.coeffs_xy = c[:, None, :, :].astype(np.float32)
        elif cur.lrf_dim == 5:
            c, _ = recon.ants_lrf_fit_sliced(cur.sensor_xy, cur.gains, cur.knots_xy, cur.n_lrf, cur.n_int_x, cur.n_int_y,
                                             cur.n_planes, signals, xyzA, group=getattr(cur, "group", None),
                                             xform=getattr(cur, "xform", None))
            nxt.coeffs_xy = c.astype(np.float32)
        elif cur.lrf_dim == 2:
            c, _ = recon.ants_lrf_fit_axial_z(cur.sensor_xy, cur.gains, cur.knots, cur.n_int_r, cur.n_int_z, signals, xyzA)
            nxt.coeffs = c[None, :, :].astype(np.float32)
        else:
            c, _ = recon.ants_lrf_fit_axial(cur.sensor_xy, cur.gains, cur.knots, cur.n_lrf, cur.n_int_r, signals, xyzA,
                                            group=getattr(cur, "group", None))
            nxt.coeffs = c[:, None, :].astype(np.float32)
            if refit_gains and cur.n_lrf == 1:
                g, _ = recon.ants_lrf_fit_gains(cur.sensor_xy, cur.knots, c[0], signals, xyzA)
                nxt.gains = recon.ants_gains_renormalise(g, cur.gains)     # gains are relative (R29)
        cur = nxt
        yield cycle, cur, n_pass
