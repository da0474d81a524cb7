"""CPU ORACLE of the LRF calculation (TEST INFRASTRUCTURE, NOT THE PRODUCT).

PAPER.md:380 (section 6): "The LRF module calculates these functions from datasets containing
photosensor signals and the corresponding event positions"; the LRFs are B-splines of the
distance to the sensor axis ("Axial"), one per sensor or one per group with a relative gain
per sensor (section 6.2); the positions are the reconstructed or the true ones
(PAPER.md:414).  The paper prints no fit criterion; the readings are DESIGN.md R21-R23:

  R21  unweighted least squares: for table m the coefficients c minimise
           sum over events e and sensors i of the table of ( y_ie - s_c(r_ie) )^2,
       y_ie = S_ie / (A_e g_i)   ("a point light source emitting ... a constant number of photons",
       PAPER.md:380: the signal is normalised by the event's energy scale A_e; g_i = 1 for per-sensor tables),
       r_ie = |p_e - P_i|, s_c the uniform cubic B-spline of oracle/ants_oracle.c (R7);
  R22  an event takes part if x, y, A are finite and A > 0 (failed events carry NaN); a pair takes part
       if r_lo <= r <= r_hi (no extrapolation data);
  R23  signals enter as they are (no clipping), in double.

Plain numpy in float64, written in the order of the definition: design rows, normal equations
M = sum B^T B, b = sum B^T y, then the library solve numpy.linalg.solve.  Shares no code with the CUDA
path.  Pins: tests/test_oracle_fit.py.
"""
from __future__ import annotations

import numpy as np


def basis4(u):
    """The four uniform cubic B-spline basis values at local coordinate u in [0, 1] (R7)."""
    return np.stack([(1.0 - u) ** 3 / 6.0,
                     (3.0 * u ** 3 - 6.0 * u ** 2 + 4.0) / 6.0,
                     (-3.0 * u ** 3 + 3.0 * u ** 2 + 3.0 * u + 1.0) / 6.0,
                     u ** 3 / 6.0], axis=-1)


def normal_equations(sensor_xy, gains, knots, n_lrf, n_int, signals, xyzA, group=None):
    """-> M [n_lrf][n+3][n+3], b [n_lrf][n+3], n_used [n_lrf] (pairs that entered each table).
    group (R28): table index of every sensor, values 0 .. n_lrf-1; the sensors of a group share one profile
    scaled by their relative gains (section 6.2).  None = the two built-in groupings:
    one group for all sensors (n_lrf = 1) or one table per sensor without gains (n_lrf = N)."""
    xy = np.asarray(sensor_xy, np.float32).astype(np.float64).reshape(-1, 2)
    N = xy.shape[0]
    g = np.ones(N) if gains is None else np.asarray(gains, np.float32).astype(np.float64)
    lo, hi = (float(np.float32(k)) for k in knots[:2])
    h = (hi - lo) / n_int
    S = np.asarray(signals, np.float32).astype(np.float64).reshape(-1, N)
    P = np.asarray(xyzA, np.float32).astype(np.float64).reshape(-1, 4)
    ok = np.isfinite(P[:, 0]) & np.isfinite(P[:, 1]) & np.isfinite(P[:, 3]) & (P[:, 3] > 0.0)     # R22
    nc = n_int + 3
    M = np.zeros((n_lrf, nc, nc))
    b = np.zeros((n_lrf, nc))
    n_used = np.zeros(n_lrf)
    for i in range(N):
        if group is not None:
            m, gi = int(group[i]), g[i]
        else:
            m = 0 if n_lrf == 1 else i
            gi = g[i] if n_lrf == 1 else 1.0
        with np.errstate(invalid="ignore"):
            r = np.hypot(P[:, 0] - xy[i, 0], P[:, 1] - xy[i, 1])
            use = ok & (r >= lo) & (r <= hi)                                                     # R22
        r_u, y = r[use], S[use, i] / (P[use, 3] * gi)                                             # R21, R23
        t = (r_u - lo) / h
        k = np.minimum(np.floor(t).astype(np.int64), n_int - 1)
        B4 = basis4(t - k)                                   # [n][4]: coefficients k .. k+3
        for a in range(4):
            np.add.at(b[m], k + a, B4[:, a] * y)
            for c in range(4):
                np.add.at(M[m], (k + a, k + c), B4[:, a] * B4[:, c])
        n_used[m] += use.sum()
    return M, b, n_used


def fit_axial(sensor_xy, gains, knots, n_lrf, n_int, signals, xyzA, group=None):
    """Least-squares B-spline coefficients [n_lrf][n_int + 3] (float64) and the pairs used per table.
    Raises numpy.linalg.LinAlgError when a table is underdetermined (an interval without data)."""
    M, b, n_used = normal_equations(sensor_xy, gains, knots, n_lrf, n_int, signals, xyzA, group)
    c = np.stack([np.linalg.solve(M[m], b[m]) for m in range(n_lrf)])
    return c, n_used


def spline_values(coeffs, lo, hi, n_int, r):
    """Uniform cubic B-spline of oracle/ants_oracle.c (R7) at r in [lo, hi], float64."""
    c = np.asarray(coeffs, np.float32).astype(np.float64)
    h = (hi - lo) / n_int
    t = (r - lo) / h
    k = np.minimum(np.floor(t).astype(np.int64), n_int - 1)
    B4 = basis4(t - k)
    return sum(c[k + a] * B4[:, a] for a in range(4))


def fit_gains(sensor_xy, knots, coeffs, n_int, signals, xyzA):
    """Relative gains for a FIXED shared profile (section 6.3: "re-calculate the relative gains
    of the photosensors within already defined groups without affecting the LRF profiles").  Reading R24:
    g_i minimises sum_e (S_ie/A_e - g_i s(r_ie))^2 over the pairs of R22, i.e.
    g_i = sum_e y s / sum_e s^2 with y = S_ie/A_e.  -> gains [N] (NaN where a sensor has no pair), pairs [N]."""
    xy = np.asarray(sensor_xy, np.float32).astype(np.float64).reshape(-1, 2)
    N = xy.shape[0]
    lo, hi = (float(np.float32(k)) for k in knots[:2])
    S = np.asarray(signals, np.float32).astype(np.float64).reshape(-1, N)
    P = np.asarray(xyzA, np.float32).astype(np.float64).reshape(-1, 4)
    ok = np.isfinite(P[:, 0]) & np.isfinite(P[:, 1]) & np.isfinite(P[:, 3]) & (P[:, 3] > 0.0)
    gains, used = np.full(N, np.nan), np.zeros(N)
    for i in range(N):
        with np.errstate(invalid="ignore"):
            r = np.hypot(P[:, 0] - xy[i, 0], P[:, 1] - xy[i, 1])
            use = ok & (r >= lo) & (r <= hi)
        s = spline_values(coeffs, lo, hi, n_int, r[use])
        y = S[use, i] / P[use, 3]
        den = float((s * s).sum())
        used[i] = use.sum()
        if den > 0.0:
            gains[i] = float((y * s).sum()) / den
    return gains, used


def fit_axial_z(sensor_xy, gains, knots, n_int_r, n_int_z, signals, xyzA):
    """Least-squares fit of the shared axial+z tensor-product LRF s(r, z) (section 6.1.2;
    PAPER.md:380 LRFs are calculated from signals + positions).  Reading R25 = R21-R23 carried to (r, z):
    y = S/(A g) against sum_b sum_a c[kz+b][kr+a] bz_b(uz) br_a(ur) (the tensor spline of
    oracle/ants_oracle.c), over events with finite x, y, z, A, A > 0 and z_lo <= z <= z_hi, pairs with
    r_lo <= r <= r_hi.  -> coefficients [n_int_z + 3][n_int_r + 3] (float64), pairs used."""
    xy = np.asarray(sensor_xy, np.float32).astype(np.float64).reshape(-1, 2)
    N = xy.shape[0]
    g = np.ones(N) if gains is None else np.asarray(gains, np.float32).astype(np.float64)
    r_lo, r_hi, z_lo, z_hi = (float(np.float32(k)) for k in knots[:4])
    hr, hz = (r_hi - r_lo) / n_int_r, (z_hi - z_lo) / n_int_z
    ncr, ncz = n_int_r + 3, n_int_z + 3
    S = np.asarray(signals, np.float32).astype(np.float64).reshape(-1, N)
    P = np.asarray(xyzA, np.float32).astype(np.float64).reshape(-1, 4)
    with np.errstate(invalid="ignore"):
        ok = (np.isfinite(P).all(axis=1) & (P[:, 3] > 0.0) & (P[:, 2] >= z_lo) & (P[:, 2] <= z_hi))
    M = np.zeros((ncz * ncr, ncz * ncr))
    b = np.zeros(ncz * ncr)
    used = 0.0
    for i in range(N):
        with np.errstate(invalid="ignore"):
            r = np.hypot(P[:, 0] - xy[i, 0], P[:, 1] - xy[i, 1])
            use = ok & (r >= r_lo) & (r <= r_hi)
        y = S[use, i] / (P[use, 3] * g[i])
        tr = (r[use] - r_lo) / hr
        kr = np.minimum(np.floor(tr).astype(np.int64), n_int_r - 1)
        Br = basis4(tr - kr)
        tz = (P[use, 2] - z_lo) / hz
        kz = np.minimum(np.floor(tz).astype(np.int64), n_int_z - 1)
        Bz = basis4(tz - kz)
        idx = [((kz + bb) * ncr + kr + aa, Bz[:, bb] * Br[:, aa]) for bb in range(4) for aa in range(4)]
        for j1, w1 in idx:
            np.add.at(b, j1, w1 * y)
            for j2, w2 in idx:
                np.add.at(M, (j1, j2), w1 * w2)
        used += use.sum()
    c = np.linalg.solve(M, b)
    return c.reshape(ncz, ncr), used


def filter_events(xyzA, score, score_max=float("nan"), energy_min=float("nan"), energy_max=float("nan"),
                  radius_max=float("nan")):
    """Event filters (section 5.2: "individual events can be filtered out according to ...
    reconstructed ... event energy, chi-squared value of the reconstruction, and the event position";
    "Only those events which pass all the activated filters are used in LRF reconstruction").  Reading R26:
    an event passes if its reconstruction did not fail (finite x, y, A, score) and, for every activated
    (non-NaN) criterion, score <= score_max, energy_min <= A <= energy_max, x^2 + y^2 <= radius_max^2
    (compared in double on the float32 values).  -> boolean mask [E] and the filtered copy of xyzA in which
    rejected rows are NaN (what the LRF calculation ignores, R22)."""
    P = np.asarray(xyzA, np.float32).reshape(-1, 4)
    s = np.asarray(score, np.float32).reshape(-1)
    Pd, sd = P.astype(np.float64), s.astype(np.float64)
    keep = np.isfinite(Pd[:, 0]) & np.isfinite(Pd[:, 1]) & np.isfinite(Pd[:, 3]) & np.isfinite(sd)
    with np.errstate(invalid="ignore"):
        if not np.isnan(score_max):
            keep &= sd <= float(np.float32(score_max))
        if not np.isnan(energy_min):
            keep &= Pd[:, 3] >= float(np.float32(energy_min))
        if not np.isnan(energy_max):
            keep &= Pd[:, 3] <= float(np.float32(energy_max))
        if not np.isnan(radius_max):
            rm = float(np.float32(radius_max))
            keep &= Pd[:, 0] * Pd[:, 0] + Pd[:, 1] * Pd[:, 1] <= rm * rm
    out = P.copy()
    out[~keep] = np.nan
    return keep, out


def group_by_radius(sensor_xy, tol=1e-3):
    """"Grouping according to the distance from the sensor center to the detector center":
    sensors whose distance from the origin agrees within tol (mm) share a group; groups are numbered by
    increasing distance.  -> (group [N] int32, n_groups)."""
    xy = np.asarray(sensor_xy, np.float64).reshape(-1, 2)
    d = np.hypot(xy[:, 0], xy[:, 1])
    order = np.argsort(d, kind="stable")
    group = np.zeros(len(d), np.int32)
    g, last = -1, None
    for i in order:
        if last is None or d[i] - last > tol:
            g += 1
            last = d[i]          # a group is anchored at its first (smallest) distance
        group[i] = g
    return group, g + 1


def renormalise_gains(gains_new, gains_prev):
    """Relative gains are defined up to a common factor ("a scaling parameter (relative gain)");
    between cycles of the iterative procedure they are carried on at the scale of the
    previous set.  Reading R29: a sensor whose new estimate is missing (NaN) or not positive keeps its previous
    gain; the set is then multiplied by mean(gains_prev) / mean(set).  -> float32 [N]."""
    gn = np.asarray(gains_new, np.float32).astype(np.float64).reshape(-1)
    gp = np.asarray(gains_prev, np.float32).astype(np.float64).reshape(-1)
    with np.errstate(invalid="ignore"):
        usable = np.isfinite(gn) & (gn > 0.0)
    g = np.where(usable, gn, gp)
    return (g * (gp.mean() / g.mean())).astype(np.float32)


def group_by_symmetry(sensor_xy, n_fold, reflect=True, tol=1e-3):
    """"Grouping based on rotation or/and reflection symmetry of the sensor array (square, rectangular or
    hexagonal)".  Reading R33: the operations are the rotations by 2 pi k / n_fold about the
    detector centre (the origin), k = 0 .. n_fold-1, and, with reflect, each of them applied after the mirror
    y -> -y (n_fold = 4 for a square array, 2 for a rectangular one, 6 for a hexagonal one).  Sensors are taken
    in index order: one that has no group yet founds the next group as its reference; every operation Q, in the
    order above, sends the reference position to Q P_ref, and a sensor within tol (mm) of that image that has no
    group yet joins with the frame T_i = Q^-1 = Q^T, so that its local coordinates (u, v) = T_i (p - P_i) are
    those of the reference sensor seen from the turned-back point.
    -> (group [N] int32, xform [N][4] float32 row-major, n_groups)."""
    xy = np.asarray(sensor_xy, np.float32).astype(np.float64).reshape(-1, 2)
    N = len(xy)
    ops = []
    for mirror in ((False, True) if reflect else (False,)):
        for k in range(int(n_fold)):
            a = 2.0 * np.pi * k / n_fold
            R = np.array([[np.cos(a), -np.sin(a)], [np.sin(a), np.cos(a)]])
            ops.append(R @ np.diag([1.0, -1.0]) if mirror else R)
    group = np.full(N, -1, np.int32)
    xform = np.zeros((N, 4), np.float32)
    n_groups = 0
    for ref in range(N):
        if group[ref] >= 0:
            continue
        for Q in ops:
            img = Q @ xy[ref]
            for i in range(N):
                if group[i] < 0 and np.hypot(xy[i, 0] - img[0], xy[i, 1] - img[1]) <= tol:
                    group[i] = n_groups
                    xform[i] = Q.T.reshape(4).astype(np.float32)
                    break
        n_groups += 1
    return group, xform, n_groups


def fit_xy(sensor_xy, gains, knots_xy, n_lrf, n_int_x, n_int_y, signals, xyzA, group=None, xform=None,
           axial=None):
    """LRF calculation for XY tables ("XY LRF"; PAPER.md:380 LRFs are calculated from signals and
    positions) and for the XY component of a Composite LRF ("During LRF calculation, the axial
    component is evaluated first, and the residual is used to calculate the XY LRF component").  Reading R35 =
    R21-R23 carried to the sensor-local coordinates (u, v) = T_i (p - P_i) of R30/R33: unweighted least squares of
        y = S / (A g_i)                              (XY LRF)
        y = S / (A g_i) - s_ax,t(|p - P_i|)          (Composite: axial = (knots, n_int_r, coeffs [n_lrf][n_int_r+3]),
                                                      the axial spline with its argument clamped as in R5)
    against sum_b sum_a c[kv+b][ku+a] bv_b bu_a, over events with finite x, y, A and A > 0 and pairs with
    u_lo <= u <= u_hi and v_lo <= v <= v_hi; table t = group[i], or 0 / i without a grouping; g_i = 1 for per-sensor
    tables.  -> coefficients [n_lrf][n_int_y + 3][n_int_x + 3] (float64), pairs used [n_lrf].
    Raises numpy.linalg.LinAlgError when a table is underdetermined (a cell without data)."""
    xy = np.asarray(sensor_xy, np.float32).astype(np.float64).reshape(-1, 2)
    N = xy.shape[0]
    g = np.ones(N) if gains is None else np.asarray(gains, np.float32).astype(np.float64)
    u_lo, u_hi, v_lo, v_hi = (float(np.float32(k)) for k in knots_xy[:4])
    hu, hv = (u_hi - u_lo) / n_int_x, (v_hi - v_lo) / n_int_y
    ncu, ncv = n_int_x + 3, n_int_y + 3
    S = np.asarray(signals, np.float32).astype(np.float64).reshape(-1, N)
    P = np.asarray(xyzA, np.float32).astype(np.float64).reshape(-1, 4)
    T = None if xform is None else np.asarray(xform, np.float32).astype(np.float64).reshape(N, 4)
    ok = np.isfinite(P[:, 0]) & np.isfinite(P[:, 1]) & np.isfinite(P[:, 3]) & (P[:, 3] > 0.0)
    M = np.zeros((n_lrf, ncv * ncu, ncv * ncu))
    b = np.zeros((n_lrf, ncv * ncu))
    used = np.zeros(n_lrf)
    for i in range(N):
        if group is not None:
            m, gi = int(group[i]), g[i]
        else:
            m = 0 if n_lrf == 1 else i
            gi = g[i] if n_lrf == 1 else 1.0
        with np.errstate(invalid="ignore"):
            dx, dy = P[:, 0] - xy[i, 0], P[:, 1] - xy[i, 1]
            u, v = (dx, dy) if T is None else (T[i, 0] * dx + T[i, 1] * dy, T[i, 2] * dx + T[i, 3] * dy)
            use = ok & (u >= u_lo) & (u <= u_hi) & (v >= v_lo) & (v <= v_hi)
        y = S[use, i] / (P[use, 3] * gi)
        if axial is not None:
            a_knots, a_n, a_c = axial
            a_lo, a_hi = float(np.float32(a_knots[0])), float(np.float32(a_knots[1]))
            r = np.clip(np.hypot(dx[use], dy[use]), a_lo, a_hi)
            y = y - spline_values(np.asarray(a_c)[m], a_lo, a_hi, a_n, r)
        tu, tv = (u[use] - u_lo) / hu, (v[use] - v_lo) / hv
        ku = np.minimum(np.floor(tu).astype(np.int64), n_int_x - 1)
        kv = np.minimum(np.floor(tv).astype(np.int64), n_int_y - 1)
        Bu, Bv = basis4(tu - ku), basis4(tv - kv)
        idx = [((kv + bb) * ncu + ku + aa, Bv[:, bb] * Bu[:, aa]) for bb in range(4) for aa in range(4)]
        for j1, w1 in idx:
            np.add.at(b[m], j1, w1 * y)
            for j2, w2 in idx:
                np.add.at(M[m], (j1, j2), w1 * w2)
        used[m] += use.sum()
    c = np.stack([np.linalg.solve(M[m], b[m]).reshape(ncv, ncu) for m in range(n_lrf)])
    return c, used


def fit_sliced(sensor_xy, gains, knots_xy, n_lrf, n_int_x, n_int_y, n_planes, signals, xyzA, group=None, xform=None):
    """LRF calculation for Sliced tables ("a set of several XY LRFs, each defined on a specific Z
    plane.  The LRF values for the points between the planes are calculated using linear interpolation of the LRF
    values at two closest points from two closest planes"; PAPER.md:380 LRFs are calculated from signals and
    positions).  The paper does not say how the planes' tables are obtained; reading R36 = R21-R23 and R35 carried
    through the evaluation rule R32, all planes of a table fitted JOINTLY: unweighted least squares of
        y = S / (A g_i)   against   (1 - w) s_p(u, v) + w s_{p+1}(u, v),
    s_p the tensor-product spline of plane p, p = min(floor((z - z_lo)/dz), n_planes - 2), w = (z - z_p)/dz,
    dz = (z_hi - z_lo)/(n_planes - 1) -- exactly the value oracle_lrf returns for the pair -- over events with
    finite x, y, z, A, A > 0 and z_lo <= z <= z_hi (no extrapolation data, as in R25) and pairs with (u, v) inside the
    tabulated ranges; table t = group[i], or 0 / i without a grouping; g_i = 1 for per-sensor tables.
    knots_xy = {u_lo, u_hi, v_lo, v_hi, z_lo, z_hi}.
    -> coefficients [n_lrf][n_planes][n_int_y + 3][n_int_x + 3] (float64), pairs used [n_lrf].
    Raises numpy.linalg.LinAlgError when a table is underdetermined."""
    xy = np.asarray(sensor_xy, np.float32).astype(np.float64).reshape(-1, 2)
    N = xy.shape[0]
    g = np.ones(N) if gains is None else np.asarray(gains, np.float32).astype(np.float64)
    u_lo, u_hi, v_lo, v_hi, z_lo, z_hi = (float(np.float32(k)) for k in knots_xy[:6])
    hu, hv = (u_hi - u_lo) / n_int_x, (v_hi - v_lo) / n_int_y
    dz = (z_hi - z_lo) / (n_planes - 1)
    ncu, ncv = n_int_x + 3, n_int_y + 3
    per_plane = ncu * ncv
    n_unknown = n_planes * per_plane
    S = np.asarray(signals, np.float32).astype(np.float64).reshape(-1, N)
    P = np.asarray(xyzA, np.float32).astype(np.float64).reshape(-1, 4)
    T = None if xform is None else np.asarray(xform, np.float32).astype(np.float64).reshape(N, 4)
    with np.errstate(invalid="ignore"):
        ok = np.isfinite(P).all(axis=1) & (P[:, 3] > 0.0) & (P[:, 2] >= z_lo) & (P[:, 2] <= z_hi)
    M = np.zeros((n_lrf, n_unknown, n_unknown))
    b = np.zeros((n_lrf, n_unknown))
    used = np.zeros(n_lrf)
    for i in range(N):
        if group is not None:
            m, gi = int(group[i]), g[i]
        else:
            m = 0 if n_lrf == 1 else i
            gi = g[i] if n_lrf == 1 else 1.0
        with np.errstate(invalid="ignore"):
            dx, dy = P[:, 0] - xy[i, 0], P[:, 1] - xy[i, 1]
            u, v = (dx, dy) if T is None else (T[i, 0] * dx + T[i, 1] * dy, T[i, 2] * dx + T[i, 3] * dy)
            use = ok & (u >= u_lo) & (u <= u_hi) & (v >= v_lo) & (v <= v_hi)
        y = S[use, i] / (P[use, 3] * gi)
        z = P[use, 2]
        p = np.clip(np.floor((z - z_lo) / dz).astype(np.int64), 0, n_planes - 2)
        w = (z - (z_lo + p * dz)) / dz
        tu, tv = (u[use] - u_lo) / hu, (v[use] - v_lo) / hv
        ku = np.minimum(np.floor(tu).astype(np.int64), n_int_x - 1)
        kv = np.minimum(np.floor(tv).astype(np.int64), n_int_y - 1)
        Bu, Bv = basis4(tu - ku), basis4(tv - kv)
        idx = []
        for side, wz in ((0, 1.0 - w), (1, w)):
            for bb in range(4):
                for aa in range(4):
                    idx.append(((p + side) * per_plane + (kv + bb) * ncu + ku + aa, wz * Bv[:, bb] * Bu[:, aa]))
        for j1, w1 in idx:
            np.add.at(b[m], j1, w1 * y)
            for j2, w2 in idx:
                np.add.at(M[m], (j1, j2), w1 * w2)
        used[m] += use.sum()
    c = np.stack([np.linalg.solve(M[m], b[m]).reshape(n_planes, ncv, ncu) for m in range(n_lrf)])
    return c, used
