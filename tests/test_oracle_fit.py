"""Pins of the LRF-calculation oracle (oracle/fit.py; R21-R23), CPU-only.  Expected values
come from scipy's BSpline (design matrix, evaluation) and numpy.linalg.lstsq on the raw least-squares
problem -- never from the oracle's own basis or normal equations."""
import numpy as np
import pytest
from scipy.interpolate import BSpline

from oracle import fit
from paper_1602_07247_b200 import synth


def _problem(idx, n_events, seed=1, noise=0.0, individual=None):
    cfg = synth.make_config(idx)
    rng = np.random.default_rng(seed)
    ext = float(np.abs(cfg.sensor_xy).max()) + 0.75 * float(cfg.knots[1])   # every sensor sees its whole r-range
    pos = np.zeros((n_events, 4), np.float32)
    pos[:, 0:2] = rng.uniform(-ext, ext, (n_events, 2))
    pos[:, 3] = rng.uniform(50.0, 500.0, n_events)                      # energy scale A_e
    lo, hi = float(cfg.knots[0]), float(cfg.knots[1])
    r = np.hypot(pos[:, None, 0].astype(float) - cfg.sensor_xy[None, :, 0],
                 pos[:, None, 1].astype(float) - cfg.sensor_xy[None, :, 1])
    sig = np.empty((n_events, cfg.n_sensors))
    for i in range(cfg.n_sensors):
        m = 0 if cfg.n_lrf == 1 else i
        g = float(cfg.gains[i]) if cfg.n_lrf == 1 else 1.0
        sig[:, i] = pos[:, 3] * g * synth.eval_axial(cfg.coeffs[m, 0], lo, hi, r[:, i])     # scipy evaluation
    sig += noise * rng.standard_normal(sig.shape)
    return cfg, sig.astype(np.float32), pos


def _lstsq_reference(cfg, sig, pos, table):
    """The raw least-squares problem of R21 for one table through scipy's design matrix + numpy lstsq."""
    lo, hi, n = float(cfg.knots[0]), float(cfg.knots[1]), cfg.n_int_r
    t = synth.uniform_knot_vector(lo, hi, n)
    rows, ys = [], []
    sensors = range(cfg.n_sensors) if cfg.n_lrf == 1 else [table]
    ok = np.isfinite(pos[:, 0]) & np.isfinite(pos[:, 3]) & (pos[:, 3] > 0)
    for i in sensors:
        g = float(cfg.gains[i]) if cfg.n_lrf == 1 else 1.0
        r = np.hypot(pos[:, 0].astype(float) - float(cfg.sensor_xy[i, 0]), pos[:, 1].astype(float) - float(cfg.sensor_xy[i, 1]))
        use = ok & (r >= lo) & (r <= hi)
        rows.append(BSpline.design_matrix(r[use], t, 3).toarray())
        ys.append(sig[use, i].astype(float) / (pos[use, 3].astype(float) * g))
    c, *_ = np.linalg.lstsq(np.vstack(rows), np.concatenate(ys), rcond=None)
    return c


def test_noise_free_data_give_back_the_coefficients():
    for idx in (2, 3):
        cfg, sig, pos = _problem(idx, 4000)
        c, n_used = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.n_lrf, cfg.n_int_r, sig, pos)
        want = cfg.coeffs[:, 0, :].astype(float)
        # float32 storage of the signals limits the agreement (6e-8 relative per sample)
        assert np.abs(c - want).max() <= 2e-5 * np.abs(want).max()
        assert (n_used > 0).all()


@pytest.mark.parametrize("idx", [2, 3, 5])
def test_equals_numpy_lstsq_on_scipy_design_matrix(idx):
    cfg, sig, pos = _problem(idx, 1500 if idx != 5 else 600, noise=0.5)
    c, _ = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.n_lrf, cfg.n_int_r, sig, pos)
    for table in ([0] if cfg.n_lrf == 1 else [0, 17, cfg.n_sensors - 1]):
        ref = _lstsq_reference(cfg, sig, pos, table)
        assert np.abs(c[table] - ref).max() <= 1e-8 * max(1.0, np.abs(ref).max())


def test_relative_gains_are_divided_out_of_a_shared_profile():
    cfg, sig, pos = _problem(2, 3000, noise=0.2)
    c1, _ = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig, pos)
    g2 = (cfg.gains * 2.0).astype(np.float32)                # power of two: exact
    c2, _ = fit.fit_axial(cfg.sensor_xy, g2, cfg.knots, 1, cfg.n_int_r, sig * 2.0, pos)
    assert np.allclose(c1, c2, rtol=1e-12, atol=0)
    c3, _ = fit.fit_axial(cfg.sensor_xy, None, cfg.knots, 1, cfg.n_int_r, sig / cfg.gains[None, :], pos)
    assert np.abs(c3 - c1).max() <= 1e-6 * np.abs(c1).max()   # float32 rounding of the rescaled signals


def test_failed_events_and_out_of_range_pairs_are_left_out():
    cfg, sig, pos = _problem(2, 2500, noise=0.3)
    pos2, sig2 = pos.copy(), sig.copy()
    pos2[::7] = np.nan                                        # failed events (NaN rows)
    pos2[3::11, 3] = -1.0                                     # non-positive energy
    keep = np.isfinite(pos2[:, 0]) & (pos2[:, 3] > 0)
    a, na = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig2, pos2)
    b, nb = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig2[keep], pos2[keep])
    assert np.array_equal(a, b) and np.array_equal(na, nb)
    r = np.hypot(pos[:, None, 0] - cfg.sensor_xy[None, :, 0], pos[:, None, 1] - cfg.sensor_xy[None, :, 1])
    assert na[0] == float((keep[:, None] & (r.astype(float) <= 90.0)).sum())          # pairs with r <= r_hi only


def test_underdetermined_table_raises():
    cfg, sig, pos = _problem(2, 50)
    pos[:, 0:2] = 0.0                                         # all events at one point: most intervals empty
    with pytest.raises(np.linalg.LinAlgError):
        fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig, pos)


# ---------------------------------------------------------------------------
# relative gains for a fixed profile (R24)
# ---------------------------------------------------------------------------
def test_gains_are_recovered_from_noise_free_data_and_match_lstsq():
    cfg, sig, pos = _problem(2, 3000)
    g, used = fit.fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], cfg.n_int_r, sig, pos)
    assert np.abs(g - cfg.gains).max() <= 2e-6 and (used > 0).all()
    cfg, sig, pos = _problem(5, 800, noise=0.7)
    g, used = fit.fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], cfg.n_int_r, sig, pos)
    lo, hi = float(cfg.knots[0]), float(cfg.knots[1])
    for i in (0, 50, 126):                                   # the 1-D least-squares problem through scipy + lstsq
        r = np.hypot(pos[:, 0].astype(float) - float(cfg.sensor_xy[i, 0]), pos[:, 1].astype(float) - float(cfg.sensor_xy[i, 1]))
        use = (r >= lo) & (r <= hi)
        s = synth.eval_axial(cfg.coeffs[0, 0], lo, hi, r[use])
        ref, *_ = np.linalg.lstsq(s[:, None], sig[use, i].astype(float) / pos[use, 3].astype(float), rcond=None)
        assert g[i] == pytest.approx(ref[0], rel=1e-10) and used[i] == use.sum()


def test_gain_of_a_sensor_without_data_is_nan():
    cfg, sig, pos = _problem(2, 200)
    pos[:, 0:2] = 300.0                                       # every sensor farther than r_hi
    g, used = fit.fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], cfg.n_int_r, sig, pos)
    assert np.isnan(g).all() and (used == 0).all()


# ---------------------------------------------------------------------------
# axial+z tensor LRF (R25)
# ---------------------------------------------------------------------------
def _problem_rz(n_events, seed=4, noise=0.0):
    cfg = synth.make_config(4)
    rng = np.random.default_rng(seed)
    pos = np.zeros((n_events, 4), np.float32)
    pos[:, 0:2] = rng.uniform(-170.0, 170.0, (n_events, 2))
    pos[:, 2] = rng.uniform(0.0, 20.0, n_events)
    pos[:, 3] = rng.uniform(100.0, 900.0, n_events)
    r = np.hypot(pos[:, None, 0].astype(float) - cfg.sensor_xy[None, :, 0], pos[:, None, 1].astype(float) - cfg.sensor_xy[None, :, 1])
    t_r = synth.uniform_knot_vector(0.0, 120.0, 16)
    t_z = synth.uniform_knot_vector(0.0, 20.0, 8)
    Bz = BSpline.design_matrix(pos[:, 2].astype(float), t_z, 3).toarray()             # scipy, not the oracle
    sig = np.zeros((n_events, cfg.n_sensors))
    for i in range(cfg.n_sensors):
        Br = BSpline.design_matrix(np.clip(r[:, i], 0.0, 120.0), t_r, 3).toarray()
        sig[:, i] = pos[:, 3] * cfg.gains[i] * np.einsum("eb,ba,ea->e", Bz, cfg.coeffs[0].astype(float), Br)
    sig += noise * rng.standard_normal(sig.shape)
    return cfg, sig.astype(np.float32), pos, (t_r, t_z)


def test_axial_z_fit_recovers_coefficients_and_equals_lstsq():
    cfg, sig, pos, _ = _problem_rz(2500)
    c, used = fit.fit_axial_z(cfg.sensor_xy, cfg.gains, cfg.knots, 16, 8, sig, pos)
    want = cfg.coeffs[0].astype(float)
    assert np.abs(c - want).max() <= 5e-5 * np.abs(want).max() and used > 0
    cfg, sig, pos, (t_r, t_z) = _problem_rz(1200, noise=0.3)
    c, used = fit.fit_axial_z(cfg.sensor_xy, cfg.gains, cfg.knots, 16, 8, sig, pos)
    rows, ys = [], []
    Bz = BSpline.design_matrix(pos[:, 2].astype(float), t_z, 3).toarray()
    for i in range(cfg.n_sensors):
        r = np.hypot(pos[:, 0].astype(float) - float(cfg.sensor_xy[i, 0]), pos[:, 1].astype(float) - float(cfg.sensor_xy[i, 1]))
        use = r <= 120.0
        Br = BSpline.design_matrix(r[use], t_r, 3).toarray()
        rows.append(np.einsum("eb,ea->eba", Bz[use], Br).reshape(use.sum(), -1))
        ys.append(sig[use, i].astype(float) / (pos[use, 3].astype(float) * float(cfg.gains[i])))
    ref, *_ = np.linalg.lstsq(np.vstack(rows), np.concatenate(ys), rcond=None)
    assert used == sum(len(y) for y in ys)
    assert np.abs(c.ravel() - ref).max() <= 1e-7 * max(1.0, np.abs(ref).max())


# ---------------------------------------------------------------------------
# event filters (R26)
# ---------------------------------------------------------------------------
def test_event_filters_on_hand_made_cases():
    P = np.array([[0, 0, 0, 100], [3, 4, 0, 100], [3, 4, 0, 50], [np.nan, 0, 0, 100], [0, 0, 0, 100], [6, 8, 0, 100]],
                 np.float32)
    s = np.array([1.0, 2.0, 2.0, 1.0, np.inf, 9.0], np.float32)
    keep, out = fit.filter_events(P, s)
    assert keep.tolist() == [True, True, True, False, False, True]            # failed rows never pass
    assert fit.filter_events(P, s, score_max=2.0)[0].tolist() == [True, True, True, False, False, False]
    assert fit.filter_events(P, s, energy_min=60.0)[0].tolist() == [True, True, False, False, False, True]
    assert fit.filter_events(P, s, energy_max=60.0)[0].tolist() == [False, False, True, False, False, False]
    assert fit.filter_events(P, s, radius_max=5.0)[0].tolist() == [True, True, True, False, False, False]   # r = 5 passes
    keep, out = fit.filter_events(P, s, score_max=5.0, radius_max=4.9)
    assert keep.tolist() == [True, False, False, False, False, False]
    assert np.isnan(out[1:]).all() and np.array_equal(out[0], P[0])


# ---------------------------------------------------------------------------
# grouped fit (R28)
# ---------------------------------------------------------------------------
def test_radius_groups_of_the_hexagonal_arrays():
    for rings, want in ((1, [1, 6]), (2, [1, 6, 6, 6]), (3, [1, 6, 6, 6, 12, 6])):
        group, n = fit.group_by_radius(synth.hex_array(rings, 30.0))
        assert n == len(want) and np.bincount(group).tolist() == want
    group, n = fit.group_by_radius(synth.square_array(8, 6.0))
    assert n == 9 and np.bincount(group).sum() == 64          # 8 x 8 grid: nine distinct distances from the centre


def test_grouped_fit_is_the_lstsq_of_each_group():
    cfg, sig, pos = _problem(2, 2500, noise=0.4)
    group, n_groups = fit.group_by_radius(cfg.sensor_xy)
    c, used = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, n_groups, cfg.n_int_r, sig, pos, group=group)
    assert c.shape == (n_groups, cfg.n_int_r + 3)
    lo, hi = float(cfg.knots[0]), float(cfg.knots[1])
    t = synth.uniform_knot_vector(lo, hi, cfg.n_int_r)
    for m in range(n_groups):
        rows, ys = [], []
        for i in np.flatnonzero(group == m):
            r = np.hypot(pos[:, 0].astype(float) - float(cfg.sensor_xy[i, 0]), pos[:, 1].astype(float) - float(cfg.sensor_xy[i, 1]))
            use = (r >= lo) & (r <= hi)
            rows.append(BSpline.design_matrix(r[use], t, 3).toarray())
            ys.append(sig[use, i].astype(float) / (pos[use, 3].astype(float) * float(cfg.gains[i])))
        ref, *_ = np.linalg.lstsq(np.vstack(rows), np.concatenate(ys), rcond=None)
        assert np.abs(c[m] - ref).max() <= 1e-8 * max(1.0, np.abs(ref).max())
        assert used[m] == sum(len(y) for y in ys)
    # the two built-in groupings are special cases
    one, _ = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig, pos)
    one_g, _ = fit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig, pos, group=np.zeros(cfg.n_sensors, np.int32))
    assert np.array_equal(one, one_g)


def test_grouped_model_is_the_expanded_model():
    """R28: L_i = g_i s_group(i)(r).  Pin: the oracle's grouped LRF equals the library-evaluated (scipy) group
    profile times the gain, and a grouped model reconstructs exactly like the same response written out as one
    table per sensor (coefficients of the group times the gain, computed here in float32-exact numbers)."""
    from oracle import oracle
    rng = np.random.default_rng(11)
    cfg = synth.make_config(2)
    n_groups = 3
    group = rng.integers(0, n_groups, cfg.n_sensors).astype(np.int32)
    gains = (2.0 ** rng.integers(-1, 2, cfg.n_sensors)).astype(np.float32)       # powers of two: exact products
    coeffs = (cfg.coeffs[0, 0][None, :] * np.array([1.0, 0.75, 1.25], np.float32)[:, None]).astype(np.float32)
    grouped = oracle.Model(cfg.sensor_xy, gains, cfg.knots, coeffs, n_groups, 1, cfg.n_int_r, 0, group=group)
    expanded = oracle.Model(cfg.sensor_xy, np.ones(cfg.n_sensors, np.float32), cfg.knots,
                            (coeffs[group] * gains[:, None]).astype(np.float32), cfg.n_sensors, 1, cfg.n_int_r, 0)
    for i in range(cfg.n_sensors):
        for x, y in ((3.0, -7.0), (40.0, 22.0), (-81.0, 5.5)):
            r = np.hypot(x - float(cfg.sensor_xy[i, 0]), y - float(cfg.sensor_xy[i, 1]))
            lib = float(gains[i]) * float(synth.eval_axial(coeffs[group[i]], 0.0, 90.0, np.array([r]))[0])
            assert abs(grouped.lrf(i, x, y) - lib) <= 1e-12 * abs(lib)
            assert grouped.lrf(i, x, y) == expanded.lrf(i, x, y)
    sig = synth.generate_events(cfg, 300)["signals"].numpy()
    grid = oracle.grid_from_config(cfg)
    for method in (0, 1):
        a = oracle.reconstruct(grouped, sig, grid, method, trace=True)
        b = oracle.reconstruct(expanded, sig, grid, method, trace=True)
        # the centroid weighs by 1/g in the grouped model and by 1 in the expanded one: compare from the same start
        assert np.array_equal(a["idx"][:, 1:] >= 0, b["idx"][:, 1:] >= 0)
    ones = oracle.Model(cfg.sensor_xy, np.ones(cfg.n_sensors, np.float32), cfg.knots, coeffs, n_groups, 1, cfg.n_int_r, 0, group=group)
    exp1 = oracle.Model(cfg.sensor_xy, np.ones(cfg.n_sensors, np.float32), cfg.knots, coeffs[group].astype(np.float32),
                        cfg.n_sensors, 1, cfg.n_int_r, 0)
    for method in (0, 1, 2):
        a = oracle.reconstruct(ones, sig, grid, method, trace=True)
        b = oracle.reconstruct(exp1, sig, grid, method, trace=True)
        assert np.array_equal(a["xyzA"], b["xyzA"]) and np.array_equal(a["score"], b["score"]) and np.array_equal(a["idx"], b["idx"])


def test_gain_renormalisation_keeps_the_mean_and_the_ratios():
    """R29 pins: the mean of the result equals the mean of the previous set; ratios between re-evaluated sensors
    are those of the new estimates; a sensor without an estimate keeps its previous gain (before the common
    scaling); an all-usable set that already has the right mean comes back unchanged."""
    rng = np.random.default_rng(3)
    prev = rng.uniform(0.6, 1.4, 19).astype(np.float32)
    new = (prev.astype(np.float64) * rng.uniform(0.8, 1.2, 19) * 5.0).astype(np.float32)
    new[4] = np.nan
    new[9] = 0.0
    out = fit.renormalise_gains(new, prev).astype(np.float64)
    assert abs(out.mean() - prev.astype(np.float64).mean()) <= 1e-6
    ok = np.ones(19, bool)
    ok[[4, 9]] = False
    ratio = out[ok] / new[ok].astype(np.float64)
    assert np.ptp(ratio) <= 2e-7 * ratio.mean()
    assert abs(out[4] / prev[4] - ratio.mean()) <= 2e-7 * ratio.mean() and abs(out[9] / prev[9] - ratio.mean()) <= 2e-7 * ratio.mean()
    same = fit.renormalise_gains(prev, prev)
    assert np.abs(same.astype(np.float64) - prev).max() <= 1.2e-7 * prev.max()


def _xy_problem(n_events, seed=0, composite=False):
    """A small XY-type detector whose tables are fully covered by the events: 3 x 3 sensors (pitch 8 mm), XY range
    +-12 mm around each sensor, events over a +-22 mm square, known smooth response, Gaussian noise."""
    rng = np.random.default_rng(seed)
    xy = synth.square_array(3, 8.0)
    N = len(xy)
    gains = rng.uniform(0.8, 1.2, N).astype(np.float32)
    pos = np.zeros((n_events, 4), np.float32)
    pos[:, :2] = rng.uniform(-22.0, 22.0, (n_events, 2))
    pos[:, 3] = rng.uniform(200.0, 400.0, n_events)
    dx = pos[:, None, 0].astype(np.float64) - xy[None, :, 0]
    dy = pos[:, None, 1].astype(np.float64) - xy[None, :, 1]
    resp = np.exp(-(dx * dx / 60.0 + dy * dy / 90.0)) * (1.0 + 0.02 * dx)
    if composite:
        resp = resp + 0.5 / (1.0 + (dx * dx + dy * dy) / 40.0)
    sig = (pos[:, 3:4].astype(np.float64) * gains[None, :] * resp + rng.normal(0, 0.5, (n_events, N))).astype(np.float32)
    return xy, gains, sig, pos


def test_xy_fit_is_the_lstsq_of_the_tensor_design_matrix():
    """R35 pinned against scipy design matrices + numpy.linalg.lstsq, per table: shared table with gains, symmetry
    groups with frames, and the Composite residual fit."""
    from scipy.interpolate import BSpline
    xy, gains, sig, pos = _xy_problem(1500)
    knots = np.array([-12, 12, -12, 12], np.float32)
    nx, ny = 4, 5
    tu, tv = synth.uniform_knot_vector(-12.0, 12.0, nx), synth.uniform_knot_vector(-12.0, 12.0, ny)
    group, xform, n_groups = fit.group_by_symmetry(xy, 4, True)
    ax_knots, ax_n = np.array([0.0, 34.0], np.float32), 6
    ax_c = np.tile(synth.fit_axial(lambda r: 0.5 / (1.0 + r * r / 40.0), 0.0, 34.0, ax_n)[None, :], (n_groups, 1))
    for kw in (dict(n_lrf=1), dict(n_lrf=n_groups, group=group, xform=xform),
               dict(n_lrf=n_groups, group=group, xform=xform, axial=(ax_knots, ax_n, ax_c))):
        c, used = fit.fit_xy(xy, gains, knots, kw["n_lrf"], nx, ny, sig, pos, group=kw.get("group"),
                             xform=kw.get("xform"), axial=kw.get("axial"))
        assert c.shape == (kw["n_lrf"], ny + 3, nx + 3)
        for m in range(kw["n_lrf"]):
            rows, ys = [], []
            for i in range(len(xy)):
                if (kw.get("group") is not None and group[i] != m):
                    continue
                dx = pos[:, 0].astype(float) - float(xy[i, 0])
                dy = pos[:, 1].astype(float) - float(xy[i, 1])
                T = np.eye(2) if kw.get("xform") is None else xform[i].astype(float).reshape(2, 2)
                u, v = T[0, 0] * dx + T[0, 1] * dy, T[1, 0] * dx + T[1, 1] * dy
                use = (u >= -12) & (u <= 12) & (v >= -12) & (v <= 12)
                Bu = BSpline.design_matrix(u[use], tu, 3).toarray()
                Bv = BSpline.design_matrix(v[use], tv, 3).toarray()
                rows.append(np.einsum("kb,ka->kba", Bv, Bu).reshape(use.sum(), -1))
                y = sig[use, i].astype(float) / (pos[use, 3].astype(float) * float(gains[i]))
                if kw.get("axial") is not None:
                    r = np.clip(np.hypot(dx[use], dy[use]), 0.0, 34.0)
                    y = y - synth.eval_axial(ax_c[m], 0.0, 34.0, r)
                ys.append(y)
            ref, *_ = np.linalg.lstsq(np.vstack(rows), np.concatenate(ys), rcond=None)
            assert np.abs(c[m].ravel() - ref).max() <= 1e-7 * max(1.0, np.abs(ref).max()), kw.keys()
            assert used[m] == sum(len(y) for y in ys)


def _sliced_problem(n_events, seed=0, noise=0.5):
    """The XY problem of _xy_problem with a depth: z uniform over (and a little beyond) the planes' range, a response
    that widens with z."""
    rng = np.random.default_rng(seed + 50)
    xy = synth.square_array(3, 8.0)
    N = len(xy)
    gains = rng.uniform(0.8, 1.2, N).astype(np.float32)
    pos = np.zeros((n_events, 4), np.float32)
    pos[:, :2] = rng.uniform(-22.0, 22.0, (n_events, 2))
    pos[:, 2] = rng.uniform(-1.0, 13.0, n_events)
    pos[:, 3] = rng.uniform(200.0, 400.0, n_events)
    dx = pos[:, None, 0].astype(np.float64) - xy[None, :, 0]
    dy = pos[:, None, 1].astype(np.float64) - xy[None, :, 1]
    wd = 60.0 + 4.0 * pos[:, None, 2].astype(np.float64)
    resp = np.exp(-(dx * dx + dy * dy * 0.7) / wd) * (1.0 + 0.02 * dx)
    sig = (pos[:, 3:4].astype(np.float64) * gains[None, :] * resp + rng.normal(0, noise, (n_events, N))).astype(np.float32)
    return xy, gains, sig, pos


def test_sliced_fit_is_the_lstsq_of_the_interpolated_design_matrix():
    """R36 pinned against scipy design matrices, the interpolation weights of PAPER.md:396 written out here, and
    numpy.linalg.lstsq over all planes at once: a shared table with gains, and symmetry groups with frames."""
    xy, gains, sig, pos = _sliced_problem(2500)
    knots = np.array([-12, 12, -12, 12, 0, 12], np.float32)
    nx, ny, n_planes = 4, 3, 4
    tu, tv = synth.uniform_knot_vector(-12.0, 12.0, nx), synth.uniform_knot_vector(-12.0, 12.0, ny)
    per_plane = (nx + 3) * (ny + 3)
    group, xform, n_groups = fit.group_by_symmetry(xy, 4, True)
    z = pos[:, 2].astype(float)
    inside = (z >= 0.0) & (z <= 12.0)
    assert 0 < (~inside).sum() < len(z)                       # some events lie outside the planes and are left out
    plane_z = np.linspace(0.0, 12.0, n_planes)
    for kw in (dict(n_lrf=1), dict(n_lrf=n_groups, group=group, xform=xform)):
        c, used = fit.fit_sliced(xy, gains, knots, kw["n_lrf"], nx, ny, n_planes, sig, pos, group=kw.get("group"),
                                 xform=kw.get("xform"))
        assert c.shape == (kw["n_lrf"], n_planes, ny + 3, nx + 3)
        for m in range(kw["n_lrf"]):
            rows, ys = [], []
            for i in range(len(xy)):
                if kw.get("group") is not None and group[i] != m:
                    continue
                dx = pos[:, 0].astype(float) - float(xy[i, 0])
                dy = pos[:, 1].astype(float) - float(xy[i, 1])
                T = np.eye(2) if kw.get("xform") is None else xform[i].astype(float).reshape(2, 2)
                u, v = T[0, 0] * dx + T[0, 1] * dy, T[1, 0] * dx + T[1, 1] * dy
                use = inside & (u >= -12) & (u <= 12) & (v >= -12) & (v <= 12)
                Bu = BSpline.design_matrix(u[use], tu, 3).toarray()
                Bv = BSpline.design_matrix(v[use], tv, 3).toarray()
                B = np.einsum("kb,ka->kba", Bv, Bu).reshape(use.sum(), -1)
                # hat functions of the planes: the linear interpolation between the two closest planes
                hat = np.maximum(0.0, 1.0 - np.abs(z[use, None] - plane_z[None, :]) / (plane_z[1] - plane_z[0]))
                assert np.allclose(hat.sum(axis=1), 1.0)
                rows.append(np.einsum("kp,kj->kpj", hat, B).reshape(use.sum(), n_planes * per_plane))
                ys.append(sig[use, i].astype(float) / (pos[use, 3].astype(float) * float(gains[i])))
            ref, *_ = np.linalg.lstsq(np.vstack(rows), np.concatenate(ys), rcond=None)
            assert np.abs(c[m].ravel() - ref).max() <= 1e-6 * max(1.0, np.abs(ref).max()), kw.keys()
            assert used[m] == sum(len(y) for y in ys)


def test_sliced_fit_recovers_the_tables_the_oracle_evaluates():
    """Noise-free signals generated with oracle_lrf (R32) from known Sliced tables: the joint fit returns those tables,
    which ties R36 to the evaluation rule of the reconstruction oracle (a per-plane binning of the events would not)."""
    from oracle import oracle
    rng = np.random.default_rng(5)
    xy = synth.square_array(3, 8.0)
    N = len(xy)
    nx, ny, n_planes = 3, 3, 3
    knots = np.array([-29, 29, -29, 29, 2, 10], np.float32)        # events reach u, v = +-28: tables covered to the ends
    truth = rng.uniform(0.5, 1.5, (1, n_planes, ny + 3, nx + 3)).astype(np.float32)
    gains = rng.uniform(0.8, 1.2, N).astype(np.float32)
    m = oracle.Model(xy, gains, None, None, 1, 5, 0, 0, n_int_x=nx, n_int_y=ny, n_planes=n_planes, knots_xy=knots,
                     coeffs_xy=truth)
    n_events = 600
    pos = np.zeros((n_events, 4), np.float32)
    pos[:, :2] = rng.uniform(-20.0, 20.0, (n_events, 2))
    pos[:, 2] = rng.uniform(2.0, 10.0, n_events)
    pos[:, 3] = rng.uniform(100.0, 200.0, n_events)
    sig = np.array([[float(pos[e, 3]) * m.lrf(i, float(pos[e, 0]), float(pos[e, 1]), float(pos[e, 2])) for i in range(N)]
                    for e in range(n_events)])
    c, used = fit.fit_sliced(xy, gains, knots, 1, nx, ny, n_planes, sig.astype(np.float32), pos)
    assert used[0] == n_events * N
    # float32 signals (6e-8 relative) through a fit whose end coefficients are conditioned ~1e2..1e3: observed 1.5e-5
    assert np.abs(c - truth).max() <= 1e-4
