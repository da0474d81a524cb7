"""GPU-vs-oracle parity of the LRF calculation (ants_lrf_fit_axial vs oracle/fit.py), -m gpu, and the
reconstruct <-> refit cycle of PAPER.md:428 (section 8) on synthetic flood data.

Tolerance: both sides accumulate the normal equations in FP64 from the same float32 inputs and solve them
in FP64; they differ by summation order (atomics) only, ~1e-13 relative on M and b, amplified by the
conditioning of the spline normal matrix (<= ~1e4 here) and then rounded to float32 on output:
|c_gpu - c_oracle| <= 2e-6 max|c| per table.  Pair counts are integers: bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import fit as ofit                                 # noqa: E402
from paper_1602_07247_b200 import recon, synth                 # noqa: E402

TOL = 2e-6


def _reconstructed(idx, n):
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, n, device="cuda")
    r = recon.Reconstructor(cfg)
    try:
        xyzA, _ = r(ev["signals"])
        torch.cuda.synchronize()
    finally:
        r.close()
    return cfg, ev, xyzA


@pytest.mark.parametrize("idx,n", [(2, 60_011), (5, 12_007), (1, 9_001)])
def test_fit_parity_on_reconstructed_positions(idx, n):
    cfg, ev, xyzA = _reconstructed(idx, n)
    c, used = recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.n_lrf, cfg.n_int_r, ev["signals"], xyzA)
    c0, used0 = ofit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.n_lrf, cfg.n_int_r,
                               ev["signals"].cpu().numpy(), xyzA.cpu().numpy())
    assert np.array_equal(used, used0)
    assert np.abs(c - c0).max() <= TOL * np.abs(c0).max()


def test_fit_parity_individual_tables():
    """Per-sensor tables (config 3's sensors) with true positions spread so that every sensor sees its whole
    r-range; a tail of failed events (NaN rows) and events with non-positive energy must be ignored."""
    cfg = synth.make_config(3)
    rng = np.random.default_rng(5)
    E = 40_009
    pos = np.zeros((E, 4), np.float32)
    pos[:, :2] = rng.uniform(-55.0, 55.0, (E, 2))
    pos[:, 3] = rng.uniform(100.0, 400.0, E)
    r = np.hypot(pos[:, None, 0] - cfg.sensor_xy[None, :, 0], pos[:, None, 1] - cfg.sensor_xy[None, :, 1])
    mean = np.stack([synth.eval_axial(cfg.coeffs[i, 0], 0.0, 40.0, r[:, i].astype(float)) for i in range(64)], axis=1)
    sig = rng.poisson(np.maximum(pos[:, 3:4] * mean, 0.0)).astype(np.float32)
    pos[::13] = np.nan
    pos[5::17, 3] = 0.0
    c, used = recon.ants_lrf_fit_axial(cfg.sensor_xy, None, cfg.knots, 64, cfg.n_int_r,
                                       torch.from_numpy(sig).cuda(), torch.from_numpy(pos).cuda())
    c0, used0 = ofit.fit_axial(cfg.sensor_xy, None, cfg.knots, 64, cfg.n_int_r, sig, pos)
    assert np.array_equal(used, used0)
    assert (np.abs(c - c0).max(axis=1) <= TOL * np.abs(c0).max(axis=1)).all()
    # and the fit is near the truth it was drawn from (statistics, not parity)
    assert np.abs(c[:, 3:9] - cfg.coeffs[:, 0, 3:9]).max() < 0.05


def test_underdetermined_table_is_reported():
    cfg = synth.make_config(2)
    pos = torch.zeros((100, 4), device="cuda")
    pos[:, 3] = 1.0
    sig = torch.ones((100, cfg.n_sensors), device="cuda")
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, sig, pos)
    assert ei.value.status == -5
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, np.array([9.0, 1.0], np.float32), 1, cfg.n_int_r, sig, pos)
    assert ei.value.status == -1


def test_reconstruct_refit_cycle_recovers_the_response():
    """PAPER.md:428 (section 8): start from a WRONG response (profile 25 % too wide), alternate
    reconstruction and LRF calculation on flood data; the fitted profile moves to the true one."""
    true = synth.make_config(2)
    ev = synth.generate_events(true, 200_000, device="cuda")
    guess = synth.make_config(2)
    guess.coeffs = synth.fit_axial(lambda r: (1.0 + (r / 25.0) ** 2) ** -1.5, 0.0, 90.0, 16)[None, None, :]
    r_probe = np.linspace(2.0, 80.0, 40)
    truth = synth.eval_axial(true.coeffs[0, 0], 0.0, 90.0, r_probe)

    def shape_error(c):
        s = synth.eval_axial(np.asarray(c, np.float32), 0.0, 90.0, r_probe)
        s = s * (truth @ s) / (s @ s)              # the overall scale trades with the energy: compare shapes
        return float(np.abs(s - truth).max() / truth.max())

    from paper_1602_07247_b200 import iterate
    err = [shape_error(guess.coeffs[0, 0])]
    for cycle, cur, n_pass in iterate.iterate_response(guess, ev["signals"], 6, score_max=60.0):
        assert n_pass > 0.8 * ev["signals"].shape[0]
        err.append(shape_error(cur.coeffs[0, 0]))
    assert err[0] > 0.03 and err[-1] < 0.5 * err[0], err


@pytest.mark.parametrize("idx,n", [(2, 50_003), (5, 10_001)])
def test_gain_evaluation_parity_and_recovery(idx, n):
    """ants_lrf_fit_gains vs oracle.fit_gains on reconstructed positions (R24): FP64 sums on both sides,
    float32 output: 1e-6 relative; pair counts bit-exact.  The gains come back near the ones the data were
    drawn with (statistics, not parity)."""
    cfg, ev, xyzA = _reconstructed(idx, n)
    g, used = recon.ants_lrf_fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], ev["signals"], xyzA)
    g0, used0 = ofit.fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], cfg.n_int_r,
                               ev["signals"].cpu().numpy(), xyzA.cpu().numpy())
    assert np.array_equal(used, used0)
    assert np.abs(g - g0).max() <= 1e-6 * np.abs(g0).max()
    assert np.abs(g / cfg.gains - 1.0).max() < 0.1       # clipped noise lifts the far, dim pairs a few per cent


def test_gain_of_a_sensor_without_data_is_nan_gpu():
    cfg = synth.make_config(2)
    pos = torch.full((64, 4), 400.0, device="cuda")
    g, used = recon.ants_lrf_fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0],
                                       torch.ones((64, cfg.n_sensors), device="cuda"), pos)
    assert np.isnan(g).all() and (used == 0).all()


def test_axial_z_fit_parity():
    """ants_lrf_fit_axial_z vs oracle.fit_axial_z (R25) on true positions of flood data (the config's disk plus a wider
    one so that every (r, z) cell gets data), some failed rows and out-of-range z; 209 unknowns: tolerance 5e-6 of max|c|."""
    cfg = synth.make_config(4)
    E = 30_011
    ev = synth.generate_events(cfg, E, device="cuda")         # flood data of the config (positions inside the array)
    sig = ev["signals"].cpu().numpy()
    pos = np.zeros((E, 4), np.float32)
    pos[:, :3] = ev["true_xyz"].cpu().numpy()
    pos[:, 3] = 0.1 * ev["n_ph"].cpu().numpy()
    # widen: a second half of events far out so that every (r, z) cell gets data
    far = synth.make_config(4)
    far.extent = 200.0
    ev2 = synth.generate_events(far, E, device="cuda", batch=1)
    sig = np.concatenate([sig, ev2["signals"].cpu().numpy()])
    pos2 = np.zeros((E, 4), np.float32)
    pos2[:, :3] = ev2["true_xyz"].cpu().numpy()
    pos2[:, 3] = 0.1 * ev2["n_ph"].cpu().numpy()
    pos = np.concatenate([pos, pos2])
    pos[::19] = np.nan
    pos[3::23, 2] = 25.0                                       # z outside the LRF range: event ignored
    c, used = recon.ants_lrf_fit_axial_z(cfg.sensor_xy, cfg.gains, cfg.knots, 16, 8,
                                         torch.from_numpy(sig).cuda(), torch.from_numpy(pos).cuda())
    c0, used0 = ofit.fit_axial_z(cfg.sensor_xy, cfg.gains, cfg.knots, 16, 8, sig, pos)
    assert used == used0
    assert np.abs(c - c0).max() <= 5e-6 * np.abs(c0).max()
    # near the truth where the LRF is large (statistics, not parity)
    assert np.abs(c[2:8, 2:8] - cfg.coeffs[0, 2:8, 2:8]).max() < 0.1 * np.abs(cfg.coeffs[0, 2:8, 2:8]).max()


def test_event_filter_is_bit_exact_and_feeds_the_fit():
    """ants_filter_events vs oracle.filter_events (R26): the pass mask and the filtered array are identical
    bit for bit (integer decisions on the same float32 values); the filtered array then drives the fit."""
    cfg, ev, xyzA = _reconstructed(2, 40_003)
    r = recon.Reconstructor(cfg)
    try:
        xyzA, score = r(ev["signals"])
    finally:
        r.close()
    ref_keep, ref_out = ofit.filter_events(xyzA.cpu().numpy(), score.cpu().numpy(), score_max=30.0, energy_min=120.0,
                                           energy_max=450.0, radius_max=50.0)
    filt = xyzA.clone()
    n_pass = recon.ants_filter_events(filt, score, score_max=30.0, energy_min=120.0, energy_max=450.0, radius_max=50.0)
    out = filt.cpu().numpy()
    assert n_pass == int(ref_keep.sum()) and 0.2 * len(ref_keep) < n_pass < 0.95 * len(ref_keep)
    assert np.array_equal(np.isnan(out[:, 0]), ~ref_keep)
    assert np.array_equal(out[ref_keep], ref_out[ref_keep])
    none = xyzA.clone()
    assert recon.ants_filter_events(none, score) == int(torch.isfinite(xyzA[:, 0]).sum())       # all criteria off
    c, used = recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, ev["signals"], filt)
    c0, used0 = ofit.fit_axial(cfg.sensor_xy, cfg.gains, cfg.knots, 1, cfg.n_int_r, ev["signals"].cpu().numpy(), ref_out)
    assert np.array_equal(used, used0) and np.abs(c - c0).max() <= TOL * np.abs(c0).max()


def test_grouped_fit_parity_and_use_in_reconstruction():
    """ants_lrf_fit_axial_grouped vs the oracle (R28) with the distance groups of the 19-PMT array; the grouped
    response then goes straight into ants_lrf_create_grouped (one table per group in shared memory) and drives a
    reconstruction in parity with the oracle's grouped model."""
    cfg, ev, xyzA = _reconstructed(2, 60_011)
    group, n_groups = recon.ants_group_by_radius(cfg.sensor_xy)
    assert n_groups == 4 and np.array_equal(group, ofit.group_by_radius(cfg.sensor_xy)[0])
    knots = np.array([0.0, 55.0], np.float32)        # the range the central PMT sees with events inside 60 mm
    c, used = recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, knots, n_groups, cfg.n_int_r, ev["signals"], xyzA,
                                       group=group)
    c0, used0 = ofit.fit_axial(cfg.sensor_xy, cfg.gains, knots, n_groups, cfg.n_int_r,
                               ev["signals"].cpu().numpy(), xyzA.cpu().numpy(), group=group)
    assert np.array_equal(used, used0)
    assert (np.abs(c - c0).max(axis=1) <= TOL * np.abs(c0).max(axis=1)).all()
    with pytest.raises(recon.AntsError):
        recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, knots, n_groups, cfg.n_int_r, ev["signals"], xyzA,
                                 group=np.full(cfg.n_sensors, 7))
    import parity_rules
    grp = synth.make_config(2)
    grp.n_lrf = n_groups
    grp.group = group
    grp.knots = knots
    grp.coeffs = c[:, None, :].astype(np.float32)
    sub = ev["signals"][:8001].contiguous()
    r = recon.Reconstructor(grp)
    try:
        assert "recon2d_pk_kernel" in r.plan()["kernel"]
        out = [t.cpu().numpy() for t in r(sub, trace=True)]
    finally:
        r.close()
    parity_rules.assert_parity(parity_rules.compare(grp, sub.cpu().numpy(), *out), "grouped response")
    with pytest.raises(recon.AntsError) as ei:           # a group index outside 0 .. n_groups-1
        recon.ants_lrf_create_grouped(grp.sensor_xy, grp.gains, np.full(cfg.n_sensors, n_groups), grp.knots, grp.coeffs,
                                      recon.LrfDims(cfg.n_sensors, n_groups, 1, cfg.n_int_r, 0))
    assert ei.value.status == -1


@pytest.mark.parametrize("method,seed", [(0, 1), (1, 2), (2, 3)])
def test_grouped_model_on_random_groups(method, seed):
    """Random groups, gains and group profiles (chi-square variants included): a grouped handle reconstructs in
    parity with the oracle's grouped model."""
    import parity_rules
    rng = np.random.default_rng(seed)
    cfg = synth.make_config(5)
    n_groups = 5
    cfg.group = rng.integers(0, n_groups, cfg.n_sensors).astype(np.int32)
    cfg.n_lrf = n_groups
    base = cfg.coeffs[0, 0].astype(np.float64)
    cfg.coeffs = (base[None, :] * rng.uniform(0.7, 1.3, (n_groups, 1))).astype(np.float32)[:, None, :]
    cfg.method = method
    cfg.n_iter = 10
    ev = synth.generate_events(cfg, 3001, device="cuda:0")
    r = recon.Reconstructor(cfg)
    try:
        out = [t.cpu().numpy() for t in r(ev["signals"], trace=True)]
    finally:
        r.close()
    parity_rules.assert_parity(parity_rules.compare(cfg, ev["signals"].cpu().numpy(), *out), f"random groups m{method}")


def test_xy_and_composite_fit_parity():
    """ants_lrf_fit_xy vs the oracle (R35): one shared XY table with gains, D4 symmetry groups with frames, and the
    XY component of a Composite LRF fitted to the residual of a given axial component; the fitted tables go straight
    into ants_lrf_create_xy."""
    from test_oracle_fit import _xy_problem
    xy, gains, sig, pos = _xy_problem(40_003, seed=3, composite=True)
    knots = np.array([-12, 12, -12, 12], np.float32)
    nx, ny = 6, 5
    group, xform, n_groups = recon.ants_group_by_symmetry(xy, 4, True)
    sig_d, pos_d = torch.from_numpy(sig).cuda(), torch.from_numpy(pos).cuda()
    ax_knots, ax_n = np.array([0.0, 34.0], np.float32), 6
    ax_c = np.tile(synth.fit_axial(lambda r: 0.5 / (1.0 + r * r / 40.0), 0.0, 34.0, ax_n)[None, :], (n_groups, 1))
    for kw in (dict(n_lrf=1), dict(n_lrf=n_groups, group=group, xform=xform),
               dict(n_lrf=n_groups, group=group, xform=xform, axial=(ax_knots, ax_c))):
        c, used = recon.ants_lrf_fit_xy(xy, gains, knots, kw["n_lrf"], nx, ny, sig_d, pos_d, group=kw.get("group"),
                                        xform=kw.get("xform"), axial=kw.get("axial"))
        ax0 = None if "axial" not in kw else (ax_knots, ax_n, ax_c)
        c0, used0 = ofit.fit_xy(xy, gains, knots, kw["n_lrf"], nx, ny, sig, pos, group=kw.get("group"),
                                xform=kw.get("xform"), axial=ax0)
        assert np.array_equal(used, used0), kw.keys()
        scale = np.abs(c0).max(axis=(1, 2), keepdims=True)
        assert (np.abs(c - c0) <= 5e-6 * scale).all(), (kw.keys(), np.abs(c - c0).max())
    # the composite model built from the two fits reconstructs
    dims = recon.LrfDims(len(xy), n_groups, 4, ax_n, 0)
    h = recon.ants_lrf_create_xy(xy, gains, ax_knots, ax_c, dims, nx, ny, 0, knots, c, xform=xform, group=group)
    grid = recon.GridParams(2, 7, 2.0, 0.0, 0.5, 6, 0, float("nan"))
    out, score = torch.empty((256, 4), device="cuda"), torch.empty(256, device="cuda")
    recon.ants_reconstruct(h, sig_d[:256].contiguous(), grid, 1, out, score)
    torch.cuda.synchronize()
    recon.ants_destroy(h)
    assert torch.isfinite(out[:, :2]).all() and (out[:, :2].abs().max() <= 40.0)
    # a cell without data: the table is underdetermined
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_xy(xy, gains, np.array([-60, 60, -60, 60], np.float32), 1, 12, 12, sig_d, pos_d)
    assert ei.value.status == -5


def test_sliced_fit_parity():
    """ants_lrf_fit_sliced vs the oracle (R36): all planes of a table jointly; one shared table with gains and D4
    symmetry groups with frames; events outside the planes' range and failed events are left out; the fitted tables go
    straight into ants_lrf_create_xy (lrf_dim 5) and reconstruct in 3-D."""
    from test_oracle_fit import _sliced_problem
    xy, gains, sig, pos = _sliced_problem(30_011, seed=4)
    pos[17] = np.nan
    pos[101, 3] = -1.0
    knots = np.array([-12, 12, -12, 12, 0, 12], np.float32)
    nx, ny, n_planes = 5, 4, 4
    group, xform, n_groups = recon.ants_group_by_symmetry(xy, 4, True)
    sig_d, pos_d = torch.from_numpy(sig).cuda(), torch.from_numpy(pos).cuda()
    for kw in (dict(n_lrf=1), dict(n_lrf=n_groups, group=group, xform=xform)):
        c, used = recon.ants_lrf_fit_sliced(xy, gains, knots, kw["n_lrf"], nx, ny, n_planes, sig_d, pos_d,
                                            group=kw.get("group"), xform=kw.get("xform"))
        c0, used0 = ofit.fit_sliced(xy, gains, knots, kw["n_lrf"], nx, ny, n_planes, sig, pos, group=kw.get("group"),
                                    xform=kw.get("xform"))
        assert c.shape == c0.shape == (kw["n_lrf"], n_planes, ny + 3, nx + 3)
        assert np.array_equal(used, used0), kw.keys()
        scale = np.abs(c0).max(axis=(1, 2, 3), keepdims=True)
        assert (np.abs(c - c0) <= 5e-6 * scale).all(), (kw.keys(), np.abs(c - c0).max())
    dims = recon.LrfDims(len(xy), n_groups, 5, 0, 0)
    h = recon.ants_lrf_create_xy(xy, gains, None, None, dims, nx, ny, n_planes, knots, c, xform=xform, group=group)
    grid = recon.GridParams(3, 5, 2.0, 1.5, 0.5, 6, 0, 6.0)
    out, score = torch.empty((256, 4), device="cuda"), torch.empty(256, device="cuda")
    recon.ants_reconstruct(h, sig_d[:256].contiguous(), grid, 0, out, score)
    torch.cuda.synchronize()
    recon.ants_destroy(h)
    ok = torch.isfinite(out[:, 0])
    assert ok.float().mean() > 0.9 and (out[ok, :2].abs().max() <= 40.0)
    # a plane without data: underdetermined
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_sliced(xy, gains, np.array([-12, 12, -12, 12, 0, 40], np.float32), 1, nx, ny, n_planes, sig_d, pos_d)
    assert ei.value.status == -5
    # limits
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_sliced(xy, gains, knots, 1, nx, ny, 1, sig_d, pos_d)
    assert ei.value.status == -1                     # ANTS_ERR_INVALID: a Sliced LRF has at least two planes


def test_sliced_fit_at_config7_table_sizes():
    """Config 7's own tables (5 planes of 23 x 23 coefficients: 2,645 unknowns, banded solve) from 200 k synthetic
    events at their true positions: the well-covered centre of every plane comes back within the Poisson noise, and
    the pair count is the definition's."""
    cfg = synth.make_config(7)
    ev = synth.generate_events(cfg, 200_000)
    sig = ev["signals"].cuda().contiguous()
    pos_h = torch.cat([ev["true_xyz"], 0.1 * ev["n_ph"][:, None]], 1).float().contiguous()
    c, used = recon.ants_lrf_fit_sliced(cfg.sensor_xy, cfg.gains, cfg.knots_xy, 1, cfg.n_int_x, cfg.n_int_y, cfg.n_planes,
                                        sig, pos_h.cuda())
    assert c.shape == cfg.coeffs_xy.shape
    p = pos_h.numpy().astype(np.float64)
    xy = cfg.sensor_xy.astype(np.float64)
    inside = (p[:, 2] >= 0.0) & (p[:, 2] <= 20.0)
    du, dv = p[:, None, 0] - xy[None, :, 0], p[:, None, 1] - xy[None, :, 1]
    n_pairs = (inside[:, None] & (np.abs(du) <= 120.0) & (np.abs(dv) <= 120.0)).sum()
    assert used[0] == n_pairs
    d = np.abs(c - cfg.coeffs_xy)[0, :, 6:17, 6:17]
    assert d.max() <= 0.05, d.max()                       # coefficients there are 0.3 .. 7.8
    # one reconstruct -> filter -> refit cycle of the iterative loop on the Sliced model
    from paper_1602_07247_b200 import iterate
    (cycle, cur, n_pass), = list(iterate.iterate_response(cfg, sig, 1))
    assert n_pass > 0.9 * sig.shape[0] and cur.coeffs_xy.shape == cfg.coeffs_xy.shape
    d = np.abs(cur.coeffs_xy - cfg.coeffs_xy)[0, :, 6:17, 6:17]
    assert d.max() <= 0.4, d.max()                        # reconstructed positions: resolution smears the peak
