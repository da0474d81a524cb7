"""Pins of the oracle's sensor selection (R19): passive photosensors (section 5.3)
and the per-event options of PAPER.md:318 (ignore sensors below a signal threshold or farther than a
given distance from the initial search position).  CPU-only.  Expected values come from the already
pinned unselected path on a model rebuilt WITHOUT the ignored sensors, and from a numpy/scipy evaluation
written here -- never from the selection code itself."""
import numpy as np
import pytest

from oracle import oracle
from paper_1602_07247_b200 import synth
from test_oracle_pins import lib_score   # scipy-based score written independently of the oracle


def _events(idx, n, **kw):
    cfg = synth.make_config(idx)
    return cfg, synth.generate_events(cfg, n, device="cpu", **kw)["signals"].numpy()


def _subset_config(cfg, keep):
    """The same detector with only the sensors `keep`: what 'ignoring' the others must equal."""
    sub = synth.make_config(int(cfg.name[3]))
    sub.sensor_xy, sub.gains = cfg.sensor_xy[keep].copy(), cfg.gains[keep].copy()
    if cfg.n_lrf > 1:
        sub.coeffs, sub.n_lrf = cfg.coeffs[keep].copy(), int(len(keep))
    sub.method, sub.dim, sub.nodes_per_axis, sub.n_iter = cfg.method, cfg.dim, cfg.nodes_per_axis, cfg.n_iter
    return sub


@pytest.mark.parametrize("idx,passive", [(2, [2, 5, 11]), (3, [0, 9, 27, 63]), (4, [7, 36])])
def test_passive_equals_the_detector_without_those_sensors(idx, passive):
    cfg, sig = _events(idx, 40 if idx != 4 else 6)
    mask = np.zeros(cfg.n_sensors, np.uint8)
    mask[passive] = 1
    keep = np.flatnonzero(mask == 0)
    cfg.passive = mask
    a = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), cfg.method, trace=True)
    sub = _subset_config(cfg, keep)
    b = oracle.reconstruct(oracle.Model.from_config(sub), sig[:, keep], oracle.grid_from_config(sub), sub.method,
                           trace=True)
    assert np.array_equal(a["xyzA"], b["xyzA"]) and np.array_equal(a["score"], b["score"])
    assert np.array_equal(a["idx"], b["idx"])


def test_options_switched_off_change_nothing():
    cfg, sig = _events(2, 64)
    base = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), cfg.method)
    cfg.passive = np.zeros(cfg.n_sensors, np.uint8)
    cfg.signal_min, cfg.dist_max = float("-inf"), float("inf")
    off = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), cfg.method)
    assert np.array_equal(base["xyzA"], off["xyzA"]) and np.array_equal(base["score"], off["score"])


@pytest.mark.parametrize("idx,thr", [(2, 12.0), (3, 2.0)])
def test_signal_threshold_matches_per_event_subset_model(idx, thr):
    """Per event, the thresholded reconstruction equals the plain one on the detector restricted to the
    sensors with S >= thr, started from the centroid of ALL sensors (R19): checked through score_at at the
    oracle's own result and at a second point, against the scipy evaluation over the subset."""
    cfg, sig = _events(idx, 12)
    cfg.signal_min = thr
    model = oracle.Model.from_config(cfg)
    res = oracle.reconstruct(model, sig, oracle.grid_from_config(cfg), cfg.method)
    n_proper = 0
    for e in range(sig.shape[0]):
        S = np.maximum(sig[e], 0.0) if cfg.method == 0 else sig[e].astype(float)
        keep = np.flatnonzero(S >= thr)
        assert len(keep) > 0
        n_proper += len(keep) < cfg.n_sensors
        sub = _subset_config(cfg, keep)
        for (x, y) in ((res["xyzA"][e, 0], res["xyzA"][e, 1]), (1.5, -2.25)):
            A_ref, s_ref = lib_score(sub, sig[e, keep], x, y)
            A, s = model.score_at(sig[e], cfg.method, x, y)
            assert A == pytest.approx(A_ref, rel=1e-9) and s == pytest.approx(s_ref, rel=1e-8, abs=1e-9)
        assert res["score"][e] == pytest.approx(lib_score(sub, sig[e, keep], *res["xyzA"][e, :2])[1], rel=1e-8)
    assert n_proper >= sig.shape[0] // 2


def test_distance_selection_is_taken_from_the_start_position():
    """One bright sensor fixes the centroid next to it; dist_max then keeps exactly the sensors within that
    distance of the centroid, and the result equals the subset detector's started from the same point."""
    cfg = synth.make_config(2)
    rng = np.random.default_rng(3)
    sig = rng.poisson(3.0, size=(8, cfg.n_sensors)).astype(np.float32)
    sig[:, 9] += 400.0                                  # sensor 9 = the array centre (0, 0)
    cfg.dist_max = 35.0
    model = oracle.Model.from_config(cfg)
    res = oracle.reconstruct(model, sig, oracle.grid_from_config(cfg), cfg.method)
    for e in range(sig.shape[0]):
        c, rc = model.centroid(sig[e], cfg.method)
        assert rc == 0
        d = np.hypot(cfg.sensor_xy[:, 0] - c[0], cfg.sensor_xy[:, 1] - c[1])
        keep = np.flatnonzero(d <= 35.0)
        assert len(keep) == 7                           # the centre and its six neighbours (pitch 30)
        sub = _subset_config(cfg, keep)
        A_ref, s_ref = lib_score(sub, sig[e, keep], *res["xyzA"][e, :2])
        assert res["score"][e] == pytest.approx(s_ref, rel=1e-8)
        assert res["xyzA"][e, 3] == pytest.approx(A_ref, rel=1e-9)


def test_passive_sensors_do_not_enter_the_centroid_and_may_hold_garbage():
    cfg, sig = _events(2, 4)
    mask = np.zeros(cfg.n_sensors, np.uint8)
    mask[[0, 18]] = 1
    cfg.passive = mask
    model = oracle.Model.from_config(cfg)
    dirty = sig.copy()
    dirty[:, 0], dirty[:, 18] = np.nan, 1e30            # a dead channel may read anything
    a = oracle.reconstruct(model, sig, oracle.grid_from_config(cfg), cfg.method)
    b = oracle.reconstruct(model, dirty, oracle.grid_from_config(cfg), cfg.method)
    assert np.array_equal(a["xyzA"], b["xyzA"]) and np.isfinite(b["xyzA"]).all()
    keep = np.flatnonzero(mask == 0)
    g = cfg.gains[keep].astype(float)
    w = np.maximum(sig[0, keep], 0.0) / g
    c, _ = model.centroid(sig[0], cfg.method)
    assert c[0] == pytest.approx((cfg.sensor_xy[keep, 0] * w).sum() / w.sum(), rel=1e-12)


def test_events_with_nothing_left_fail():
    cfg, sig = _events(2, 3)
    cfg.signal_min = 1e9
    r = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), cfg.method)
    assert np.isnan(r["xyzA"]).all() and np.isposinf(r["score"]).all()
    cfg.signal_min = float("nan")
    cfg.passive = np.ones(cfg.n_sensors, np.uint8)
    r = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), cfg.method)
    assert np.isnan(r["xyzA"]).all() and np.isposinf(r["score"]).all()


# ---------------------------------------------------------------------------
# start position = the strongest sensor (R20)
# ---------------------------------------------------------------------------
from test_oracle_pins import np_grid_argmin   # noqa: E402  (numpy/scipy evaluation of one grid iteration)


def test_strongest_sensor_start_position():
    cfg, sig = _events(2, 16)
    model = oracle.Model.from_config(cfg)
    for e in range(sig.shape[0]):
        xy, rc = model.start(sig[e], cfg.method, seed_mode=1)
        i = int(np.argmax(sig[e]))                       # numpy's argmax: first maximum
        assert rc == 0 and tuple(xy) == (float(cfg.sensor_xy[i, 0]), float(cfg.sensor_xy[i, 1]))
        assert np.array_equal(model.start(sig[e], cfg.method, seed_mode=0)[0], model.centroid(sig[e], cfg.method)[0])
    tie = np.zeros(cfg.n_sensors, np.float32)
    tie[[4, 11]] = 7.0                                   # equal maxima: the first sensor wins
    assert tuple(model.start(tie, 0, 1)[0]) == tuple(cfg.sensor_xy[4].astype(float))
    cfg.passive = np.zeros(cfg.n_sensors, np.uint8)
    cfg.passive[4] = 1                                   # a passive sensor cannot be the start
    assert tuple(oracle.Model.from_config(cfg).start(tie, 0, 1)[0]) == tuple(cfg.sensor_xy[11].astype(float))
    assert model.start(np.zeros(cfg.n_sensors, np.float32), 0, 1)[1] == 1        # sum S = 0: unusable
    bad = sig[0].copy()
    bad[3] = np.nan
    assert model.start(bad, 0, 1)[1] == 1


@pytest.mark.parametrize("idx", [1, 3])
def test_first_iteration_from_the_strongest_sensor_equals_numpy_argmin(idx):
    cfg, sig = _events(idx, 6)
    cfg.seed_mode, cfg.n_iter = 1, 1
    res = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), cfg.method, trace=True)
    for e in range(sig.shape[0]):
        S = np.maximum(sig[e], 0.0) if cfg.method == 0 else sig[e]
        i = int(np.argmax(S))
        centre = (float(cfg.sensor_xy[i, 0]), float(cfg.sensor_xy[i, 1]), 0.0)
        k, sc = np_grid_argmin(cfg, sig[e], centre, cfg.step0_xy, cfg.step0_z)
        assert res["idx"][e, 0] == k
        assert res["best"][e, 0] == pytest.approx(sc[k], rel=1e-9)


def test_distance_selection_follows_the_chosen_start():
    """With seed_mode = 1 the 'initial search position' of PAPER.md:318 is the strongest sensor's axis."""
    cfg, sig = _events(2, 10)
    cfg.seed_mode, cfg.dist_max = 1, 31.0
    model = oracle.Model.from_config(cfg)
    res = oracle.reconstruct(model, sig, oracle.grid_from_config(cfg), cfg.method)
    for e in range(sig.shape[0]):
        i = int(np.argmax(sig[e]))
        d = np.hypot(cfg.sensor_xy[:, 0] - cfg.sensor_xy[i, 0], cfg.sensor_xy[:, 1] - cfg.sensor_xy[i, 1])
        keep = np.flatnonzero(d <= 31.0)
        sub = _subset_config(cfg, keep)
        A_ref, s_ref = lib_score(sub, sig[e, keep], *res["xyzA"][e, :2])
        assert res["score"][e] == pytest.approx(s_ref, rel=1e-8) and res["xyzA"][e, 3] == pytest.approx(A_ref, rel=1e-9)


# ---------------------------------------------------------------------------
# least squares with the paper's sum-ratio energy (method 2; R27)
# ---------------------------------------------------------------------------
def test_sum_ratio_least_squares_matches_its_definition():
    from test_oracle_pins import lib_lrf
    for idx in (2, 3):
        cfg, sig = _events(idx, 8)
        model = oracle.Model.from_config(cfg)
        rng = np.random.default_rng(idx)
        for e in range(sig.shape[0]):
            x, y = rng.uniform(-20, 20, 2)
            L = lib_lrf(cfg, x, y)                                  # scipy evaluation of every sensor's LRF
            S = sig[e].astype(float)
            A_ref = S.sum() / L.sum()
            chi2_ref = ((S - A_ref * L) ** 2 / np.maximum(S, 1.0)).sum()
            A, sc = model.score_at(sig[e], 2, x, y)
            assert A == pytest.approx(A_ref, rel=1e-10) and sc == pytest.approx(chi2_ref, rel=1e-9)
            # the weighted minimiser of method 1 can only do better on the same chi-square
            assert model.score_at(sig[e], 1, x, y)[1] <= sc * (1 + 1e-12)


def test_sum_ratio_first_iteration_equals_numpy_argmin():
    from test_oracle_pins import lib_lrf
    cfg, sig = _events(3, 4)
    cfg.method, cfg.n_iter = 2, 1
    res = oracle.reconstruct(oracle.Model.from_config(cfg), sig, oracle.grid_from_config(cfg), 2, trace=True)
    G, half = cfg.nodes_per_axis, 0.5 * (cfg.nodes_per_axis - 1)
    model = oracle.Model.from_config(cfg)
    for e in range(sig.shape[0]):
        c, _ = model.centroid(sig[e], 2)
        S = sig[e].astype(float)
        sc = np.empty(G * G)
        for iy in range(G):
            for ix in range(G):
                L = lib_lrf(cfg, c[0] + (ix - half) * cfg.step0_xy, c[1] + (iy - half) * cfg.step0_xy)
                A = S.sum() / L.sum()
                sc[iy * G + ix] = ((S - A * L) ** 2 / np.maximum(S, 1.0)).sum()
        assert res["idx"][e, 0] == int(np.argmin(sc)) and res["best"][e, 0] == pytest.approx(sc.min(), rel=1e-9)
