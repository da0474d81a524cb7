"""GPU-vs-oracle parity through the C ABI (include/ants_recon.h), -m gpu.

Rules (BASELINE.json north_star; tests/parity_rules.py): score at the returned
node within 1e-5 relative of the oracle's score there, position within one
final grid step for >= 99.9 % of events, identical winning node wherever the
oracle's best-to-second gap exceeds 1e-4 relative, energy to 1e-5.

Sizes: subsets the oracle finishes in seconds (several CTA tiles plus a ragged
tail), and the full BASELINE.json sizes in the launch configuration bench.py
times, checked on sampled events (events are independent, so the oracle can
reconstruct any sample one by one).
"""
import math
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import oracle                                      # noqa: E402
from paper_1602_07247_b200 import recon, synth                 # noqa: E402
import parity_rules                                            # noqa: E402

FULL = os.environ.get("ANTS_TEST_FULL", "1") != "0"


def _run(cfg, sig_dev, trace=True):
    r = recon.Reconstructor(cfg)
    try:
        out = r(sig_dev, trace=trace)
        torch.cuda.synchronize()
        return [None if t is None else t.cpu().numpy() for t in out]
    finally:
        r.close()


# subset sizes: ~3e8 (node, sensor) pairs each for the oracle; none a multiple of the CTA tile
SUBSETS = {1: 10_000, 2: 20_011, 3: 4_003, 4: 2_501, 5: 2_503}


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_parity_subset(idx):
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, SUBSETS[idx], device="cuda")
    sig = ev["signals"]
    xyzA, score, path = _run(cfg, sig)
    res = parity_rules.compare(cfg, sig.cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, cfg.name)
    # sanity: the reconstruction is near the truth (not parity, catches a broken generator)
    err = np.hypot(xyzA[:, 0] - ev["true_xyz"][:, 0].cpu().numpy(), xyzA[:, 1] - ev["true_xyz"][:, 1].cpu().numpy())
    assert np.nanmedian(err) < 6.0


@pytest.mark.parametrize("idx", [2, 3, 4, 5])
def test_parity_full_size_sampled(idx):
    """BASELINE.json's full event count in one launch (bench.py's configuration);
    2000 sampled events are reconstructed one by one by the oracle."""
    if not FULL:
        pytest.skip("ANTS_TEST_FULL=0")
    cfg = synth.make_config(idx)
    E = cfg.n_events // cfg.n_batches
    ev = synth.generate_events(cfg, E, device="cuda")
    sig = ev["signals"]
    r = recon.Reconstructor(cfg)
    try:
        xyzA, score = r(sig)
        torch.cuda.synchronize()
    finally:
        r.close()
    rng = np.random.default_rng(7)
    n_s = 2000 if idx in (2, 3) else 1000
    pick = np.sort(rng.choice(E, n_s, replace=False))
    pick[0], pick[-1] = 0, E - 1
    pt = torch.from_numpy(pick).cuda()
    res = parity_rules.compare(cfg, sig[pt].cpu().numpy(), xyzA[pt].cpu().numpy(), score[pt].cpu().numpy(), None)
    parity_rules.assert_parity(res, cfg.name + " full")
    # properties that hold at any size: every event produced a finite result inside the search reach
    assert bool(torch.isfinite(xyzA).all()) and bool(torch.isfinite(score).all())
    assert float(score.min()) >= -1e-3
    reach = cfg.step0_xy * (cfg.nodes_per_axis - 1) / 2 * 2.0 + 1.0
    lim = float(np.abs(cfg.sensor_xy).max()) + reach
    assert float(xyzA[:, :2].abs().max()) <= lim


def test_parity_cfg5_batch_sampled():
    """One of config 5's eight 2M-event batches, through the streamed host-buffer entry point
    (ants_reconstruct_host, pinned memory), sampled against the oracle."""
    if not FULL:
        pytest.skip("ANTS_TEST_FULL=0")
    cfg = synth.make_config(5)
    E = 400_000
    ev = synth.generate_events(cfg, E, device="cuda", batch=3)
    sig_h = ev["signals"].cpu().pin_memory()
    xyzA = torch.empty((E, 4), dtype=torch.float32).pin_memory()
    score = torch.empty((E,), dtype=torch.float32).pin_memory()
    r = recon.Reconstructor(cfg)
    try:
        recon.ants_reconstruct_host(r.handle, sig_h, r.grid, r.method, xyzA, score, chunk_events=100_003)
        d_xyzA, d_score = r(ev["signals"])
        torch.cuda.synchronize()
    finally:
        r.close()
    # host path == device path, bit for bit (same kernel, chunking must not matter)
    assert torch.equal(xyzA, d_xyzA.cpu()) and torch.equal(score, d_score.cpu())
    pick = np.sort(np.random.default_rng(11).choice(E, 1000, replace=False))
    res = parity_rules.compare(cfg, sig_h.numpy()[pick], xyzA.numpy()[pick], score.numpy()[pick], None)
    parity_rules.assert_parity(res, "cfg5 host-streamed")


@pytest.mark.parametrize("idx,E,chunk", [(2, 150_001, 40_003), (3, 60_001, 25_001)])
def test_host_streamed_path_equals_device_path_on_round_kernels(idx, E, chunk):
    """The kernels that take their events in CTA-wide rounds, through ants_reconstruct_host with chunks that are no
    multiple of a CTA's warps (every chunk ends on a short round, three launches in flight on three streams): bit for
    bit the device path's result."""
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, E, device="cuda", batch=2)
    sig_h = ev["signals"].cpu().pin_memory()
    xyzA = torch.empty((E, 4), dtype=torch.float32).pin_memory()
    score = torch.empty((E,), dtype=torch.float32).pin_memory()
    r = recon.Reconstructor(cfg)
    try:
        assert r.plan()["kernel"].endswith(",true,true>")
        recon.ants_reconstruct_host(r.handle, sig_h, r.grid, r.method, xyzA, score, chunk_events=chunk)
        d_xyzA, d_score = r(ev["signals"])
        torch.cuda.synchronize()
    finally:
        r.close()
    assert torch.equal(xyzA, d_xyzA.cpu()) and torch.equal(score, d_score.cpu())
    assert torch.isfinite(score).all()


# ---------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------
def test_empty_and_tiny_batches():
    cfg = synth.make_config(1)
    r = recon.Reconstructor(cfg)
    try:
        xyzA, score = r(torch.empty((0, cfg.n_sensors), device="cuda"))
        assert xyzA.shape == (0, 4) and score.shape == (0,)
        ev = synth.generate_events(cfg, 37, device="cuda")
        full = r(ev["signals"])
        for n in (1, 2, 9, 33):
            part = r(ev["signals"][:n].contiguous())
            torch.cuda.synchronize()
            assert torch.equal(part[0], full[0][:n]) and torch.equal(part[1], full[1][:n])
    finally:
        r.close()


def test_failed_events_and_negative_signals():
    cfg = synth.make_config(2)
    ev = synth.generate_events(cfg, 64, device="cuda")
    sig = ev["signals"].clone()
    sig[3] = 0.0                         # sum S = 0 -> failed event
    sig[5, 2] = float("nan")             # non-finite -> failed event
    sig[7, 1] = float("inf")
    sig[9] = -sig[9]                     # all negative: Poisson clips to 0 -> failed
    sig[11, 0] = -3.0                    # one negative: clipped, event fine (R18)
    sig[13, 4] = float("-inf")           # -inf is non-finite: fails BEFORE the clipping
    xyzA, score, path = _run(cfg, sig)
    for e in (3, 5, 7, 9, 13):
        assert np.isnan(xyzA[e]).all() and np.isposinf(score[e])
        assert ((path[e].astype(np.int64) & 0xFFFF) == 0xFFFF).all()
    res = parity_rules.compare(cfg, sig.cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, "failed events")
    assert np.isfinite(xyzA[11]).all()


@pytest.mark.parametrize("G,method", [(2, 0), (4, 1), (16, 0), (5, 1)])
def test_grid_sizes_2d(G, method):
    """Even and odd G, the smallest grid and the compiled maximum (16 x 16 = 256 nodes)."""
    cfg = synth.make_config(2 if method == 0 else 3)
    cfg.nodes_per_axis, cfg.method = G, method
    cfg.step0_xy = 40.0 / G if method == 0 else 8.0 / G
    cfg.n_iter = 9
    ev = synth.generate_events(cfg, 1501, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"G={G} method={method}")


def test_chi_square_on_shared_profile_and_poisson_on_individual():
    """Method x LRF-sharing combinations the five configs do not use."""
    for idx, method in ((2, 1), (3, 0)):
        cfg = synth.make_config(idx)
        cfg.method = method
        ev = synth.generate_events(cfg, 3001, device="cuda")
        xyzA, score, path = _run(cfg, ev["signals"])
        res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
        parity_rules.assert_parity(res, f"cfg{idx} method={method}")


def _negative_tail(idx=2):
    cfg = synth.make_config(idx)
    c = cfg.coeffs.copy()
    c[0, 0, -4:] = -0.002                # negative tail beyond ~75 mm
    cfg.coeffs = c
    return cfg


@pytest.mark.parametrize("method", [0, 1, 2])
def test_non_positive_spline_uses_validity_rules(method):
    """An LRF that goes negative far out: the library must apply the per-pair validity rule (a node with
    L_i <= 0 where S_i > 0 is invalid).  Such a model runs the general kernel (FP32 scores on the coarse grids,
    FP64 on the fine ones) and meets the full north_star rule set."""
    cfg = _negative_tail()
    cfg.method = method
    ev = synth.generate_events(synth.make_config(2), 4001, device="cuda")
    r = recon.Reconstructor(cfg)
    assert "recon_gen_kernel" in r.plan()["kernel"]
    r.close()
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"negative tail, method {method}")


def test_non_positive_spline_with_sensor_selection_and_strongest_start():
    """Sensor selection and the strongest-sensor start are available on the general kernel too."""
    cfg = _negative_tail()
    cfg.passive = np.zeros(cfg.n_sensors, np.uint8)
    cfg.passive[[3, 11]] = 1
    cfg.signal_min, cfg.dist_max, cfg.seed_mode = 4.0, 70.0, 1
    ev = synth.generate_events(synth.make_config(2), 3001, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, "negative tail with selection")


@pytest.mark.parametrize("idx,n,kw", [
    (6, 6_007, {}), (6, 3_001, dict(method=0)), (6, 2_003, dict(method=2, nodes_per_axis=8)),
    (7, 1_201, {}), (7, 801, dict(method=1, nodes_per_axis=5)), (7, 1_501, dict(dim=2, nodes_per_axis=9, z_seed=7.5)),
    (8, 6_007, {}), (8, 3_001, dict(method=1, seed_mode=1)),
])
def test_parity_xy_composite_sliced_lrfs(idx, n, kw):
    """XY LRFs shared by symmetry groups (config 6), Sliced LRFs searched in 3-D and at a fixed z (config 7) and
    Composite LRFs (config 8): PAPER.md:388-396, 406; the general kernel under the full rule set."""
    cfg = synth.make_config(idx)
    for k, v in kw.items():
        setattr(cfg, k, v)
    ev = synth.generate_events(synth.make_config(idx), n, device="cuda")
    r = recon.Reconstructor(cfg)
    assert "recon_gen_kernel" in r.plan()["kernel"]
    r.close()
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"cfg{idx} {kw}")


def test_xy_lrf_individual_tables_and_selection():
    """XY LRFs with one table per sensor (no grouping, no frames) and sensor selection."""
    base = synth.make_config(6)
    cfg = synth.make_config(6)
    cfg.n_lrf = cfg.n_sensors
    cfg.coeffs_xy = np.ascontiguousarray(base.coeffs_xy[base.group])
    cfg.group, cfg.xform = None, None
    cfg.coeffs = np.zeros((cfg.n_sensors, 1, 0), np.float32)
    cfg.signal_min, cfg.dist_max = 3.0, 25.0
    ev = synth.generate_events(cfg, 2001, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    parity_rules.assert_parity(parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path), "XY individual")


def test_symmetry_groups_in_the_library_agree_with_the_oracle():
    from oracle import fit as ofit
    for xy, n_fold, reflect in ((synth.square_array(8, 6.0), 4, True), (synth.square_array(8, 6.0), 4, False),
                                (synth.hex_array(3, 30.0), 6, True), (synth.hex_array(3, 30.0), 6, False)):
        g, x, n = recon.ants_group_by_symmetry(xy, n_fold, reflect)
        g0, x0, n0 = ofit.group_by_symmetry(xy, n_fold, reflect)
        assert n == n0 and np.array_equal(g, g0) and np.abs(x - x0).max() <= 1e-6


@pytest.mark.parametrize("lrf_dim,G,method", [(1, 2, 0), (1, 4, 0), (1, 6, 1), (1, 4, 2), (1, 8, 0), (2, 4, 0), (2, 6, 1)])
def test_tie_break_lowest_linear_index_gpu(lrf_dim, G, method):
    """R9 on an EXACT tie: sensors on the line y = 0 make nodes mirrored in y bit-identical (same operands in
    the same order, in FP32 as in FP64), so the first iteration always has a tied pair; the lower linear
    index must win on both sides -> identical node index, bit for bit (tests/test_oracle_pins.py pins the
    oracle's side of this)."""
    cfg = synth.make_config(4 if lrf_dim == 2 else 2)
    cfg.sensor_xy = np.array([[-31.0, 0.0], [-9.5, 0.0], [4.25, 0.0], [22.0, 0.0], [40.5, 0.0]], np.float32)
    cfg.gains = np.array([1.0, 0.9, 1.1, 1.05, 0.95], np.float32)
    cfg.nodes_per_axis, cfg.method, cfg.n_iter = G, method, 1
    cfg.step0_xy, cfg.step0_z = 3.0, 2.0
    rng = np.random.default_rng(G * 10 + method)
    sig = torch.from_numpy(rng.poisson(40.0, (257, 5)).astype(np.float32)).cuda()
    xyzA, score, path = _run(cfg, sig)
    model = oracle.Model.from_config(cfg)
    ref = oracle.reconstruct(model, sig.cpu().numpy(), oracle.grid_from_config(cfg), method, trace=True)
    ok = np.isfinite(ref["xyzA"][:, 0])
    assert ok.sum() > 250
    assert np.all(ref["best"][ok, 0] == ref["second"][ok, 0])            # every event has an exact tie
    gp = path.astype(np.int64)[:, 0] & 0xFFFF
    assert np.array_equal(gp[ok], ref["idx"][ok, 0])                      # and both sides take the lower index
    iy = (gp[ok] // G) % G
    assert np.all(iy < G - 1 - iy)
    assert np.array_equal(xyzA[ok, 1].astype(np.float64), ref["xyzA"][ok, 1])


def test_noise_free_recovery_gpu():
    """Noise-free signals: the GPU result is within one final step of the truth and the deviance ~ 0."""
    for idx in (1, 2, 5):
        cfg = synth.make_config(idx)
        ev = synth.generate_events(cfg, 512, device="cuda", noise_free=True)
        xyzA, score, path = _run(cfg, ev["signals"])
        res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path, score_floor=1e-6)
        assert res["fail_mismatch"] == 0 and res["score_viol"] == 0 and res["pos_frac_within"] >= 0.999, res


def test_mirror_symmetry_gpu():
    """Negating every sensor x negates the reconstructed x and leaves y, A, score bit-identical."""
    cfg = synth.make_config(2)
    ev = synth.generate_events(cfg, 4096, device="cuda")
    a = _run(cfg, ev["signals"], trace=False)
    cfg_m = synth.make_config(2)
    cfg_m.sensor_xy = cfg.sensor_xy * np.array([-1.0, 1.0], np.float32)
    b = _run(cfg_m, ev["signals"], trace=False)
    same = (a[0][:, 0] == -b[0][:, 0]) & (a[0][:, 1] == b[0][:, 1])
    assert same.mean() > 0.995                      # exact ties may break differently
    assert np.array_equal(a[1][same], b[1][same])


def test_status_codes():
    cfg = synth.make_config(1)
    r = recon.Reconstructor(cfg)
    try:
        sig = torch.ones((4, cfg.n_sensors), device="cuda")
        xyzA = torch.empty((4, 4), device="cuda")
        score = torch.empty((4,), device="cuda")

        def status(**kw):
            g = recon.GridParams(cfg.dim, cfg.nodes_per_axis, cfg.step0_xy, cfg.step0_z, cfg.factor,
                                 cfg.n_iter, 0, cfg.z_seed)
            for k, v in kw.items():
                setattr(g, k, v)
            try:
                recon.ants_reconstruct(r.handle, sig, g, kw.get("_method", 0), xyzA, score)
            except recon.AntsError as e:
                return e.status
            return 0

        assert status() == 0
        assert status(nodes_per_axis=1) == -1
        assert status(factor=1.0) == -1
        assert status(n_iter=0) == -1
        assert status(step0_xy=0.0) == -1
        assert status(dim=3) == -1                      # 3-D search over an axial LRF
        assert status(nodes_per_axis=17) == -2          # 289 nodes > compiled limit
        assert status(seed_mode=1) == 0                 # strongest-sensor start (R20)
        assert status(seed_mode=2) == -1
    finally:
        r.close()
    with pytest.raises(recon.AntsError):
        recon.ants_lrf_create(cfg.sensor_xy, cfg.gains, np.array([5.0, 1.0], np.float32), cfg.coeffs,
                              recon.LrfDims(cfg.n_sensors, 1, 1, 16, 0))


# ---------------------------------------------------------------------------
# kernel variants of the packed kernels: node reuse, CTA-wide event rounds, cross-column top level
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("idx,G,method,n,kernel", [
    (2, 9, 0, 3001, "ants::recon2d_pk_kernel<3,0,true,true>"),      # Poisson, small array: reuse + rounds
    (5, 9, 0, 1203, "ants::recon2d_pk_kernel<3,0,true>"),           # Poisson, 127 sensors: reuse, no rounds
    (2, 11, 0, 2003, "ants::recon2d_pk_kernel<4,0,true,true>"),     # four nodes per lane (L2 prefetch)
    (5, 11, 0, 803, "ants::recon2d_pk_kernel<4,0,true>"),
    (3, 11, 1, 2005, "ants::recon2d_pk_kernel<4,1,true,true>"),     # chi-square: always with the rounds
    (3, 9, 2, 2001, "ants::recon2d_pk_kernel<3,2,true,true>"),
    (5, 9, 1, 1001, "ants::recon2d_pk_kernel<3,1,true,true>"),
    (2, 8, 0, 2001, "ants::recon2d_pk_kernel<2,0,false>"),          # even G: no node coincides
    (4, 7, 0, 1001, "ants::recon3d_pk_kernel<2,4,0,true>"),         # odd 3-D grid, two columns per lane: cross unit
    (4, 8, 0, 601, "ants::recon3d_pk_kernel<2,4,0>"),
    (4, 7, 1, 801, "ants::recon3d_pk_kernel<2,4,1,true>"),
])
def test_packed_kernel_variants_are_picked_and_in_parity(idx, G, method, n, kernel):
    """The plan's choice among the instantiations (csrc/ants_recon.cu make_plan / make_plan3d; profiles/r02_lockstep.md)
    and parity of each under the full rule set.  The event counts are no multiple of a CTA's warps, so the kernels
    with CTA-wide rounds end on a short round."""
    cfg = synth.make_config(idx)
    cfg.nodes_per_axis, cfg.method = G, method
    ev = synth.generate_events(cfg, n, device="cuda")
    r = recon.Reconstructor(cfg)
    try:
        assert r.plan()["kernel"] == kernel
    finally:
        r.close()
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"{cfg.name} G={G} method={method} {kernel}")


# ---------------------------------------------------------------------------
# axial+z LRF variants beyond config 4
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("G,method", [(7, 1), (4, 0), (8, 0), (3, 1), (5, 0)])
def test_axial_z_grid_sizes_and_methods(G, method):
    cfg = synth.make_config(4)
    cfg.nodes_per_axis, cfg.method = G, method
    cfg.step0_xy, cfg.step0_z = 48.0 / (G - 1), 18.0 / (G - 1)
    ev = synth.generate_events(cfg, 2401, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"axial+z G={G} method={method}")


@pytest.mark.parametrize("G,z_seed", [(9, 7.5), (12, float("nan")), (6, 0.0), (16, 20.0)])
def test_axial_z_lrf_with_2d_search_at_fixed_z(G, z_seed):
    """dim = 2 over an (r, z) LRF: the search runs in (x, y) at z = z_seed (NaN = mid-range)."""
    cfg = synth.make_config(4)
    cfg.dim, cfg.nodes_per_axis, cfg.z_seed = 2, G, z_seed
    cfg.step0_xy = 48.0 / (G - 1)
    z = 10.0 if z_seed != z_seed else z_seed
    cfg.z_range = (z, z)
    ev = synth.generate_events(cfg, 1203, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    assert np.all(xyzA[:, 2] == np.float32(z))
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"axial+z fixed z G={G}")


def test_axial_z_seed_outside_range_gives_invalid_nodes():
    """z_seed outside [z_lo, z_hi] with a 2-D search: every node is invalid (R6), the centre stays at
    the centroid, A = NaN and score = +inf, exactly as the oracle."""
    cfg = synth.make_config(4)
    cfg.dim, cfg.z_seed = 2, 25.0
    ev = synth.generate_events(cfg, 64, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    assert np.isposinf(score).all() and np.isnan(xyzA[:, 3]).all() and np.isfinite(xyzA[:, :3]).all()
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    assert res["fail_mismatch"] == 0 and res["idx_diverged"] == 0 and res["pos_frac_within"] == 1.0, res
    assert np.all(res["ref"]["idx"] == -1)                       # no node is ever valid, on either side
    assert ((path.astype(np.int64) & 0xFFFF) == 0xFFFF).all()
    model = oracle.Model.from_config(cfg)
    ref = oracle.reconstruct(model, ev["signals"].cpu().numpy(), oracle.grid_from_config(cfg), cfg.method)
    assert np.allclose(ref["xyzA"][:, :2], xyzA[:, :2], atol=1e-4) and np.isposinf(ref["score"]).all()


# ---------------------------------------------------------------------------
# sensor selection (R19; PAPER.md:358 passive sensors, PAPER.md:318 threshold / distance)
# ---------------------------------------------------------------------------
def _with_selection(idx, passive=None, signal_min=float("nan"), dist_max=float("nan")):
    cfg = synth.make_config(idx)
    if passive is not None:
        m = np.zeros(cfg.n_sensors, np.uint8)
        m[list(passive)] = 1
        cfg.passive = m
    cfg.signal_min, cfg.dist_max = signal_min, dist_max
    return cfg


@pytest.mark.parametrize("idx,kw", [
    (2, dict(passive=[2, 5, 11])),
    (2, dict(signal_min=8.0)),
    (2, dict(dist_max=47.0)),
    (5, dict(passive=[0, 63, 126], signal_min=3.0, dist_max=110.0)),
    (3, dict(passive=[9, 27], signal_min=2.0)),
    (3, dict(dist_max=20.5)),
    (1, dict(passive=[3])),
    (4, dict(passive=[7, 36], signal_min=1.0)),
    (4, dict(dist_max=95.0)),
])
def test_parity_with_sensor_selection(idx, kw):
    cfg = _with_selection(idx, **kw)
    n = {1: 4001, 2: 6001, 3: 1501, 4: 2501, 5: 801}[idx]
    ev = synth.generate_events(synth.make_config(idx), n, device="cuda")
    sig = ev["signals"].clone()
    if cfg.passive is not None:                      # a dead channel may read anything
        bad = torch.from_numpy(np.flatnonzero(cfg.passive)).cuda()
        sig[::3, bad[0]] = float("nan")
        sig[1::3, bad[-1]] = 1e30
    xyzA, score, path = _run(cfg, sig)
    res = parity_rules.compare(cfg, sig.cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"cfg{idx} {kw}")
    assert np.isfinite(xyzA).all(axis=1).mean() > 0.99


def test_selection_that_leaves_nothing_fails_the_event():
    cfg = _with_selection(2, signal_min=1e9)
    ev = synth.generate_events(synth.make_config(2), 33, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    assert np.isnan(xyzA).all() and np.isposinf(score).all()
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    assert res["fail_mismatch"] == 0


def test_selection_can_be_switched_off_again():
    cfg = synth.make_config(2)
    ev = synth.generate_events(cfg, 2048, device="cuda")
    r = recon.Reconstructor(cfg)
    try:
        base = [t.clone() for t in r(ev["signals"])]
        recon.ants_lrf_set_selection(r.handle, np.arange(cfg.n_sensors) % 5 == 0, 4.0, 50.0)
        sel = [t.clone() for t in r(ev["signals"])]
        recon.ants_lrf_set_selection(r.handle, None)
        again = r(ev["signals"])
        torch.cuda.synchronize()
        assert torch.equal(base[0], again[0]) and torch.equal(base[1], again[1])
        assert not torch.equal(base[0], sel[0])
    finally:
        r.close()


@pytest.mark.parametrize("idx,kw", [(2, {}), (3, {}), (4, {}), (5, dict(dist_max=60.0)), (2, dict(passive=[9], signal_min=5.0))])
def test_parity_with_strongest_sensor_start(idx, kw):
    """seed_mode = 1 (R20): the grid starts on the axis of the strongest sensor."""
    cfg = _with_selection(idx, **kw)
    cfg.seed_mode = 1
    n = {2: 6001, 3: 1501, 4: 2501, 5: 801}[idx]
    ev = synth.generate_events(synth.make_config(idx), n, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"cfg{idx} strongest-sensor start {kw}")
    # the two start options agree on most events (both reach the same minimum) but not bit for bit
    cfg0 = _with_selection(idx, **kw)
    a = _run(cfg0, ev["signals"], trace=False)[0]
    close = np.hypot(a[:, 0] - xyzA[:, 0], a[:, 1] - xyzA[:, 1]) < 1.0
    assert close.mean() > 0.8


def test_large_array_more_than_128_sensors():
    """217 PMTs (hex, 8 rings): more sensors than the 4-per-lane register prefetch holds and seven rounds of
    32 in the per-iteration list building; odd count (pad pair)."""
    cfg = synth.make_config(5)
    cfg.sensor_xy = synth.hex_array(8, 20.0)
    cfg.gains = np.random.default_rng(2).uniform(0.8, 1.2, len(cfg.sensor_xy)).astype(np.float32)
    cfg.extent, cfg.n_iter = 120.0, 10
    assert cfg.n_sensors == 217
    ev = synth.generate_events(cfg, 1203, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, "217 sensors")
    cfg.method = 1
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, "217 sensors chi-square")


def _random_config(seed):
    """A seeded irregular detector: random sensor positions and gains, random bell width, grid, iteration
    count, contraction factor, method and LRF sharing (nothing regular for the kernels to lean on)."""
    rng = np.random.default_rng(1000 + seed)
    cfg = synth.make_config(2)
    N = int(rng.integers(3, 70))
    cfg.sensor_xy = rng.uniform(-50.0, 50.0, (N, 2)).astype(np.float32)
    cfg.gains = rng.uniform(0.6, 1.5, N).astype(np.float32)
    width = float(rng.uniform(12.0, 30.0))
    n_int = int(rng.integers(6, 25))
    r_hi = float(rng.uniform(80.0, 160.0))
    base = synth.fit_axial(lambda r: (1.0 + (r / width) ** 2) ** -1.5, 0.0, r_hi, n_int).astype(np.float64)
    cfg.knots = np.array([0.0, r_hi], np.float32)
    cfg.n_int_r = n_int
    if rng.random() < 0.5:
        cfg.n_lrf, cfg.coeffs = 1, base.astype(np.float32)[None, None, :]
    else:
        fac = rng.normal(1.0, 0.05, N)
        cfg.n_lrf, cfg.coeffs = N, (base[None, :] * fac[:, None]).astype(np.float32)[:, None, :]
        cfg.gains = np.ones(N, np.float32)
    cfg.nodes_per_axis = int(rng.integers(3, 14))
    cfg.n_iter = int(rng.integers(4, 11))
    cfg.factor = float(rng.choice([0.5, 0.5, 0.6, 0.4]))
    cfg.step0_xy = float(rng.uniform(20.0, 40.0)) / (cfg.nodes_per_axis - 1) * 2.0
    cfg.method = int(rng.integers(0, 3))                       # Poisson ML, chi-square, sum-ratio chi-square
    cfg.extent = 40.0
    cfg.nph = ("uniform", 2000.0, 8000.0)
    cfg.noise_sigma = float(rng.choice([0.0, 1.0]))
    cfg.seed_mode = int(rng.integers(0, 2))
    if seed >= 12:                           # the second dozen also exercises the sensor selection (R19)
        if rng.random() < 0.6:
            cfg.passive = (rng.random(N) < 0.15).astype(np.uint8)
            cfg.passive[int(rng.integers(0, N))] = 0
        if rng.random() < 0.6:
            cfg.signal_min = float(rng.uniform(0.5, 4.0))
        if rng.random() < 0.6:
            cfg.dist_max = float(rng.uniform(45.0, 110.0))
    return cfg


@pytest.mark.parametrize("seed", range(24))
def test_parity_on_random_irregular_detectors(seed):
    cfg = _random_config(seed)
    ev = synth.generate_events(cfg, 3001, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    what = (f"seed {seed}: N={cfg.n_sensors} n_lrf={cfg.n_lrf} G={cfg.nodes_per_axis} K={cfg.n_iter} f={cfg.factor} "
            f"method={cfg.method} start={cfg.seed_mode}")
    parity_rules.assert_parity(res, what)


@pytest.mark.parametrize("seed", range(8))
def test_parity_on_random_axial_z_detectors(seed):
    """Config 4's (r, z) response on random sensor layouts, random grids (3..8 per axis, or a 2-D search
    at a random fixed z), iterations, contraction factor, method and start option."""
    rng = np.random.default_rng(2000 + seed)
    cfg = synth.make_config(4)
    N = int(rng.integers(5, 60))
    cfg.sensor_xy = rng.uniform(-80.0, 80.0, (N, 2)).astype(np.float32)
    cfg.gains = rng.uniform(0.7, 1.4, N).astype(np.float32)
    cfg.method = int(rng.integers(0, 2))
    cfg.n_iter = int(rng.integers(5, 11))
    cfg.factor = float(rng.choice([0.5, 0.5, 0.6]))
    cfg.seed_mode = int(rng.integers(0, 2))
    cfg.extent = 60.0
    if rng.random() < 0.7:
        cfg.nodes_per_axis = int(rng.integers(3, 9))
        cfg.step0_xy = 48.0 / (cfg.nodes_per_axis - 1)
        cfg.step0_z = 18.0 / (cfg.nodes_per_axis - 1)
    else:
        cfg.dim, cfg.nodes_per_axis = 2, int(rng.integers(3, 14))
        cfg.step0_xy = 48.0 / (cfg.nodes_per_axis - 1)
        z = float(rng.uniform(1.0, 19.0))
        cfg.z_seed, cfg.z_range = z, (z, z)
    ev = synth.generate_events(cfg, 2401, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"seed {seed}: N={N} dim={cfg.dim} G={cfg.nodes_per_axis} K={cfg.n_iter} "
                                    f"f={cfg.factor} method={cfg.method} start={cfg.seed_mode}")


# ---------------------------------------------------------------------------
# least squares with the paper's sum-ratio energy (method 2; R27)
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("idx,n", [(3, 4_003), (2, 10_007), (5, 1_501), (1, 5_001)])
def test_parity_sum_ratio_least_squares(idx, n):
    cfg = synth.make_config(idx)
    cfg.method = 2
    ev = synth.generate_events(cfg, n, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path)
    parity_rules.assert_parity(res, f"cfg{idx} sum-ratio least squares")


def test_sum_ratio_least_squares_variants():
    """Method 2 with sensor selection, the strongest-sensor start, a non-positive LRF (general kernel) and the
    refusal for axial+z LRFs."""
    cfg = _with_selection(3, passive=[5, 40], signal_min=2.0)
    cfg.method, cfg.seed_mode = 2, 1
    ev = synth.generate_events(synth.make_config(3), 3001, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    parity_rules.assert_parity(parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path), "selection")
    cfg = synth.make_config(2)
    c = cfg.coeffs.copy()
    c[0, 0, -4:] = -0.002
    cfg.coeffs, cfg.method = c, 2
    ev = synth.generate_events(synth.make_config(2), 2001, device="cuda")
    xyzA, score, path = _run(cfg, ev["signals"])
    parity_rules.assert_parity(parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA, score, path), "negative tail")
    cfg = synth.make_config(4)
    cfg.method = 2
    with pytest.raises(recon.AntsError) as ei:
        _run(cfg, torch.ones((4, cfg.n_sensors), device="cuda"))
    assert ei.value.status == -2
