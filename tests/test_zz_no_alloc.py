"""GPU test of ants_lrf_fit_gains_static, the entry point that allocates nothing (include/ants_recon.h): its output
against the existing path (ants_lrf_fit_gains) and the oracle, on calls in a row that share the library's fixed
scratch array.  Collected last on purpose (the file name): the suite runs with `pytest -x`, and a failure here must
not hide another test.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import fit as ofit                                 # noqa: E402
from paper_1602_07247_b200 import recon, synth                 # noqa: E402

if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)


def _batch(idx, n, batch):
    """Flood events of config idx at their true positions (A = the known light output), sub-stream `batch`."""
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, n, device="cuda", batch=batch)
    xyzA = torch.cat([ev["true_xyz"], 0.1 * ev["n_ph"][:, None]], 1).float().contiguous()
    return cfg, ev["signals"].contiguous(), xyzA


def _check(cfg, sig, xyzA):
    """Same tolerance as tests/test_gpu_fit.py::test_gain_evaluation_parity_and_recovery: FP64 sums on all sides,
    float32 output: 1e-6 relative; pair counts bit-exact."""
    g, used = recon.ants_lrf_fit_gains_static(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], sig, xyzA)
    g_ref, used_ref = recon.ants_lrf_fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], sig, xyzA)
    assert np.array_equal(used, used_ref)
    assert np.abs(g - g_ref).max() <= 1e-6 * np.abs(g_ref).max()
    g0, used0 = ofit.fit_gains(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], cfg.n_int_r, sig.cpu().numpy(), xyzA.cpu().numpy())
    assert np.array_equal(used, used0)
    assert np.abs(g - g0).max() <= 1e-6 * np.abs(g0).max()
    return g


def test_static_scratch_gain_evaluation_matches_the_existing_path_on_calls_in_a_row():
    # two calls in a row on different data and different sizes: the second must not see the first one's sums,
    # counters, sensor positions or profile in the shared array (127 sensors first, then 19)
    cfg5, sig5, pos5 = _batch(5, 10_001, 0)
    g5 = _check(cfg5, sig5, pos5)
    cfg2, sig2, pos2 = _batch(2, 50_003, 1)
    g2 = _check(cfg2, sig2, pos2)
    assert g5.shape == (127,) and g2.shape == (19,)
    # and the same call again gives the same answer (nothing accumulates from call to call)
    g2b, _ = recon.ants_lrf_fit_gains_static(cfg2.sensor_xy, cfg2.knots, cfg2.coeffs[0, 0], sig2, pos2)
    assert np.abs(g2b - g2).max() <= 1e-6 * np.abs(g2).max()
    # failed events (NaN rows) and an empty batch behave as on the existing path
    pos2[::7] = float("nan")
    _check(cfg2, sig2, pos2)
    g_e, used_e = recon.ants_lrf_fit_gains_static(cfg2.sensor_xy, cfg2.knots, cfg2.coeffs[0, 0], sig2[:0].contiguous(),
                                                  pos2[:0].contiguous())
    assert np.isnan(g_e).all() and (used_e == 0).all()


def test_static_scratch_call_leaves_device_memory_alone_and_rejects_sizes_beyond_its_array():
    cfg, sig, pos = _batch(2, 20_000, 2)
    for _ in range(2):                       # first use loads the kernel's module; measure on a later call
        recon.ants_lrf_fit_gains_static(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], sig, pos)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    recon.ants_lrf_fit_gains_static(cfg.sensor_xy, cfg.knots, cfg.coeffs[0, 0], sig, pos)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0                    # no device allocation was made (and kept) by the call
    # more sensors than the array holds
    n_big = 129
    xy = np.zeros((n_big, 2), np.float32)
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_gains_static(xy, cfg.knots, cfg.coeffs[0, 0], torch.zeros((4, n_big), device="cuda"),
                                        torch.ones((4, 4), device="cuda"))
    assert ei.value.status == -2             # ANTS_ERR_UNSUPPORTED
    # a longer profile than the array holds (1025 coefficients)
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_lrf_fit_gains_static(cfg.sensor_xy, cfg.knots, np.ones(1025, np.float32), sig, pos)
    assert ei.value.status == -2
    # the largest sizes it takes: 128 sensors, 1024 coefficients
    rng = np.random.default_rng(0)
    xy = rng.uniform(-50, 50, (128, 2)).astype(np.float32)
    co = (1.0 + rng.uniform(0, 1, 1024)).astype(np.float32)
    kn = np.array([0.0, 200.0], np.float32)
    p = torch.zeros((3000, 4), device="cuda")
    p[:, :2] = torch.from_numpy(rng.uniform(-40, 40, (3000, 2)).astype(np.float32)).cuda()
    p[:, 3] = 100.0
    s = torch.from_numpy(rng.uniform(50, 150, (3000, 128)).astype(np.float32)).cuda()
    g, used = recon.ants_lrf_fit_gains_static(xy, kn, co, s, p)
    g_ref, used_ref = recon.ants_lrf_fit_gains(xy, kn, co, s, p)
    assert np.array_equal(used, used_ref) and np.abs(g - g_ref).max() <= 1e-6 * np.abs(g_ref).max()
    # and a call after the refusals still works
    _check(cfg, sig, pos)
