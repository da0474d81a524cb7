"""CPU pins of the oracle's continuous refinement (R34; the gradient-based
minimisation "versus two (XY) or three (XYZ) spatial coordinates" that Minuit2 performs in ANTS2, here a
Levenberg-Marquardt iteration on the node score with the energy eliminated).

Expected values: central differences of the (already pinned) score, scipy.optimize.minimize on that score from the
same start, and the monotone decrease the accept rule guarantees."""
import numpy as np
import pytest
from scipy.optimize import minimize

from oracle import oracle
from paper_1602_07247_b200 import synth


def _setup(idx, method, n=12, k_grid=5):
    cfg = synth.make_config(idx)
    cfg.method = method
    ev = synth.generate_events(cfg, n)
    sig = ev["signals"].numpy()
    m = oracle.Model.from_config(cfg)
    coarse = synth.make_config(idx)
    coarse.method, coarse.n_iter = method, k_grid
    start = oracle.reconstruct(m, sig, oracle.grid_from_config(coarse), method)
    return cfg, m, sig, start


@pytest.mark.parametrize("idx", [2, 3, 4, 6, 7, 8])
def test_lrf_gradient_against_central_differences(idx):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    rng = np.random.default_rng(idx)
    h = 1e-5
    for _ in range(40):
        i = int(rng.integers(cfg.n_sensors))
        x, y = rng.uniform(-0.8 * cfg.extent, 0.8 * cfg.extent, 2)
        z = rng.uniform(2.0, 18.0)
        v, g = oracle.lrf_grad(m, i, x, y, z)
        assert abs(v - m.lrf(i, x, y, z)) <= 1e-14 * max(1.0, abs(v))
        num = np.array([(m.lrf(i, x + h, y, z) - m.lrf(i, x - h, y, z)) / (2 * h),
                        (m.lrf(i, x, y + h, z) - m.lrf(i, x, y - h, z)) / (2 * h),
                        (m.lrf(i, x, y, z + h) - m.lrf(i, x, y, z - h)) / (2 * h)])
        if cfg.lrf_dim == 5:                      # piecewise linear in z: skip points next to a plane
            zp = np.linspace(0, 20, cfg.n_planes)
            if np.min(np.abs(zp - z)) < 2 * h:
                continue
        assert np.allclose(g, num, rtol=2e-5, atol=1e-7 * max(1.0, abs(v))), (idx, i, x, y, z, g, num)


@pytest.mark.parametrize("idx,method", [(2, 0), (3, 1), (3, 2), (4, 0), (6, 1), (7, 0), (8, 0)])
def test_score_gradient_against_central_differences(idx, method):
    cfg, m, sig, start = _setup(idx, method, n=6)
    dim = cfg.dim
    h = 1e-5
    for e in range(len(sig)):
        x, y, z = start["xyzA"][e, :3] + np.array([0.31, -0.23, 0.17 if dim == 3 else 0.0])
        if dim == 3:
            z = min(max(z, 0.5), 19.5)           # stay inside the z range: outside it the node is invalid (R6)
        A, F, g, H, rc = oracle.score_grad(m, sig[e], method, x, y, z, dim=dim)
        assert rc == 0
        A0, F0 = m.score_at(sig[e], method, x, y, z)
        assert abs(F - F0) <= 1e-10 * abs(F0) and abs(A - A0) <= 1e-12 * abs(A0)
        f = lambda p: m.score_at(sig[e], method, p[0], p[1], p[2])[1]
        p0 = np.array([x, y, z])
        for a in range(dim):
            d = np.zeros(3)
            d[a] = h
            num = (f(p0 + d) - f(p0 - d)) / (2 * h)
            assert abs(g[a] - num) <= 2e-5 * max(abs(num), 1.0), (idx, e, a, g[a], num)
        assert np.allclose(H, H.T) and np.all(np.linalg.eigvalsh(H[:dim, :dim]) > 0)


@pytest.mark.parametrize("idx,method", [(1, 0), (2, 0), (3, 1), (3, 2), (4, 0), (5, 0), (6, 1), (7, 0), (8, 0)])
def test_refinement_reaches_the_scipy_minimum_and_never_increases(idx, method):
    """The objective is only piecewise smooth (a clamped radius, R5, and the z planes of a Sliced LRF put kinks in
    it), so a quasi-Newton library routine is a reference only where it converges: there the LM result must be as
    good and at the same place; everywhere F must fall monotonically with the number of steps."""
    cfg, m, sig, start = _setup(idx, method, n=8 if idx in (5, 7) else 12)
    dim = cfg.dim
    runs = [oracle.refine(m, sig, method, start["xyzA"][:, :3], n, dim=dim) for n in (0, 1, 3, 8, 30)]
    zlo, zhi = (0.0, 20.0) if dim == 3 else (None, None)
    n_checked = 0
    for e in range(len(sig)):
        if not np.isfinite(start["score"][e]):
            continue
        F = [r["score"][e] for r in runs]
        assert abs(F[0] - start["score"][e]) <= 1e-10 * abs(F[0])           # zero steps: the start point's own score
        assert all(F[i + 1] <= F[i] for i in range(len(F) - 1)), F
        res = runs[-1]
        # energy and score at the refined point are the pinned definition
        A, Fd = m.score_at(sig[e], method, *res["xyzA"][e, :3])
        assert abs(Fd - res["score"][e]) <= 1e-10 * abs(Fd) and abs(A - res["xyzA"][e, 3]) <= 1e-12 * abs(A)

        def f(p):
            z = p[2] if dim == 3 else start["xyzA"][e, 2]
            return m.score_at(sig[e], method, p[0], p[1], z)[1]
        def jac(p):            # the analytic gradient, itself pinned against central differences above
            z = p[2] if dim == 3 else start["xyzA"][e, 2]
            return oracle.score_grad(m, sig[e], method, p[0], p[1], z, dim=dim)[2][:dim]
        x0 = start["xyzA"][e, :dim]
        bounds = None if dim == 2 else [(None, None), (None, None), (zlo, zhi)]
        ref = minimize(f, x0, jac=jac, method="L-BFGS-B" if dim == 3 else "BFGS", bounds=bounds,
                       options=dict(gtol=1e-7, ftol=1e-15) if dim == 3 else dict(gtol=1e-7))
        assert res["score"][e] <= ref.fun + 2e-4 * abs(ref.fun), (idx, e, res["score"][e], ref.fun)
        if ref.success and (dim == 2 or 0.05 < ref.x[2] < 19.95):
            n_checked += 1
            assert res["score"][e] <= ref.fun + 1e-8 * abs(ref.fun), (idx, e, res["score"][e], ref.fun)
            assert np.abs(res["xyzA"][e, :dim] - ref.x).max() <= 2e-3, (idx, e, res["xyzA"][e], ref.x)
    assert n_checked >= 3


def test_refinement_leaves_failed_events_and_handles_selection():
    cfg = synth.make_config(2)
    cfg.signal_min, cfg.dist_max = 3.0, 70.0
    m = oracle.Model.from_config(cfg)
    sig = synth.generate_events(cfg, 10)["signals"].numpy()
    sig[3, 5] = np.nan
    start = oracle.reconstruct(m, sig, oracle.grid_from_config(cfg), 0)
    assert np.isnan(start["xyzA"][3, 0])
    res = oracle.refine(m, sig, 0, start["xyzA"][:, :3], 6)
    assert np.isnan(res["xyzA"][3]).all() or np.isnan(res["xyzA"][3, 0])
    ok = np.isfinite(start["score"])
    assert (res["score"][ok] <= start["score"][ok] * (1 + 1e-12)).all()
    # the refined score is the score over the event's active sensors (same selection as the grid search)
    for e in np.flatnonzero(ok)[:4]:
        A, F = m.score_at(sig[e], 0, *res["xyzA"][e, :3])
        assert abs(F - res["score"][e]) <= 1e-10 * abs(F)
