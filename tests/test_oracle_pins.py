"""Pins of the CPU oracle against what the paper and the mathematics fix
(SURVEY.md section 8(c) "What pins the oracle"; the paper prints no worked
example, PAPER.md has three display equations only).  CPU-only.

Every expected value here comes from a closed form, a library routine
(scipy BSpline, numpy argmin, scipy minimize_scalar) or brute force written in
this file -- never from the oracle itself and never from the CUDA path.
"""
import itertools
import math

import numpy as np
import pytest
from scipy.interpolate import BSpline
from scipy.optimize import minimize_scalar

from oracle import oracle
from paper_1602_07247_b200 import synth


# ---------------------------------------------------------------------------
# helpers written independently of the oracle (library spline + numpy)
# ---------------------------------------------------------------------------
def lib_lrf(cfg, x, y, z=0.0):
    """All sensors' LRF values at one position through scipy's BSpline."""
    r = np.hypot(x - cfg.sensor_xy[:, 0].astype(float), y - cfg.sensor_xy[:, 1].astype(float))
    out = np.empty(cfg.n_sensors)
    for i in range(cfg.n_sensors):
        m = 0 if cfg.n_lrf == 1 else i
        g = float(cfg.gains[i]) if cfg.n_lrf == 1 else 1.0
        if cfg.lrf_dim == 1:
            s = synth.eval_axial(cfg.coeffs[m, 0], float(cfg.knots[0]), float(cfg.knots[1]), r[i:i + 1])[0]
        else:
            s = synth.eval_axial_z(cfg.coeffs[m], cfg.knots[0:2], cfg.knots[2:4], r[i:i + 1],
                                   np.array([z]))[0, 0]
        out[i] = g * s
    return out


def lib_score(cfg, S, x, y, z=0.0):
    """(A, score) by the definitions of PAPER.md:316/328 from library LRF values."""
    L = lib_lrf(cfg, x, y, z)
    S = np.asarray(S, float)
    if cfg.method == 0:
        S = np.maximum(S, 0.0)
        A = S.sum() / L.sum()
        mu = A * L
        t = np.where(S > 0, mu - S - S * np.log(np.where(S > 0, mu / np.where(S > 0, S, 1), 1.0)), mu)
        return A, 2.0 * t.sum()
    w = 1.0 / np.maximum(S, 1.0)
    A = (w * S * L).sum() / (w * L * L).sum()
    return A, (w * (S - A * L) ** 2).sum()


def noise_free(cfg, pos, nph):
    return np.array([0.1 * nph * lib_lrf(cfg, *p) for p in pos], dtype=np.float64)


def blossom_coeffs(lo, hi, n, power):
    h = (hi - lo) / n
    t = lo + (np.arange(n + 7) - 3) * h
    j = np.arange(n + 3)
    a, b, c = t[j + 1], t[j + 2], t[j + 3]
    return {0: np.ones(n + 3), 1: (a + b + c) / 3.0, 2: (a * b + a * c + b * c) / 3.0, 3: a * b * c}[power]


# ---------------------------------------------------------------------------
# spline basis ("B-splines"; reading R7)
# ---------------------------------------------------------------------------
def test_partition_of_unity():
    x = np.linspace(-5, 95, 401)
    assert np.allclose(oracle.spline1(np.ones(19), 0.0, 90.0, x), 1.0, atol=1e-15)


@pytest.mark.parametrize("power", [1, 2, 3])
def test_polynomial_reproduction_by_blossoming(power):
    lo, hi, n = 2.0, 10.0, 8            # knots at integers: coefficients exact in float32
    c = 3.0 * blossom_coeffs(lo, hi, n, power)      # x3: the blossom's /3 would not be exact
    assert np.all(c == c.astype(np.float32))
    x = np.linspace(lo, hi, 257)
    assert np.allclose(oracle.spline1(c, lo, hi, x), 3.0 * x ** power, rtol=1e-13, atol=1e-12)


def test_spline_clamps_outside_range():
    c = np.random.default_rng(1).normal(size=11)
    assert oracle.spline1(c, 1.0, 9.0, -3.0) == oracle.spline1(c, 1.0, 9.0, 1.0)
    assert oracle.spline1(c, 1.0, 9.0, 50.0) == oracle.spline1(c, 1.0, 9.0, 9.0)


def test_spline_matches_scipy_and_is_c2():
    rng = np.random.default_rng(2)
    lo, hi, n = 0.0, 90.0, 16
    c = rng.normal(size=n + 3).astype(np.float32)
    spl = BSpline(synth.uniform_knot_vector(lo, hi, n), c.astype(float), 3)
    x = np.linspace(lo, hi, 1001)
    assert np.allclose(oracle.spline1(c, lo, hi, x), spl(x), rtol=1e-12, atol=1e-13)
    # C2 across every interior knot: one-sided second differences agree
    h, e = (hi - lo) / n, 1e-3
    for k in range(1, n):
        t = lo + k * h
        f = lambda v: oracle.spline1(c, lo, hi, v)
        left = (f(t) - 2 * f(t - e) + f(t - 2 * e)) / e ** 2
        right = (f(t + 2 * e) - 2 * f(t + e) + f(t)) / e ** 2
        assert abs(f(t + 1e-9) - f(t - 1e-9)) < 1e-7
        assert abs(left - right) < 20 * e * np.abs(c).max()      # third derivative jumps only


def test_fit_reproduces_cubic():
    p = lambda r: 1.0 - 0.02 * r + 3e-4 * r ** 2 - 1e-6 * r ** 3
    c = synth.fit_axial(p, 0.0, 90.0, 16)
    x = np.linspace(0, 90, 333)
    assert np.allclose(oracle.spline1(c, 0.0, 90.0, x), p(x), atol=2e-6)


def test_tensor_spline_separable_and_scipy():
    rng = np.random.default_rng(3)
    a, b = rng.normal(size=19).astype(np.float32), rng.normal(size=11).astype(np.float32)
    c = np.outer(b.astype(np.float64), a.astype(np.float64))
    # separable coefficients exactly representable: use small integers
    a = rng.integers(-4, 5, 19).astype(np.float32)
    b = rng.integers(-4, 5, 11).astype(np.float32)
    c = np.outer(b, a).astype(np.float32)
    for r, z in [(0.0, 0.0), (17.3, 4.4), (119.9, 19.9), (120.0, 20.0), (63.0, 10.0)]:
        want = oracle.spline1(a, 0, 120, r) * oracle.spline1(b, 0, 20, z)
        assert math.isclose(oracle.spline2(c, (0, 120), (0, 20), r, z), want, rel_tol=1e-12, abs_tol=1e-12)
    # non-separable coefficients against the library's design matrices
    c = rng.normal(size=(11, 19)).astype(np.float32)
    rr, zz = np.array([3.0, 55.5, 119.0]), np.array([0.5, 9.0, 19.5])
    lib = synth.eval_axial_z(c, (0, 120), (0, 20), rr, zz)
    for j, z in enumerate(zz):
        for i, r in enumerate(rr):
            assert math.isclose(oracle.spline2(c, (0, 120), (0, 20), r, z), lib[j, i], rel_tol=1e-11, abs_tol=1e-12)
    # a transposed coefficient matrix must NOT pass (guards the [z][r] layout)
    assert not math.isclose(oracle.spline2(c, (0, 120), (0, 20), 55.5, 9.0),
                            synth.eval_axial_z(c[:, ::-1], (0, 120), (0, 20), rr, zz)[1, 1], rel_tol=1e-6)


# ---------------------------------------------------------------------------
# LRF: axial distance, gain scaling, individual tables
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("idx", [2, 3, 4])
def test_lrf_matches_library(idx):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    rng = np.random.default_rng(idx)
    for _ in range(5):
        x, y, z = rng.uniform(-70, 70), rng.uniform(-70, 70), rng.uniform(0, 20)
        want = lib_lrf(cfg, x, y, z)
        got = np.array([m.lrf(i, x, y, z) for i in range(cfg.n_sensors)])
        assert np.allclose(got, want, rtol=1e-11, atol=1e-13)


# ---------------------------------------------------------------------------
# centroid
# ---------------------------------------------------------------------------
def test_centroid_special_cases():
    cfg = synth.make_config(2)
    m = oracle.Model.from_config(cfg)
    N = cfg.n_sensors
    for i in (0, 7, 18):                       # one non-zero sensor -> its position
        s = np.zeros(N, np.float32); s[i] = 5.0
        xy, rc = m.centroid(s)
        assert rc == 0 and np.allclose(xy, cfg.sensor_xy[i], atol=1e-12)
    xy, rc = m.centroid(cfg.gains * 3.0)       # S_i = 3 g_i on a symmetric array -> origin
    assert rc == 0 and np.allclose(xy, 0.0, atol=1e-5)
    # gains enter as S_i/g_i: weights 1 and 2 on sensors a, b
    a, b = 3, 11
    s = np.zeros(N, np.float32); s[a] = cfg.gains[a]; s[b] = 2 * cfg.gains[b]
    xy, _ = m.centroid(s)
    assert np.allclose(xy, (cfg.sensor_xy[a].astype(float) + 2 * cfg.sensor_xy[b]) / 3.0, atol=1e-5)
    # unusable events
    assert m.centroid(np.zeros(N, np.float32))[1] == 1
    s = np.ones(N, np.float32); s[4] = np.nan
    assert m.centroid(s)[1] == 1


# ---------------------------------------------------------------------------
# energy and score
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("idx", [2, 3, 4])
def test_score_matches_definition_and_energy_is_the_minimiser(idx):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    ev = synth.generate_events(cfg, 6)
    sig = ev["signals"].numpy()
    pos = ev["true_xyz"].numpy().astype(float)
    for e in range(6):
        x, y, z = pos[e] + np.array([1.3, -0.7, 0.4 if cfg.lrf_dim == 2 else 0.0])
        A, sc = m.score_at(sig[e], cfg.method, x, y, z)
        A_ref, sc_ref = lib_score(cfg, sig[e], x, y, z)
        assert math.isclose(A, A_ref, rel_tol=1e-10) and math.isclose(sc, sc_ref, rel_tol=1e-9)
        # brute-force 1-D minimisation over the energy scale of the same mismatch
        L = lib_lrf(cfg, x, y, z)
        S = sig[e].astype(float)
        if cfg.method == 0:
            S = np.maximum(S, 0)
            nll = lambda a: 2 * np.sum(a * L - S - np.where(S > 0, S * np.log(a * L / np.where(S > 0, S, 1)), 0.0))
        else:
            w = 1 / np.maximum(S, 1)
            nll = lambda a: np.sum(w * (S - a * L) ** 2)
        res = minimize_scalar(nll, bracket=(0.5 * A, 1.5 * A), tol=1e-12)
        assert math.isclose(res.x, A, rel_tol=2e-6)
        assert nll(A) <= nll(A * 1.001) and nll(A) <= nll(A * 0.999)
        assert math.isclose(nll(A), sc, rel_tol=1e-9)


def test_poisson_deviance_zero_iff_mu_equals_s():
    cfg = synth.make_config(1)
    m = oracle.Model.from_config(cfg)
    p = (4.0, -7.5)
    S = noise_free(cfg, [p], 2000.0)[0].astype(np.float32)
    A, D = m.score_at(S, 0, *p)
    assert math.isclose(A, 200.0, rel_tol=1e-6) and 0 <= D < 1e-8
    for q in [(4.5, -7.5), (4.0, -6.5), (-4.0, 7.5)]:
        assert m.score_at(S, 0, *q)[1] > 1e-3
    rng = np.random.default_rng(5)
    for _ in range(20):
        S = rng.poisson(30, cfg.n_sensors).astype(np.float32)
        assert m.score_at(S, 0, rng.uniform(-20, 20), rng.uniform(-20, 20))[1] >= 0.0
    # S_i = 0 terms contribute mu_i; negative signals are clipped in ML mode
    S0 = np.array([0, 10, 20, 0, 5, 0, 3], np.float32)
    Sneg = S0.copy(); Sneg[0] = -2.5
    assert m.score_at(S0, 0, 1.0, 2.0) == m.score_at(Sneg, 0, 1.0, 2.0)
    assert math.isclose(m.score_at(S0, 0, 1.0, 2.0)[1], lib_score(cfg, S0, 1.0, 2.0)[1], rel_tol=1e-10)


def test_invalid_nodes():
    cfg = synth.make_config(4)
    m = oracle.Model.from_config(cfg)
    S = np.full(cfg.n_sensors, 10, np.float32)
    for z in (-0.01, 20.01):                                 # R6: z outside the LRF range
        A, sc = m.score_at(S, 0, 0.0, 0.0, z)
        assert math.isnan(A) and sc == math.inf
    assert np.isfinite(m.score_at(S, 0, 0.0, 0.0, 20.0)[1])
    # L_i <= 0 with S_i > 0 (Poisson) -> invalid
    cfg1 = synth.make_config(1)
    neg = oracle.Model(cfg1.sensor_xy, cfg1.gains, cfg1.knots, -cfg1.coeffs, 1, 1, 16, 0)
    assert neg.score_at(np.ones(7, np.float32), 0, 0.0, 0.0)[1] == math.inf


# ---------------------------------------------------------------------------
# search
# ---------------------------------------------------------------------------
def np_grid_argmin(cfg, S, centre, h_xy, h_z):
    """Independent numpy evaluation of one grid iteration: (index, scores)."""
    G = cfg.nodes_per_axis
    half = 0.5 * (G - 1)
    Gz = G if cfg.dim == 3 else 1
    sc = np.empty(Gz * G * G)
    for iz, iy, ix in itertools.product(range(Gz), range(G), range(G)):
        z = centre[2] + (iz - half) * h_z if cfg.dim == 3 else centre[2]
        if cfg.lrf_dim == 2 and not (cfg.knots[2] <= z <= cfg.knots[3]):
            sc[(iz * G + iy) * G + ix] = np.inf
            continue
        sc[(iz * G + iy) * G + ix] = lib_score(cfg, S, centre[0] + (ix - half) * h_xy,
                                               centre[1] + (iy - half) * h_xy, z)[1]
    return int(np.argmin(sc)), sc


@pytest.mark.parametrize("idx,n_ev", [(1, 12), (3, 3), (4, 2)])
def test_single_iteration_equals_numpy_argmin(idx, n_ev):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    sig = synth.generate_events(cfg, n_ev)["signals"].numpy()
    g = oracle.grid_params(cfg.dim, cfg.nodes_per_axis, cfg.step0_xy, cfg.step0_z, cfg.factor, 1)
    out = oracle.reconstruct(m, sig, g, cfg.method, trace=True)
    G, half = cfg.nodes_per_axis, 0.5 * (cfg.nodes_per_axis - 1)
    for e in range(n_ev):
        xy, _ = m.centroid(sig[e], cfg.method)
        z0 = 0.5 * (cfg.knots[2] + cfg.knots[3]) if cfg.lrf_dim == 2 else 0.0
        idx_np, sc = np_grid_argmin(cfg, sig[e], (xy[0], xy[1], z0), cfg.step0_xy, cfg.step0_z)
        assert out["idx"][e, 0] == idx_np
        srt = np.sort(sc)
        assert math.isclose(out["best"][e, 0], srt[0], rel_tol=1e-9)
        assert math.isclose(out["second"][e, 0], srt[1], rel_tol=1e-9)
        ix, iy, iz = idx_np % G, (idx_np // G) % G, idx_np // (G * G)
        want = [xy[0] + (ix - half) * cfg.step0_xy, xy[1] + (iy - half) * cfg.step0_xy,
                z0 + (iz - half) * cfg.step0_z if cfg.dim == 3 else z0]
        assert np.allclose(out["xyzA"][e, :3], want, atol=1e-12)
        assert math.isclose(out["score"][e], srt[0], rel_tol=1e-9)


def test_multi_iteration_walk_matches_numpy_replay():
    """K iterations = K independent numpy argmins chained by 'recentre, halve the step'."""
    cfg = synth.make_config(1)
    m = oracle.Model.from_config(cfg)
    sig = synth.generate_events(cfg, 3)["signals"].numpy()
    K = 4
    g = oracle.grid_params(2, 9, 5.0, 0.0, 0.5, K)
    out = oracle.reconstruct(m, sig, g, 0, trace=True)
    for e in range(3):
        c = list(m.centroid(sig[e])[0]) + [0.0]
        h = 5.0
        for k in range(K):
            i, _ = np_grid_argmin(cfg, sig[e], c, h, 0.0)
            assert out["idx"][e, k] == i
            c[0] += (i % 9 - 4) * h
            c[1] += (i // 9 - 4) * h
            h *= 0.5
        assert np.allclose(out["xyzA"][e, :2], c[:2], atol=1e-12)


def lib_lrf_fast(cfg, x, y, z=0.0):
    """lib_lrf with one library call per table instead of one per sensor (same scipy evaluation)."""
    r = np.hypot(x - cfg.sensor_xy[:, 0].astype(float), y - cfg.sensor_xy[:, 1].astype(float))
    if cfg.n_lrf != 1:
        return lib_lrf(cfg, x, y, z)
    if cfg.lrf_dim == 1:
        s = synth.eval_axial(cfg.coeffs[0, 0], float(cfg.knots[0]), float(cfg.knots[1]), r)
    else:
        s = synth.eval_axial_z(cfg.coeffs[0], cfg.knots[0:2], cfg.knots[2:4], r, np.array([z]))[0]
    return cfg.gains.astype(float) * s


def np_walk(cfg, S, start, K, G, h_xy, h_z, f):
    """The contracting-grid walk of PAPER.md:328 replayed with numpy: per iteration an argmin (first
    minimum in linear-index order) over library-evaluated node scores, then recentre and contract."""
    half = 0.5 * (G - 1)
    Gz = G if cfg.dim == 3 else 1
    c = list(start)
    path = []
    for _ in range(K):
        sc = np.full(Gz * G * G, np.inf)
        for iz, iy, ix in itertools.product(range(Gz), range(G), range(G)):
            z = c[2] + (iz - half) * h_z if cfg.dim == 3 else c[2]
            if cfg.lrf_dim == 2 and not (cfg.knots[2] <= z <= cfg.knots[3]):
                continue
            L = lib_lrf_fast(cfg, c[0] + (ix - half) * h_xy, c[1] + (iy - half) * h_xy, z)
            Sv = np.asarray(S, float)
            if cfg.method == 0:
                Sv = np.maximum(Sv, 0.0)
                mu = Sv.sum() / L.sum() * L
                t = np.where(Sv > 0, mu - Sv - Sv * np.log(np.where(Sv > 0, mu / np.where(Sv > 0, Sv, 1), 1.0)), mu)
                sc[(iz * G + iy) * G + ix] = 2.0 * t.sum()
            else:
                w = 1.0 / np.maximum(Sv, 1.0)
                A = (w * Sv * L).sum() / (w * L * L).sum()
                sc[(iz * G + iy) * G + ix] = (w * (Sv - A * L) ** 2).sum()
        i = int(np.argmin(sc))                 # numpy: the first occurrence of the minimum
        path.append(i)
        ix, iy, iz = i % G, (i // G) % G, i // (G * G)
        c[0] += (ix - half) * h_xy
        c[1] += (iy - half) * h_xy
        if cfg.dim == 3:
            c[2] += (iz - half) * h_z
        h_xy *= f
        h_z *= f
    return path, c


@pytest.mark.parametrize("idx,G,K,f,n_ev", [(3, 5, 4, 0.5, 2),      # chi-square, one table per sensor
                                            (4, 4, 3, 0.5, 2),      # 3-D, z recentring, even G
                                            (4, 3, 4, 0.6, 1),      # 3-D with f != 0.5
                                            (2, 7, 5, 0.4, 3),      # f != 0.5, gains, noise
                                            (1, 6, 4, 0.7, 3)])     # even G, f != 0.5
def test_multi_iteration_walk_matches_numpy_replay_other_configs(idx, G, K, f, n_ev):
    """The chained walk for chi-square (config 3), the 3-D search with z recentring (config 4) and
    contraction factors other than 0.5 (h_k = h_0 f^k, R1)."""
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    sig = synth.generate_events(cfg, n_ev)["signals"].numpy()
    h_xy = cfg.step0_xy * (cfg.nodes_per_axis - 1) / (G - 1)
    h_z = cfg.step0_z * (cfg.nodes_per_axis - 1) / (G - 1) if cfg.dim == 3 else 0.0
    g = oracle.grid_params(cfg.dim, G, h_xy, h_z, f, K)
    out = oracle.reconstruct(m, sig, g, cfg.method, trace=True)
    for e in range(n_ev):
        xy, _ = m.centroid(sig[e], cfg.method)
        z0 = 0.5 * (float(cfg.knots[2]) + float(cfg.knots[3])) if cfg.lrf_dim == 2 else 0.0
        path, c = np_walk(cfg, sig[e], (xy[0], xy[1], z0), K, G, float(np.float32(h_xy)), float(np.float32(h_z)),
                          float(np.float32(f)))
        assert list(out["idx"][e]) == path
        assert np.allclose(out["xyzA"][e, :3], c, atol=1e-11)


# ---------------------------------------------------------------------------
# tie-break (R9): the first strict minimum in linear-index order
# ---------------------------------------------------------------------------
def _collinear_model(lrf_dim):
    """Sensors on the line y = 0: nodes mirrored in y see bit-identical distances, so their scores tie
    EXACTLY (same operands in the same order), and the centroid's y is exactly 0."""
    base = synth.make_config(4 if lrf_dim == 2 else 2)
    xy = np.array([[-31.0, 0.0], [-9.5, 0.0], [4.25, 0.0], [22.0, 0.0], [40.5, 0.0]], np.float32)
    g = np.array([1.0, 0.9, 1.1, 1.05, 0.95], np.float32)
    return base, oracle.Model(xy, g, base.knots, base.coeffs, 1, lrf_dim, base.n_int_r, base.n_int_z)


@pytest.mark.parametrize("method", [0, 1, 2])
@pytest.mark.parametrize("G", [2, 4, 6])
def test_tie_break_lowest_linear_index_2d(G, method):
    base, m = _collinear_model(1)
    S = np.array([[12, 55, 80, 31, 7], [3, 9, 40, 90, 60]], np.float32)
    g = oracle.grid_params(2, G, 3.0, 0.0, 0.5, 1)
    out = oracle.reconstruct(m, S, g, method, trace=True)
    for e in range(2):
        xy, _ = m.centroid(S[e], method)
        assert xy[1] == 0.0
        # scores of all nodes, through the oracle's own score_at (the pin is the ORDER rule, not the score)
        half = 0.5 * (G - 1)
        sc = np.array([m.score_at(S[e], method, xy[0] + (ix - half) * 3.0, (iy - half) * 3.0)[1]
                       for iy in range(G) for ix in range(G)])
        best = sc.min()
        tied = np.flatnonzero(sc == best)
        assert len(tied) >= 2                         # the mirrored partner ties exactly
        assert tied[0] // G == G - 1 - tied[-1] // G and tied[0] % G == tied[-1] % G
        assert out["idx"][e, 0] == tied[0]            # the LOWEST linear index wins
        assert out["best"][e, 0] == best and out["second"][e, 0] == best
        assert out["xyzA"][e, 1] == (tied[0] // G - half) * 3.0


def test_tie_break_lowest_linear_index_3d():
    base, m = _collinear_model(2)
    S = np.array([[12, 55, 80, 31, 7]], np.float32)
    G = 4
    g = oracle.grid_params(3, G, 3.0, 2.0, 0.5, 1)
    out = oracle.reconstruct(m, S, g, 0, trace=True)
    i = int(out["idx"][0, 0])
    ix, iy, iz = i % G, (i // G) % G, i // (G * G)
    assert iy < G - 1 - iy                            # the partner (ix, G-1-iy, iz) has the higher index
    assert out["best"][0, 0] == out["second"][0, 0]   # and ties exactly
    xy, _ = m.centroid(S[0], 0)
    half = 0.5 * (G - 1)
    p = (xy[0] + (ix - half) * 3.0, (iy - half) * 3.0, 10.0 + (iz - half) * 2.0)
    a = m.score_at(S[0], 0, p[0], p[1], p[2])[1]
    b = m.score_at(S[0], 0, p[0], -p[1], p[2])[1]
    assert a == b == out["best"][0, 0]


def test_lattice_brute_force_tiny():
    """With factor 0.5 every visited node lies on seed + m*h_K: the exhaustive minimum
    over that lattice (window = everything the search could reach) is <= the oracle's
    score, with equality on a unimodal (noise-free) surface."""
    cfg = synth.make_config(1)
    m = oracle.Model.from_config(cfg)
    K = 4
    g = oracle.grid_params(2, 5, 4.0, 0.0, 0.5, K)
    hK = 4.0 * 0.5 ** (K - 1)
    pos = [(3.0, -5.0), (-11.0, 8.0)]
    sig_clean = noise_free(cfg, pos, 2000.0).astype(np.float32)
    sig_noisy = synth.generate_events(cfg, 2)["signals"].numpy()
    for sig, unimodal in ((sig_clean, True), (sig_noisy, False)):
        out = oracle.reconstruct(m, sig, g, 0)
        for e in range(2):
            xy, _ = m.centroid(sig[e])
            reach = int(round(2 * sum(4.0 * 0.5 ** k for k in range(K)) / hK))
            best = math.inf
            for jy in range(-reach, reach + 1):
                for jx in range(-reach, reach + 1):
                    best = min(best, lib_score(cfg, sig[e], xy[0] + jx * hK, xy[1] + jy * hK)[1])
            assert best <= out["score"][e] * (1 + 1e-9) + 1e-12
            if unimodal:
                assert abs(best - out["score"][e]) <= 1e-9 + 1e-9 * best


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_noise_free_recovery(idx):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    rng = np.random.default_rng(10 + idx)
    n = 6 if idx != 4 else 3
    ext = 0.5 * cfg.extent
    pos = [(rng.uniform(-ext, ext) * 0.7, rng.uniform(-ext, ext) * 0.7,
            rng.uniform(4, 16) if cfg.lrf_dim == 2 else 0.0) for _ in range(n)]
    sig = noise_free(cfg, pos, 3000.0).astype(np.float32)
    out = oracle.reconstruct(m, sig, oracle.grid_from_config(cfg), cfg.method)
    hxy, hz = cfg.final_step()
    for e, p in enumerate(pos):
        assert abs(out["xyzA"][e, 0] - p[0]) <= hxy and abs(out["xyzA"][e, 1] - p[1]) <= hxy
        if cfg.dim == 3:
            assert abs(out["xyzA"][e, 2] - p[2]) <= hz
        assert math.isclose(out["xyzA"][e, 3], 300.0, rel_tol=1e-3)


def test_mirror_symmetry():
    """Negating every sensor x negates the reconstructed x and changes nothing else
    (IEEE negation is exact and an odd G makes the grid its own mirror image)."""
    cfg = synth.make_config(2)
    sig = synth.generate_events(cfg, 64)["signals"].numpy()
    m = oracle.Model.from_config(cfg)
    xy_m = cfg.sensor_xy.copy(); xy_m[:, 0] = -xy_m[:, 0]
    mm = oracle.Model(xy_m, cfg.gains, cfg.knots, cfg.coeffs, 1, 1, 16, 0)
    g = oracle.grid_from_config(cfg)
    a, b = oracle.reconstruct(m, sig, g, 0, trace=True), oracle.reconstruct(mm, sig, g, 0, trace=True)
    same = np.all(a["idx"] % 9 == 8 - b["idx"] % 9, axis=1) & np.all(a["idx"] // 9 == b["idx"] // 9, axis=1)
    assert same.mean() > 0.9                      # exact ties may resolve differently
    assert np.array_equal(a["xyzA"][same, 0], -b["xyzA"][same, 0])
    assert np.array_equal(a["xyzA"][same, 1:], b["xyzA"][same, 1:])
    assert np.array_equal(a["score"][same], b["score"][same])


@pytest.mark.parametrize("idx", [1, 3])
def test_power_of_two_scaling(idx):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    sig = synth.generate_events(cfg, 16)["signals"].numpy()
    sig = np.maximum(sig, 1.0)                    # keeps max(S,1) weights scaling exactly
    g = oracle.grid_from_config(cfg)
    a, b = oracle.reconstruct(m, sig, g, cfg.method), oracle.reconstruct(m, 2 * sig, g, cfg.method)
    assert np.array_equal(a["xyzA"][:, :3], b["xyzA"][:, :3])
    assert np.allclose(2 * a["xyzA"][:, 3], b["xyzA"][:, 3], rtol=1e-14)
    assert np.allclose(2 * a["score"], b["score"], rtol=1e-12)


def test_failed_events_and_all_invalid_grid():
    cfg = synth.make_config(1)
    m = oracle.Model.from_config(cfg)
    sig = synth.generate_events(cfg, 3)["signals"].numpy()
    sig[1] = 0.0
    out = oracle.reconstruct(m, sig, oracle.grid_from_config(cfg), 0, trace=True)
    assert np.all(np.isnan(out["xyzA"][1])) and out["score"][1] == np.inf and np.all(out["idx"][1] == -1)
    assert np.all(np.isfinite(out["xyzA"][[0, 2]]))
    # a non-finite RAW signal fails the event, -inf included (it must not be clipped to 0 first)
    for bad in (np.nan, np.inf, -np.inf):
        for method in (0, 1):
            s2 = sig.copy()
            s2[2, 3] = bad
            o2 = oracle.reconstruct(m, s2, oracle.grid_from_config(cfg), method)
            assert np.all(np.isnan(o2["xyzA"][2])) and o2["score"][2] == np.inf and np.all(np.isfinite(o2["xyzA"][0]))
            assert m.centroid(s2[2], method)[1] == 1 and m.start(s2[2], method, 1)[1] == 1
    with pytest.raises(ValueError):
        oracle.reconstruct(m, sig, oracle.grid_params(2, 1, 5.0, 0, 0.5, 3), 0)
    with pytest.raises(ValueError):
        oracle.reconstruct(m, sig, oracle.grid_params(3, 5, 5.0, 1.0, 0.5, 3), 0)   # 3-D needs L(r,z)


def test_statistics_sanity():
    """Sanity, not parity: flood-field resolution and energy are in the expected range."""
    cfg = synth.make_config(2)
    ev = synth.generate_events(cfg, 1500)
    out = oracle.reconstruct(oracle.Model.from_config(cfg), ev["signals"].numpy(),
                             oracle.grid_from_config(cfg), 0)
    err = out["xyzA"][:, :2] - ev["true_xyz"].numpy()[:, :2]
    assert 0.8 < np.sqrt((err ** 2).mean()) < 3.0
    ratio = out["xyzA"][:, 3] / (0.1 * ev["n_ph"].numpy())
    assert 0.97 < ratio.mean() < 1.05
