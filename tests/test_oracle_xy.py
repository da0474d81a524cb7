"""CPU pins of the oracle's XY-type LRF parameterisations (section 6.1: "XY LRF", "Composite
LRF", "Sliced LRF") and of the symmetry grouping, readings R30-R33 of DESIGN.md.

Expected values come from scipy design matrices, closed forms and numpy loops written here, never from the
oracle or the CUDA path."""
import numpy as np
import pytest

from oracle import fit as ofit
from oracle import oracle
from paper_1602_07247_b200 import synth


def _scipy_xy(cfg, tab, plane, u, v):
    """library evaluation of table `tab`, plane `plane`, at local coordinates (u, v)"""
    k = cfg.knots_xy
    return float(synth.eval_xy_points(cfg.coeffs_xy[tab, plane], (float(k[0]), float(k[1])), (float(k[2]), float(k[3])),
                                      np.array([u]), np.array([v]))[0])


def _local(cfg, i, x, y):
    dx, dy = x - float(cfg.sensor_xy[i, 0]), y - float(cfg.sensor_xy[i, 1])
    if cfg.xform is None:
        return dx, dy
    T = cfg.xform[i].astype(np.float64)
    return T[0] * dx + T[1] * dy, T[2] * dx + T[3] * dy


def _lrf_ref(cfg, i, x, y, z):
    """L_i(p) from the definitions R30-R32 with library spline evaluations"""
    tab = int(cfg.group[i]) if cfg.group is not None else (0 if cfg.n_lrf == 1 else i)
    g = float(cfg.gains[i]) if (cfg.group is not None or cfg.n_lrf == 1) else 1.0
    u, v = _local(cfg, i, x, y)
    if cfg.lrf_dim == 3:
        return g * _scipy_xy(cfg, tab, 0, u, v)
    if cfg.lrf_dim == 4:
        r = np.hypot(x - float(cfg.sensor_xy[i, 0]), y - float(cfg.sensor_xy[i, 1]))
        ax = float(synth.eval_axial(cfg.coeffs[tab, 0], float(cfg.knots[0]), float(cfg.knots[1]), np.array([r]))[0])
        return g * (ax + _scipy_xy(cfg, tab, 0, u, v))
    z_lo, z_hi = float(cfg.knots_xy[4]), float(cfg.knots_xy[5])
    dz = (z_hi - z_lo) / (cfg.n_planes - 1)
    zc = min(max(z, z_lo), z_hi)
    p = min(int(np.floor((zc - z_lo) / dz)), cfg.n_planes - 2)
    w = (zc - (z_lo + p * dz)) / dz
    return g * ((1 - w) * _scipy_xy(cfg, tab, p, u, v) + w * _scipy_xy(cfg, tab, p + 1, u, v))


@pytest.mark.parametrize("idx", [6, 7, 8])
def test_xy_type_lrfs_equal_the_library_evaluation(idx):
    cfg = synth.make_config(idx)
    m = oracle.Model.from_config(cfg)
    rng = np.random.default_rng(idx)
    for _ in range(120):
        i = int(rng.integers(cfg.n_sensors))
        x, y = rng.uniform(-cfg.extent * 1.3, cfg.extent * 1.3, 2)        # also outside the tabulated range (clamped, R5)
        z = rng.uniform(0.0, 20.0)
        ref = _lrf_ref(cfg, i, x, y, z)
        assert abs(m.lrf(i, x, y, z) - ref) <= 1e-11 * max(1.0, abs(ref)), (idx, i, x, y, z)


def test_xy_spline_is_transposition_sensitive_and_separable():
    """c[b][a] = beta_b alpha_a gives the product of two 1-D splines: u runs along the fastest index."""
    rng = np.random.default_rng(0)
    al, be = rng.uniform(0.5, 1.5, 9).astype(np.float32), rng.uniform(0.5, 1.5, 7).astype(np.float32)
    c = (be[:, None].astype(np.float64) * al[None, :].astype(np.float64)).astype(np.float32)
    m = oracle.Model([[0.0, 0.0]], [1.0], None, None, 1, 3, 0, 0, n_int_x=6, n_int_y=4,
                     knots_xy=[-6, 6, -4, 4], coeffs_xy=c[None, None])
    for u, v in ((-5.1, 3.3), (0.2, -0.7), (4.9, 1.1)):
        want = oracle.spline1(al, -6, 6, u) * oracle.spline1(be, -4, 4, v)
        got = m.lrf(0, u, v)
        # the products c[b][a] were rounded to float32: compare with a tolerance of that rounding
        assert abs(got - want) <= 2e-7 * abs(want)
    assert abs(m.lrf(0, 3.3, -5.1 * 4 / 6) - m.lrf(0, -5.1, 3.3)) > 1e-3      # not symmetric under u <-> v


def test_sliced_lrf_on_planes_midway_and_linear_between():
    cfg = synth.make_config(7)
    m = oracle.Model.from_config(cfg)
    i, x, y = 5, 11.0, -23.0
    u, v = _local(cfg, i, x, y)
    planes = np.linspace(0.0, 20.0, 5)
    on = [_scipy_xy(cfg, 0, p, u, v) for p in range(5)]
    for p, zp in enumerate(planes):
        assert abs(m.lrf(i, x, y, zp) - on[p]) <= 1e-12 * on[p]                      # on a plane: that plane's XY LRF
    for p in range(4):
        zm = 0.5 * (planes[p] + planes[p + 1])
        assert abs(m.lrf(i, x, y, zm) - 0.5 * (on[p] + on[p + 1])) <= 1e-12 * on[p]  # midway: the mean of the two
        a, b, c = (m.lrf(i, x, y, planes[p] + f * 5.0) for f in (0.2, 0.5, 0.8))
        assert abs(a - 2 * b + c) <= 1e-12 * abs(b)                                   # linear in z between planes
    # outside the z range the node is invalid (R6)
    sig = synth.generate_events(cfg, 4)["signals"].numpy()
    assert m.score_at(sig[0], 0, x, y, 20.5)[1] == np.inf and m.score_at(sig[0], 0, x, y, -0.1)[1] == np.inf
    assert np.isfinite(m.score_at(sig[0], 0, x, y, 20.0)[1])


def test_composite_is_the_sum_of_its_components():
    cfg = synth.make_config(8)
    m = oracle.Model.from_config(cfg)
    ax = oracle.Model(cfg.sensor_xy, cfg.gains, cfg.knots, cfg.coeffs, 1, 1, cfg.n_int_r, 0)
    xy = oracle.Model(cfg.sensor_xy, cfg.gains, None, None, 1, 3, 0, 0, n_int_x=cfg.n_int_x, n_int_y=cfg.n_int_y,
                      knots_xy=cfg.knots_xy, coeffs_xy=cfg.coeffs_xy)
    for i, x, y in ((0, 3.0, 4.0), (7, -31.0, 12.5), (18, 55.0, -40.0)):
        assert abs(m.lrf(i, x, y) - (ax.lrf(i, x, y) + xy.lrf(i, x, y))) <= 1e-15 + 1e-14 * abs(m.lrf(i, x, y))


def test_symmetry_groups_orbit_counts_and_frames():
    """R33.  Orbit counts from group theory: an 8 x 8 square grid has 16 orbits under the 4 rotations and 10 under
    D4 (one quadrant of 16 cells folded over its diagonal: 4 + 6); a hexagonal array of 3 rings has, ring by ring,
    1 + 1 + 2 + 3 = 7 orbits under the 6 rotations and 1 + 1 + 2 + 2 = 6 with the mirror.  Frames: turning a
    sensor's position back by its own frame gives its group's reference position."""
    sq, hx = synth.square_array(8, 6.0), synth.hex_array(3, 30.0)
    for xy, n_fold, reflect, want in ((sq, 4, False, 16), (sq, 4, True, 10), (hx, 6, False, 7), (hx, 6, True, 6),
                                      (sq, 2, True, 16), (synth.hex_array(2, 30.0), 6, True, 4)):
        group, xform, n = ofit.group_by_symmetry(xy, n_fold, reflect)
        assert n == want and group.min() == 0 and group.max() == n - 1
        for gi in range(n):
            members = np.flatnonzero(group == gi)
            ref = members[0]
            assert np.array_equal(xform[ref], [1, 0, 0, 1])
            for i in members:
                T = xform[i].astype(np.float64).reshape(2, 2)
                assert abs(np.linalg.det(T)) == pytest.approx(1.0, abs=1e-6)
                assert np.allclose(T @ xy[i].astype(np.float64), xy[ref].astype(np.float64), atol=1e-3)
    g2, x2, n2 = synth.symmetry_groups(sq, 4, True)          # the input generator's own version agrees
    g1, x1, n1 = ofit.group_by_symmetry(sq, 4, True)
    assert n1 == n2 and np.array_equal(g1, g2) and np.allclose(x1, x2, atol=1e-6)


def test_symmetric_sharing_turns_the_response_with_the_sensor():
    """A sensor that the rotation Q maps the reference onto responds at Q p as the reference does at p."""
    cfg = synth.make_config(6)
    m = oracle.Model.from_config(cfg)
    rng = np.random.default_rng(2)
    P = cfg.sensor_xy.astype(np.float64)
    for gi in range(cfg.n_lrf):
        members = np.flatnonzero(cfg.group == gi)
        ref = members[0]
        for i in members[1:]:
            Q = cfg.xform[i].astype(np.float64).reshape(2, 2).T          # T_i = Q^T
            assert np.allclose(Q @ P[ref], P[i], atol=1e-3)
            p = rng.uniform(-20, 20, 2)
            q = Q @ p
            assert abs(m.lrf(i, q[0], q[1]) - m.lrf(ref, p[0], p[1])) <= 1e-6 * abs(m.lrf(ref, p[0], p[1])) + 1e-9


def test_event_generator_evaluates_the_same_xy_splines():
    """synth's torch evaluation of the XY-type LRFs (used to draw the signals) equals the scipy evaluation."""
    for idx in (6, 7, 8):
        cfg = synth.make_config(idx)
        ev = synth.generate_events(cfg, 40, noise_free=True)
        sig, pos, nph = ev["signals"].numpy().astype(np.float64), ev["true_xyz"].numpy().astype(np.float64), ev["n_ph"].numpy()
        for e in range(0, 40, 7):
            for i in range(0, cfg.n_sensors, 5):
                want = 0.1 * float(nph[e]) * _lrf_ref(cfg, i, pos[e, 0], pos[e, 1], pos[e, 2])
                assert abs(sig[e, i] - max(want, 0.0)) <= 2e-3 * max(abs(want), 1e-3), (idx, e, i)


@pytest.mark.parametrize("idx,method", [(6, 1), (7, 0), (8, 0), (6, 0)])
def test_one_iteration_equals_a_numpy_argmin(idx, method):
    """K = 1 of the search over an XY-type model against scores computed here from library LRF values."""
    cfg = synth.make_config(idx)
    cfg.method, cfg.n_iter = method, 1
    if idx == 7:
        cfg.nodes_per_axis = 3
    sig = synth.generate_events(cfg, 6)["signals"].numpy()
    m = oracle.Model.from_config(cfg)
    res = oracle.reconstruct(m, sig, oracle.grid_from_config(cfg), method, trace=True)
    G, half = cfg.nodes_per_axis, 0.5 * (cfg.nodes_per_axis - 1)
    Gz = G if cfg.dim == 3 else 1
    for e in range(len(sig)):
        S = sig[e].astype(np.float64)
        if method == 0:
            S = np.maximum(S, 0.0)
        g = cfg.gains.astype(np.float64)
        c = np.array([(cfg.sensor_xy[:, 0] * S / g).sum() / (S / g).sum(), (cfg.sensor_xy[:, 1] * S / g).sum() / (S / g).sum()])
        z0 = 10.0 if cfg.dim == 3 else 0.0
        scores = np.full(G * G * Gz, np.inf)
        for iz in range(Gz):
            for iy in range(G):
                for ix in range(G):
                    x, y = c[0] + (ix - half) * cfg.step0_xy, c[1] + (iy - half) * cfg.step0_xy
                    z = z0 + (iz - half) * cfg.step0_z if cfg.dim == 3 else 0.0
                    if cfg.dim == 3 and not (0.0 <= z <= 20.0):
                        continue
                    L = np.array([_lrf_ref(cfg, i, x, y, z) for i in range(cfg.n_sensors)])
                    if not L.sum() > 0:
                        continue
                    if method == 0:
                        mu = S.sum() / L.sum() * L
                        if np.any((L <= 0) & (S > 0)):
                            continue
                        with np.errstate(divide="ignore", invalid="ignore"):
                            t = np.where(S > 0, mu - S - S * np.log(mu / np.where(S > 0, S, 1.0)), mu)
                        scores[(iz * G + iy) * G + ix] = 2.0 * t.sum()
                    else:
                        w = 1.0 / np.maximum(S, 1.0)
                        A = (w * S * L).sum() / (w * L * L).sum()
                        scores[(iz * G + iy) * G + ix] = (w * (S - A * L) ** 2).sum()
        best = int(np.argmin(scores))
        assert res["idx"][e, 0] == best
        assert abs(res["best"][e, 0] - scores[best]) <= 1e-9 * abs(scores[best])


@pytest.mark.parametrize("idx", [6, 7, 8])
def test_noise_free_recovery_with_xy_type_lrfs(idx):
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, 60, noise_free=True)
    res = oracle.reconstruct(oracle.Model.from_config(cfg), ev["signals"].numpy(), oracle.grid_from_config(cfg), cfg.method)
    truth = ev["true_xyz"].numpy().astype(np.float64)
    inside = np.hypot(truth[:, 0], truth[:, 1]) <= 0.6 * cfg.extent
    h_xy, h_z = cfg.final_step()
    d = np.abs(res["xyzA"][:, :3] - truth)
    assert inside.sum() >= 10
    assert (d[inside, 0] <= h_xy * 1.01).all() and (d[inside, 1] <= h_xy * 1.01).all()
    if cfg.dim == 3:
        zin = inside & (truth[:, 2] > 1.0) & (truth[:, 2] < 19.0)
        assert (d[zin, 2] <= h_z * 1.01).all()
