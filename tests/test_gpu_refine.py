"""GPU parity of the continuous refinement (ants_refine, R34) against the oracle's
Levenberg-Marquardt iteration.  Both sides run the same algorithm in double precision from the same float32 start
positions; they differ only in summation order, so positions agree to the float32 output rounding except where a
borderline accept/reject decision (gain ratio within rounding of 0) goes the other way -- those events must still
reach a score that is not worse than the oracle's by more than 1e-5 relative."""
import os
import sys

import numpy as np
import pytest
import torch

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from oracle import oracle                                      # noqa: E402
from paper_1602_07247_b200 import recon, synth                 # noqa: E402

pytestmark = pytest.mark.gpu


def _grid_then_refine(cfg, n, k_grid, n_steps, seed_mode=0):
    ev = synth.generate_events(cfg, n, device="cuda")
    coarse = synth.make_config(1)
    coarse.__dict__.update(cfg.__dict__)
    coarse.n_iter = k_grid
    r = recon.Reconstructor(coarse)
    try:
        xyzA, score = r(ev["signals"])
        start = xyzA.clone()
        recon.ants_refine(r.handle, ev["signals"], cfg.method, xyzA, score, n_steps, dim=cfg.dim, seed_mode=seed_mode)
        torch.cuda.synchronize()
    finally:
        r.close()
    sig = ev["signals"].cpu().numpy()
    m = oracle.Model.from_config(cfg)
    ref = oracle.refine(m, sig, cfg.method, start[:, :3].cpu().numpy().astype(np.float64), n_steps, dim=cfg.dim,
                        seed_mode=seed_mode)
    return sig, m, start.cpu().numpy(), xyzA.cpu().numpy(), score.cpu().numpy(), ref


def _check(cfg, sig, m, start, xyzA, score, ref, what):
    ok_ref, ok_gpu = np.isfinite(ref["xyzA"][:, 0]), np.isfinite(xyzA[:, 0])
    assert np.array_equal(ok_ref, ok_gpu), what
    v = ok_ref & np.isfinite(ref["score"])
    assert np.array_equal(np.isfinite(score), np.isfinite(ref["score"])), what
    # the GPU's score and energy are the oracle's definition at the GPU's own point
    A_at, s_at = oracle.score_at_many(m, sig, cfg.method, xyzA[:, :3].astype(np.float64), getattr(cfg, "seed_mode", 0))
    assert (np.abs(score[v] - s_at[v]) <= 1e-5 * np.abs(s_at[v]) + np.abs(np.float32(s_at[v])) * 2.0 ** -23).all(), what
    assert (np.abs(xyzA[v, 3] - A_at[v]) <= 1e-5 * np.abs(A_at[v])).all(), what
    # same iterates: positions agree to the float32 rounding of the output
    d = np.abs(xyzA[v, :3].astype(np.float64) - ref["xyzA"][v, :3])
    tol = 4e-6 + 2.0 ** -22 * np.abs(ref["xyzA"][v, :3])
    same = (d <= tol).all(axis=1)
    assert same.mean() >= 0.995, (what, same.mean(), d.max())
    # the rest took another branch at a borderline decision: still as good a point
    assert (score[v][~same] <= ref["score"][v][~same] * (1 + 1e-5) + 1e-6).all(), what
    # refinement never makes the score worse than the grid's
    s0 = oracle.score_at_many(m, sig, cfg.method, start[:, :3].astype(np.float64), getattr(cfg, "seed_mode", 0))[1]
    assert (score[v] <= s0[v] * (1 + 1e-6) + 1e-6).all(), what


@pytest.mark.parametrize("idx,n,method", [(1, 3001, 0), (2, 4001, 0), (3, 2001, 1), (3, 1501, 2), (4, 1501, 0), (5, 1001, 0),
                                          (6, 1501, 1), (7, 801, 0), (8, 2001, 0), (4, 801, 1)])
def test_refine_parity(idx, n, method):
    cfg = synth.make_config(idx)
    cfg.method = method
    out = _grid_then_refine(cfg, n, 5, 8)
    _check(cfg, *out, f"cfg{idx} method {method}")


def test_refine_with_selection_failed_events_and_zero_steps():
    cfg = synth.make_config(2)
    cfg.passive = np.zeros(cfg.n_sensors, np.uint8)
    cfg.passive[[4]] = 1
    cfg.signal_min, cfg.dist_max, cfg.seed_mode = 3.0, 75.0, 1
    out = _grid_then_refine(cfg, 2001, 5, 6, seed_mode=1)
    _check(cfg, *out, "selection + strongest start")
    # zero steps: the FP64 score and energy at the start point; NaN rows stay NaN
    cfg = synth.make_config(2)
    ev = synth.generate_events(cfg, 64, device="cuda")
    sig = ev["signals"].clone()
    sig[5, 3] = float("nan")
    r = recon.Reconstructor(cfg)
    xyzA, score = r(sig)
    before = xyzA.clone()
    recon.ants_refine(r.handle, sig, 0, xyzA, score, 0)
    torch.cuda.synchronize()
    r.close()
    assert torch.isnan(xyzA[5]).all() and torch.isinf(score[5])
    ok = torch.ones(64, dtype=torch.bool, device="cuda")
    ok[5] = False
    assert torch.equal(xyzA[ok, :3], before[ok, :3])
    assert torch.allclose(xyzA[ok, 3], before[ok, 3], rtol=1e-6)


def test_refine_status_codes():
    cfg = synth.make_config(2)
    r = recon.Reconstructor(cfg)
    sig = torch.ones((4, cfg.n_sensors), device="cuda")
    xyzA, score = torch.zeros((4, 4), device="cuda"), torch.zeros(4, device="cuda")
    with pytest.raises(recon.AntsError) as ei:
        recon.ants_refine(r.handle, sig, 0, xyzA, score, 4, dim=3)          # an axial LRF has no z
    assert ei.value.status == -1
    with pytest.raises(recon.AntsError):
        recon.ants_refine(r.handle, sig, 7, xyzA, score, 4)
    with pytest.raises(ValueError):
        recon.ants_refine(r.handle, sig, 0, xyzA[:2], score, 4)
    r.close()
