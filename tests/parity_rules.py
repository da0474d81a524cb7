"""The north_star parity rules, GPU vs CPU oracle, made operational (SURVEY.md 8(c),
DESIGN.md "Parity rules").  Used by the -m gpu tests; imports the oracle (test
infrastructure) and takes the GPU results as plain numpy arrays.

 (i)   score:    |s_gpu - oracle.score_at(e, p_gpu)| <= 1e-5 |s_oracle_at_p_gpu|  (every event)
 (ii)  position: per axis |p_gpu - p_oracle| <= 1.01 h_K for >= 99.9 % of events
 (iii) index:    at the first iteration where the winning node differs, the oracle's
                 (second - best)/|best| must be <= 1e-4
 (iv)  energy:   |A_gpu - A_oracle_at_p_gpu| <= 1e-5 |A|                           (every event)
"""
from __future__ import annotations

import numpy as np

from oracle import oracle


def compare(cfg, signals: np.ndarray, gpu_xyzA: np.ndarray, gpu_score: np.ndarray,
            gpu_path: np.ndarray | None, threads: int = 0, score_floor: float = 0.0) -> dict:
    model = oracle.Model.from_config(cfg)
    grid = oracle.grid_from_config(cfg)
    ref = oracle.reconstruct(model, signals, grid, cfg.method, threads=threads, trace=True)
    E = signals.shape[0]
    gx = gpu_xyzA.astype(np.float64)
    ok_ref = np.isfinite(ref["xyzA"][:, 0])
    ok_gpu = np.isfinite(gx[:, 0])
    out = {"n_events": E, "fail_mismatch": int((ok_ref != ok_gpu).sum())}
    v = ok_ref & ok_gpu
    # (i) + (iv): oracle evaluated at the GPU's returned position
    A_at, s_at = oracle.score_at_many(model, signals, cfg.method, gx[:, :3], getattr(cfg, "seed_mode", 0))
    gs = gpu_score.astype(np.float64)
    both_inf = np.isinf(gs) & np.isinf(s_at)
    tol = 1e-5 * np.abs(s_at) + score_floor
    # the GPU rounds its FP64 score to float32 on output: half an ulp of slack
    tol = tol + np.abs(np.float32(s_at).astype(np.float64)) * 2.0 ** -24
    s_err = np.where(both_inf, 0.0, np.abs(gs - s_at))
    bad_s = v & ~(s_err <= tol)
    out["score_viol"] = int(bad_s.sum())
    with np.errstate(invalid="ignore", divide="ignore"):
        out["score_max_rel"] = float(np.nanmax(np.where(v & ~both_inf, s_err / np.abs(s_at), 0.0))) if v.any() else 0.0
        a_err = np.abs(gx[:, 3] - A_at) / np.abs(A_at)
    bad_a = v & np.isfinite(A_at) & ~(a_err <= 1e-5 + 2.0 ** -23)
    out["A_viol"] = int(bad_a.sum())
    out["A_max_rel"] = float(np.nanmax(np.where(v & np.isfinite(A_at), a_err, 0.0))) if v.any() else 0.0
    # (ii)
    h_xy, h_z = cfg.final_step()
    d = np.abs(gx[:, :3] - ref["xyzA"][:, :3])
    within = (d[:, 0] <= 1.01 * h_xy) & (d[:, 1] <= 1.01 * h_xy)
    if cfg.dim == 3:
        within &= d[:, 2] <= 1.01 * h_z
    out["pos_frac_within"] = float(within[v].mean()) if v.any() else 1.0
    out["pos_max_steps"] = float((d[v][:, :2].max() / h_xy)) if v.any() else 0.0
    out["pos_exact_frac"] = float(((d[:, 0] <= 0.01 * h_xy) & (d[:, 1] <= 0.01 * h_xy))[v].mean()) if v.any() else 1.0
    # (iii)
    if gpu_path is not None:
        gp = gpu_path.astype(np.int64) & 0xFFFF
        gp = np.where(gp == 0xFFFF, -1, gp)
        rp = ref["idx"].astype(np.int64)
        diff = gp != rp
        first = np.where(diff.any(axis=1), diff.argmax(axis=1), -1)
        rows = np.nonzero(v & (first >= 0))[0]
        k = first[rows]
        best, second = ref["best"][rows, k], ref["second"][rows, k]
        with np.errstate(invalid="ignore", divide="ignore"):
            gap = (second - best) / np.abs(best)
        viol = ~(gap <= 1e-4)
        out["idx_diverged"] = int(rows.size)
        out["idx_viol"] = int(viol.sum())
        out["idx_max_gap"] = float(gap[np.isfinite(gap)].max()) if np.isfinite(gap).any() else 0.0
        out["idx_viol_iters"] = np.bincount(k[viol], minlength=cfg.n_iter).tolist() if viol.any() else []
        out["idx_div_iters"] = np.bincount(k, minlength=cfg.n_iter).tolist()
        out["idx_identical_frac"] = float(1.0 - rows.size / max(int(v.sum()), 1))
    out["ref"] = ref
    return out


def assert_parity(res: dict, what: str = ""):
    msg = {k: v for k, v in res.items() if k != "ref"}
    assert res["fail_mismatch"] == 0, (what, msg)
    assert res["score_viol"] == 0, (what, msg)
    assert res["A_viol"] == 0, (what, msg)
    assert res["pos_frac_within"] >= 0.999, (what, msg)
    if "idx_viol" in res:
        assert res["idx_viol"] == 0, (what, msg)
