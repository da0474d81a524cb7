"""Large-sample parity soak: every workload (BASELINE.json configs 1-5 and the XY / Sliced / Composite workloads 6-8)
against the oracle on 4e3 ... 2e5 seeded events (sub-stream 5, not the one the other tests use) under the north_star
rules of tests/parity_rules.py.  `python -m pytest tests/test_gpu_soak.py -s -q` prints one summary row per
workload (profiles/r02_parity_soak.md is that output)."""
import os
import sys

import pytest
import torch

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import parity_rules                                            # noqa: E402
from paper_1602_07247_b200 import recon, synth                 # noqa: E402

pytestmark = pytest.mark.gpu

KEYS = ("fail_mismatch", "score_viol", "score_max_rel", "A_viol", "pos_frac_within", "pos_max_steps", "idx_diverged",
        "idx_viol", "idx_max_gap", "idx_identical_frac")


@pytest.mark.parametrize("idx,n", [(1, 10_000), (2, 200_000), (3, 40_000), (4, 20_000), (5, 25_000), (6, 20_000),
                                   (7, 4_000), (8, 50_000)])
def test_soak(idx, n):
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, n, device="cuda", batch=5)
    r = recon.Reconstructor(cfg)
    try:
        kernel = r.plan()["kernel"]
        xyzA, score, path = r(ev["signals"], trace=True)
        torch.cuda.synchronize()
    finally:
        r.close()
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA.cpu().numpy(), score.cpu().numpy(), path.cpu().numpy())
    print("\nSOAK", cfg.name, n, kernel, {k: res[k] for k in KEYS}, flush=True)
    parity_rules.assert_parity(res, f"soak {cfg.name}")
    assert res["idx_max_gap"] <= 1e-4
