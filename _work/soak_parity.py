"""Large-sample parity soak (needs a GPU; not collected by pytest): every config against the oracle on 1e4..3e5
events with the rules of tests/parity_rules.py.  Run from the repo root: python tests/soak_parity.py"""
import sys, os, time
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
import numpy as np, torch
import parity_rules
from paper_1602_07247_b200 import recon, synth
for idx, n in ((2, 300_000), (1, 10_000), (3, 40_000), (5, 25_000), (4, 20_000)):
    cfg = synth.make_config(idx)
    ev = synth.generate_events(cfg, n, device="cuda", batch=5)
    r = recon.Reconstructor(cfg)
    xyzA, score, path = r(ev["signals"], trace=True)
    torch.cuda.synchronize(); r.close()
    t0 = time.time()
    res = parity_rules.compare(cfg, ev["signals"].cpu().numpy(), xyzA.cpu().numpy(), score.cpu().numpy(), path.cpu().numpy())
    print(cfg.name, n, {k: v for k, v in res.items() if k in ("fail_mismatch", "score_viol", "score_max_rel", "A_viol", "pos_frac_within", "pos_max_steps", "idx_diverged", "idx_viol", "idx_max_gap", "idx_identical_frac")}, "oracle s %.1f" % (time.time() - t0), flush=True)
