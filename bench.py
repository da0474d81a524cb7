#!/usr/bin/env python
"""bench.py -- events/s of the contracting-grid reconstruction on B200 (BASELINE.json metric).

One "step" = one pass of the whole hot path (load, centroid seed,
K grid iterations of LRF evaluation + energy + score + argmin, store) over one batch of seeded
synthetic flood-field events = ONE kernel launch through the C ABI (ants_reconstruct).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

The headline is config 5 (the largest single-GPU configuration: 127 PMTs, 16 M events in 8 batches of
2 M); `per_config` carries the same measurements for all five BASELINE.json configs (N = 1), each
with `cycle`: one reconstruct -> filter -> LRF-calculation cycle of the iterative response
reconstruction on one batch.
Prints ONE JSON line (rank 0).  `value` is device-resident throughput (CUDA events on the
launching stream, L2 flushed between steps, max over ranks); `e2e` is the same metric through
ants_reconstruct_host with pinned HOST buffers (H2D and D2H inside the timed region);
`roofline` is the FP32-ALU roofline of the one kernel; `cpu_baseline` is the double-precision
oracle (oracle/, test infrastructure) timed on this box's host cores on a bounded sample.
`--impl reference` times that oracle as the reference arm (there is no reference code: the
paper ships none).

Multi-GPU (torchrun, one process per GPU): events are independent and the path has no exchange
step, so every rank reconstructs its own seeded batch -- replicas, weak scaling, no collective
on the data path; only the timing is reduced (max over ranks).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/sec reconstructed on 1 B200; achieved % of FP32 peak"
UNIT = "events/s"

# nominal algorithmic flop per (node, sensor) pair:
# FMA = 2, sqrt / log / div = 1; every one of the K * G^d * N evaluations counts.
FLOP_PER_PAIR = {"axial_poisson": 20.0, "axial_chi2": 25.0, "axialz_poisson": 35.0}
# XY-type parameterisations (configs 6-8, outside BASELINE.json's five): local frame (6) +
# two interval/fraction look-ups (6) + two 4-weight cubic bases (2 x 11) + 4 x 4 tensor contraction (16 + 4 FMA = 40)
# = 74 per XY evaluation; a Sliced LRF contracts two planes (+ 40) and interpolates (3); a Composite adds the axial
# evaluation (15); the score terms add 5 (Poisson) or 10 (chi-square) as for the axial LRFs.
FLOP_XY = {3: 74.0, 4: 89.0, 5: 117.0}
FP32_LANES_PER_SM = 128          # B200 SM: 4 sub-partitions x 32 FP32 lanes, 1 FMA/lane/clk


def flop_per_pair(cfg) -> float:
    if cfg.lrf_dim >= 3:
        return FLOP_XY[cfg.lrf_dim] + (5.0 if cfg.method == 0 else 10.0)
    if cfg.lrf_dim == 2:
        return FLOP_PER_PAIR["axialz_poisson"]
    return FLOP_PER_PAIR["axial_chi2" if cfg.method == 1 else "axial_poisson"]


# ---------------------------------------------------------------------------
# clocks during the timed region (NVML; the recipe's clocks line)
# ---------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
               0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index: int, period: float = 0.05):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.period = period
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                try:
                    phys = int(vis.split(",")[index])
                except (ValueError, IndexError):
                    phys = index
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        while not self._stop.is_set():
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                mask = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if mask & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self) -> dict:
        med = statistics.median(self.samples) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ---------------------------------------------------------------------------
# helpers shared by the arms (host logic; covered by the gloo test)
# ---------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def rank_batch(rank: int, step: int, n_resident: int) -> int:
    """Which resident batch a rank reconstructs at a step (rotates so that inputs exceed L2)."""
    return (step + rank) % max(n_resident, 1)


def rank_seed_batch(rank: int, j: int, n_resident: int) -> int:
    """Sub-stream id of resident batch j on a rank: ranks never share events (replicas of the
    path, distinct data)."""
    return rank * n_resident + j


def max_over_ranks(local_ms: float, dist, device) -> float:
    """Timing reduction: the slowest rank defines the job's time."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(local_ms)
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(v: float, dist, device) -> float:
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(v)
    t = torch.tensor([v], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def oracle_rate(cfg, signals_np, budget_s: float, threads: int = 0):
    """Time the oracle, as it stands, on a bounded sample: calibrate on a small slice, then run
    as many of the leading events as fit in ~budget_s.  Returns (events/s, n_events, threads)."""
    from oracle import oracle
    model = oracle.Model.from_config(cfg)
    grid = oracle.grid_from_config(cfg)
    used = oracle.n_threads(threads)
    n0 = min(len(signals_np), max(64, 8 * used))
    t0 = time.perf_counter()
    oracle.reconstruct(model, signals_np[:n0], grid, cfg.method, threads=threads)
    t1 = time.perf_counter() - t0
    n = int(min(len(signals_np), max(n0, n0 * budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    oracle.reconstruct(model, signals_np[:n], grid, cfg.method, threads=threads)
    dt = time.perf_counter() - t0
    return n / dt, n, used


# ---------------------------------------------------------------------------
# reference arm = the oracle on host cores (rank 0 only)
# ---------------------------------------------------------------------------
def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from paper_1602_07247_b200 import synth
    cfg = synth.make_config(args.config)
    from oracle import oracle
    model = oracle.Model.from_config(cfg)
    grid = oracle.grid_from_config(cfg)
    used = oracle.n_threads(0)
    # bounded sample per step: sized from a calibration slice so that one step takes ~step_s
    n_pool = 262_144 if cfg.pairs_per_event < 50_000 else 32_768       # a step never needs more (oracle: ~1e4 events/s)
    pool = synth.generate_events(cfg, min(cfg.n_events // cfg.n_batches, n_pool), device="cpu")["signals"].numpy()
    n0 = max(64, 8 * used)
    t0 = time.perf_counter()
    oracle.reconstruct(model, pool[:n0], grid, cfg.method)
    per_ev = (time.perf_counter() - t0) / n0
    n = int(max(n0, min(len(pool), args.ref_step_seconds / per_ev)))
    for _ in range(args.warmup):
        oracle.reconstruct(model, pool[:n], grid, cfg.method)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.reconstruct(model, pool[:n], grid, cfg.method)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = f"first {n} events of the seeded {cfg.name} flood field per step, {args.steps} steps"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(cfg, n, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(cfg, events_per_step: int, n_gpus: int) -> dict:
    return {"workload": cfg.name, "events_per_step_per_gpu": int(events_per_step), "n_sensors": cfg.n_sensors,
            "grid": "x".join([str(cfg.nodes_per_axis)] * cfg.dim), "n_iter": cfg.n_iter,
            "method": "poisson_ml" if cfg.method == 0 else "chi_square",
            "pairs_per_event": cfg.pairs_per_event, "parallelism": f"replicas x{n_gpus} (no collective)",
            "events_total": int(cfg.n_events), "batches": int(cfg.n_batches),
            "l2": "256 MiB scratch write between timed steps; resident batches rotate"}


# ---------------------------------------------------------------------------
# instruction mix and DRAM traffic per kernel: read from the committed ncu summary (never hard-coded here)
# ---------------------------------------------------------------------------
MIX_CSV = os.path.join(ROOT, "profiles", "r02_kernel_mix.csv")


def kernel_mix(workload: str, kernel: str):
    """Row of profiles/r02_kernel_mix.csv (made from `ncu --set full --import-source on` captures of this very
    bench command, see profiles/r02_kernel_mix.md) for this workload, if it describes the kernel that is
    dispatched now; else None -- a stale row is dropped, not reported."""
    try:
        import csv
        with open(MIX_CSV, newline="") as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["kernel"] == kernel:
                    return row
    except OSError:
        pass
    return None


def fp32_peak_tflops(prop, max_mhz: float) -> float:
    return prop.multi_processor_count * FP32_LANES_PER_SM * 2 * max_mhz * 1e6 / 1e12


def roofline_of(cfg, plan: dict, E: int, launch_ms: float, prop, max_mhz: float) -> dict:
    """FP32-ALU roofline of the one kernel.  `frac` is nominal: SURVEY.md 8(d)'s flop per
    (node, sensor) pair x ALL K G^d N pairs of the method (the kernels skip pairs whose LRF is constant over the
    grid; no credit is taken for that) / launch time / peak.  `frac_executed`, `mix_ceiling` and `traffic` come
    from the committed ncu capture of the same kernel, labelled with their source."""
    peak = fp32_peak_tflops(prop, max_mhz)
    pairs = float(cfg.pairs_per_event) * E
    t = launch_ms * 1e-3
    achieved = flop_per_pair(cfg) * pairs / t / 1e12
    alg_bytes = E * (4 * cfg.n_sensors + 20)
    out = {"bound": "alu", "kernel": plan.get("kernel"), "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
           "frac": achieved / peak, "frac_kind": "nominal flop/pair x all K*G^d*N pairs",
           "peak_source": "derived: SMs x 128 FP32 lanes x 2 x clocks.max.sm (MEASURED_PEAKS.json has no FP32 "
                          "entry); cross-checked by profiles/r02_fp32_peak.md",
           "flop_per_pair_nominal": flop_per_pair(cfg), "pairs_per_s": pairs / t,
           "algorithmic_bytes_per_launch": alg_bytes, "hbm_gbs_signal_stream": alg_bytes / t / 1e9,
           "launch_ms": launch_ms, "traffic": None, "frac_executed": None, "mix_ceiling": None}
    row = kernel_mix(cfg.name, plan.get("kernel") or "")
    if row is not None:
        out["traffic"] = float(row["dram_bytes_per_event"]) * E
        out["frac_executed"] = float(row["flop_executed_per_pair"]) * pairs / t / 1e12 / peak
        out["mix_ceiling"] = float(row["mix_ceiling_frac"])
        out["thread_inst_per_pair"] = float(row["thread_inst_per_pair"])
        out["mix_source"] = "profiles/r02_kernel_mix.csv (ncu capture of this kernel; see profiles/r02_kernel_mix.md)"
    return out


# ---------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------
def measure_config(idx: int, args, device, rank: int, world: int, dist, steps: int, warmup: int,
                   cpu_seconds: float) -> dict:
    """Device-resident throughput, end-to-end throughput, roofline and oracle baseline of one BASELINE.json config.
    A step = one launch of ants_reconstruct over one batch (config 5: one of its eight 2 M-event batches)."""
    import torch
    from paper_1602_07247_b200 import recon, synth
    cfg = synth.make_config(idx)
    # variants of a config for kernel studies (profiles/r02_lockstep.md): another grid size or scoring method on the
    # same detector and events; the workload name says so, and such a line is not a BASELINE.json config
    if getattr(args, "grid_nodes", None) or getattr(args, "method", None) is not None:
        import dataclasses
        G = args.grid_nodes or cfg.nodes_per_axis
        meth = cfg.method if args.method is None else args.method
        cfg = dataclasses.replace(cfg, nodes_per_axis=G, method=meth, name=f"{cfg.name}+G{G}m{meth}")
    E = cfg.n_events // cfg.n_batches if args.events is None else args.events
    n_resident = max(2, cfg.n_batches) if args.resident is None else args.resident
    r = recon.Reconstructor(cfg)
    sigs = [synth.generate_events(cfg, E, device=device, batch=rank_seed_batch(rank, j, n_resident))["signals"]
            for j in range(n_resident)]
    xyzA = torch.empty((E, 4), dtype=torch.float32, device=device)
    score = torch.empty((E,), dtype=torch.float32, device=device)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)
    stream = torch.cuda.current_stream()

    def one(step):
        recon.ants_reconstruct(r.handle, sigs[rank_batch(rank, step, n_resident)], r.grid, r.method, xyzA, score,
                               stream.cuda_stream)

    for s in range(warmup):
        one(s)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    launches0 = recon.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    sampler = ClockSampler(device.index or 0)
    torch.cuda.synchronize()
    with sampler:
        for s in range(steps):
            flush.fill_(s & 0xFF)                 # evict L2 (126 MB) between timed steps
            ev[s][0].record(stream)
            one(warmup + s)
            ev[s][1].record(stream)
        torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    gpu_launches = recon.launch_count() - launches0
    local_ms = sum(step_ms)
    total_ms = max_over_ranks(local_ms, dist, device)
    total_events = sum_over_ranks(float(E * steps), dist, device)
    out = {"config": workload_config(cfg, E, world), "value": total_events / (total_ms * 1e-3), "unit": UNIT,
           "steps": steps, "warmup": warmup, "ms_per_step": total_ms / steps, "step_ms": step_ms,
           "gpu_launches": int(gpu_launches), "clocks": sampler.summary()}
    del flush

    # ---- latency of one call (launch-bound workloads: config 1) ------------------------------------
    if E <= 100_000:
        n_calls = 200
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for s in range(n_calls):
            one(s)
        t_issue = time.perf_counter() - t0
        torch.cuda.synchronize()
        t_all = time.perf_counter() - t0
        out["us_per_call"] = {"host_issue": 1e6 * t_issue / n_calls, "back_to_back": 1e6 * t_all / n_calls,
                              "device_kernel": 1e3 * statistics.median(step_ms), "calls": n_calls}

    # ---- end to end: pinned host buffers through ants_reconstruct_host -------------------------------
    # config 5: the whole 16 M-event job as BASELINE.json states it (8 streamed batches of 2 M); others: one batch
    n_e2e_batches = cfg.n_batches if args.events is None else 1
    E2 = E * n_e2e_batches
    sig_h = torch.empty((E2, cfg.n_sensors), dtype=torch.float32).pin_memory()
    for j in range(n_e2e_batches):
        sig_h[j * E:(j + 1) * E].copy_(sigs[j])
    xyzA_h = torch.empty((E2, 4), dtype=torch.float32).pin_memory()
    score_h = torch.empty((E2,), dtype=torch.float32).pin_memory()
    chunk = E if n_e2e_batches > 1 else max(1, min(E, args.e2e_chunk))
    torch.cuda.synchronize()
    recon.ants_reconstruct_host(r.handle, sig_h, r.grid, r.method, xyzA_h, score_h, chunk)     # allocates the ring
    if dist is not None:
        dist.barrier()
    e2e_steps = 1 if n_e2e_batches > 1 else max(1, min(steps, 5))
    l0 = recon.launch_count()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        recon.ants_reconstruct_host(r.handle, sig_h, r.grid, r.method, xyzA_h, score_h, chunk)
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_launches = recon.launch_count() - l0
    e2e_ms = max_over_ranks(e2e_ms, dist, device)
    e2e_value = sum_over_ranks(float(E2 * e2e_steps), dist, device) / (e2e_ms * 1e-3)
    assert torch.equal(xyzA_h[:1024].to(device), r(sigs[0][:1024].contiguous())[0])   # same kernel, same bits
    out["e2e"] = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": E2 * cfg.n_sensors * 4,
                  "d2h_bytes_per_step": E2 * 20, "steps": e2e_steps, "events_per_step": E2, "chunk_events": chunk,
                  "ms_per_step": e2e_ms / e2e_steps, "gpu_launches": int(e2e_launches),
                  "api": "ants_reconstruct_host (pinned host buffers, 3-stream ring)"}

    # ---- roofline of the one kernel --------------------------------------------------------------------
    prop = torch.cuda.get_device_properties(device)
    max_mhz = out["clocks"]["sm_max_mhz"] or 1965.0
    out["plan"] = r.plan()
    out["roofline"] = roofline_of(cfg, out["plan"], E, local_ms / max(gpu_launches, 1), prop, max_mhz)

    # ---- one reconstruct -> filter -> LRF-calculation cycle on the first resident batch (N = 1) ----------------
    if world == 1 and not args.no_cycle:
        try:
            res = time_cycle(recon, cfg, r, sigs[0], xyzA, score, stream, 3, 1)
            t_c = sum(res["ms"]) / len(res["ms"])
            out["cycle"] = {"value": E / (t_c * 1e-3), "unit": "events/s through one reconstruct -> filter -> LRF calculation",
                            "ms_per_cycle": t_c, "lrf_calculation_ms": sum(res["fit_ms"]) / len(res["fit_ms"]),
                            "events_passing_filter": res["n_pass"], "gpu_launches": res["gpu_launches"]}
        except recon.AntsError as ex:      # e.g. a table the batch does not cover
            out["cycle"] = {"unavailable": str(ex)}

    # ---- oracle beside it (rank 0, N = 1) --------------------------------------------------------------
    if rank == 0 and world == 1 and not args.no_cpu_baseline and cpu_seconds > 0:
        n_pool = min(E, 262_144)
        rate, n, used = oracle_rate(cfg, sig_h[:n_pool].numpy(), cpu_seconds)
        out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": used, "kind": "oracle",
                               "sample": f"first {n} events of the same {cfg.name} batch, one pass, "
                                         f"double precision, OpenMP over events"}
    r.close()
    del sigs, sig_h, xyzA_h, score_h, xyzA, score
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    from paper_1602_07247_b200 import recon
    recon.load()

    head = measure_config(args.config, args, device, rank, world, dist, args.steps, args.warmup, args.cpu_seconds)
    line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": head["config"], "clocks": head["clocks"], "e2e": head["e2e"],
            "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "step_ms": head["step_ms"],
            "plan": head["plan"]}
    if "cpu_baseline" in head:
        line["cpu_baseline"] = head["cpu_baseline"]
    for k in ("us_per_call", "cycle"):
        if k in head:
            line[k] = head[k]

    # ---- every BASELINE.json config beside the headline (N = 1 only: north_star asks for all five) -----
    if world == 1 and not args.no_per_config and args.events is None and not args.grid_nodes and args.method is None:
        per = []
        for idx in (1, 2, 3, 4, 5):
            m = head if idx == args.config else measure_config(
                idx, args, device, rank, world, dist, min(args.steps, 20), args.warmup, args.per_config_cpu_seconds)
            entry = {k: m[k] for k in ("value", "unit", "ms_per_step", "steps", "warmup", "gpu_launches", "roofline",
                                        "e2e", "plan", "clocks", "config") if k in m}
            entry["config_index"] = idx
            for k in ("cpu_baseline", "us_per_call", "cycle"):
                if k in m:
                    entry[k] = m[k]
            per.append(entry)
        line["per_config"] = per
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_peak(args):
    """FP32 / MUFU / FP64 issue-rate probes behind the derived peak (`--workload peak`): ants_probe_throughput."""
    import torch
    from paper_1602_07247_b200 import recon
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    prop = torch.cuda.get_device_properties(0)
    sampler = ClockSampler(0)
    kinds = {0: "ffma", 1: "ffma2_packed", 2: "mufu_lg2", 3: "dfma", 4: "ffma_3_distinct_regs"}
    res = {}
    with sampler:
        for kind, name in kinds.items():
            best = 0.0
            for _ in range(max(args.steps, 3)):
                ops, ms = recon.ants_probe_throughput(kind, 8192)
                best = max(best, ops)
            res[name] = best
    clocks = sampler.summary()
    mhz = clocks["sm_max_mhz"] or 1965.0
    cyc = prop.multi_processor_count * mhz * 1e6
    line = {"metric": "dependent-free instruction throughput (ants_probe_throughput)", "unit": "lane-ops/s",
            "n_gpus": 1, "sms": prop.multi_processor_count, "clocks": clocks,
            "lane_ops_per_s": res, "lane_ops_per_clk_per_sm": {k: v / cyc for k, v in res.items()},
            "fp32_tflops_ffma": 2 * res["ffma"] / 1e12, "fp32_tflops_ffma2": 2 * res["ffma2_packed"] / 1e12,
            "fp64_tflops_dfma": 2 * res["dfma"] / 1e12,
            "fp32_peak_derived_tflops": fp32_peak_tflops(prop, mhz)}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------
# secondary workload: the LRF calculation (ants_lrf_fit_axial), `--workload fit`
# ---------------------------------------------------------------------------
def run_fit(args):
    import numpy as np
    """Times ants_lrf_fit_axial (normal equations on the GPU + host solve) on the config's batch with the
    positions reconstructed by the library.  HBM roofline: the call must read the signals (4N B) and the
    positions (16 B) of every event once; peak = MEASURED_PEAKS.json hbm_gbs (fallback 6650, said so)."""
    import torch
    from paper_1602_07247_b200 import recon, synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    device = torch.device("cuda", 0)
    cfg = synth.make_config(args.config)
    E = cfg.n_events // cfg.n_batches if args.events is None else args.events
    sig = synth.generate_events(cfg, E, device=device)["signals"]
    r = recon.Reconstructor(cfg)
    xyzA, _ = r(sig)
    r.close()
    if cfg.n_lrf > 1:       # per-sensor tables need data over the whole r-range of every sensor: use all of it they see
        knots = cfg.knots.copy()
        knots[1] = min(float(knots[1]), 30.0)
    else:
        knots = cfg.knots
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()
    def call():
        if cfg.lrf_dim == 2:
            c, u = recon.ants_lrf_fit_axial_z(cfg.sensor_xy, cfg.gains, knots, cfg.n_int_r, cfg.n_int_z, sig, xyzA)
            return c, np.array([u])
        return recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, knots, cfg.n_lrf, cfg.n_int_r, sig, xyzA)

    for _ in range(args.warmup):
        call()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    n1 = recon.launch_count()
    for a, b in ev:
        a.record(stream)
        coeffs, used = call()
        b.record(stream)
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in ev]
    t = sum(ms) / len(ms) * 1e-3
    peak, src = 6650.0, "fallback"
    try:
        peak, src = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured"
    except Exception:
        pass
    bytes_alg = E * (4 * cfg.n_sensors + 16)
    line = {"metric": "events/s whose signals enter one LRF calculation (ants_lrf_fit_axial)", "value": E / t,
            "unit": "events/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name + " LRF calculation", "events_per_step_per_gpu": E, "n_sensors": cfg.n_sensors,
                       "n_lrf": cfg.n_lrf, "n_int_r": cfg.n_int_r, "pairs_used": float(used.sum())},
            "gpu_launches": recon.launch_count() - n1,
            "roofline": {"bound": "hbm", "achieved": bytes_alg / t / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": bytes_alg / t / 1e9 / peak, "traffic": None, "peak_source": src + " hbm_gbs",
                         "pairs_per_s": float(used.sum()) / t, "smem_fp64_atomics_per_s": (152.0 if cfg.lrf_dim == 2 else 14.0) * float(used.sum()) / t},
            "step_ms": ms}
    print(json.dumps(line), flush=True)
    return 0


def lrf_calculation(recon, cfg, sig, xyzA):
    """The LRF calculation that belongs to the config's parameterisation, as iterate.py calls it;
    per-sensor axial tables are fitted up to 30 mm (a flood batch does not cover every sensor's far intervals)."""
    knots = cfg.knots.copy()
    if cfg.n_lrf > 1 and cfg.lrf_dim == 1:
        knots[1] = min(float(knots[1]), 30.0)
    group, xform = getattr(cfg, "group", None), getattr(cfg, "xform", None)
    if cfg.lrf_dim == 2:
        return recon.ants_lrf_fit_axial_z(cfg.sensor_xy, cfg.gains, knots, cfg.n_int_r, cfg.n_int_z, sig, xyzA)
    if cfg.lrf_dim == 5:
        return recon.ants_lrf_fit_sliced(cfg.sensor_xy, cfg.gains, cfg.knots_xy, cfg.n_lrf, cfg.n_int_x, cfg.n_int_y,
                                         cfg.n_planes, sig, xyzA, group=group, xform=xform)
    axial = None
    if cfg.lrf_dim in (1, 4):
        ca, used = recon.ants_lrf_fit_axial(cfg.sensor_xy, cfg.gains, knots, cfg.n_lrf, cfg.n_int_r, sig, xyzA, group=group)
        if cfg.lrf_dim == 1:
            return ca, used
        axial = (knots, ca)
    return recon.ants_lrf_fit_xy(cfg.sensor_xy, cfg.gains, cfg.knots_xy, cfg.n_lrf, cfg.n_int_x, cfg.n_int_y, sig, xyzA,
                                 group=group, xform=xform, axial=axial)


def time_cycle(recon, cfg, r, sig, xyzA, score, stream, steps, warmup):
    """One cycle of the iterative response reconstruction: reconstruct the batch, filter on the score,
    recalculate the LRFs; CUDA events on the launching stream around the cycle and around its LRF calculation."""
    import torch

    def cycle(ev=None):
        recon.ants_reconstruct(r.handle, sig, r.grid, r.method, xyzA, score, stream.cuda_stream)
        n_pass = recon.ants_filter_events(xyzA, score, score_max=4.0 * cfg.n_sensors)
        if ev:
            ev[0].record(stream)
        lrf_calculation(recon, cfg, sig, xyzA)
        if ev:
            ev[1].record(stream)
        return n_pass

    for _ in range(warmup):
        cycle()
    n0 = recon.launch_count()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    for a, f0, f1, b in ev:
        a.record(stream)
        n_pass = cycle((f0, f1))
        b.record(stream)
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, _, _, b in ev]
    fit_ms = [f0.elapsed_time(f1) for _, f0, f1, _ in ev]
    return {"ms": ms, "fit_ms": fit_ms, "n_pass": int(n_pass), "gpu_launches": int(recon.launch_count() - n0)}


def run_cycle(args):
    """Times one cycle of the iterative response reconstruction: reconstruct the batch,
    filter on the score, recalculate the LRFs.  Secondary workload (`--workload cycle`)."""
    import torch
    from paper_1602_07247_b200 import recon, synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    device = torch.device("cuda", 0)
    cfg = synth.make_config(args.config)
    E = cfg.n_events // cfg.n_batches if args.events is None else args.events
    sig = synth.generate_events(cfg, E, device=device)["signals"]
    r = recon.Reconstructor(cfg)
    xyzA = torch.empty((E, 4), dtype=torch.float32, device=device)
    score = torch.empty((E,), dtype=torch.float32, device=device)
    res = time_cycle(recon, cfg, r, sig, xyzA, score, torch.cuda.current_stream(), args.steps, args.warmup)
    ms, n_pass = res["ms"], res["n_pass"]
    t = sum(ms) / len(ms) * 1e-3
    r.close()
    print(json.dumps({"metric": "events/s through one reconstruct -> filter -> LRF-calculation cycle", "value": E / t,
                      "unit": "events/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32+f64",
                      "data": "synthetic", "config": {"workload": cfg.name + " response-reconstruction cycle",
                                                      "events_per_step_per_gpu": E, "events_passing_filter": n_pass},
                      "gpu_launches": res["gpu_launches"], "step_ms": ms, "lrf_calculation_ms": res["fit_ms"]}), flush=True)
    return 0


def run_refine(args):
    """Times `--grid-iters` contracting-grid iterations followed by `--refine-steps` Levenberg-Marquardt steps
    (ants_refine, the role Minuit2 plays in PAPER.md:320-324) against the config's full grid search, on the same
    batch.  Secondary workload (`--workload refine`)."""
    import copy
    import torch
    from paper_1602_07247_b200 import recon, synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    device = torch.device("cuda", 0)
    cfg = synth.make_config(args.config)
    E = cfg.n_events // cfg.n_batches if args.events is None else args.events
    sig = synth.generate_events(cfg, E, device=device)["signals"]
    short = copy.copy(cfg)
    short.n_iter = args.grid_iters
    r_full, r_short = recon.Reconstructor(cfg), recon.Reconstructor(short)
    xyzA = torch.empty((E, 4), dtype=torch.float32, device=device)
    score = torch.empty((E,), dtype=torch.float32, device=device)
    stream = torch.cuda.current_stream()

    def full():
        recon.ants_reconstruct(r_full.handle, sig, r_full.grid, r_full.method, xyzA, score, stream.cuda_stream)

    def hybrid():
        recon.ants_reconstruct(r_short.handle, sig, r_short.grid, r_short.method, xyzA, score, stream.cuda_stream)
        recon.ants_refine(r_short.handle, sig, cfg.method, xyzA, score, args.refine_steps, dim=cfg.dim)

    out = {}
    for name, fn in (("grid_only", full), ("grid_then_refine", hybrid)):
        for _ in range(args.warmup):
            fn()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        n0 = recon.launch_count()
        for a, b in ev:
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        ms = [a.elapsed_time(b) for a, b in ev]
        t = sum(ms) / len(ms) * 1e-3
        ok = torch.isfinite(score)
        out[name] = {"events_per_s": E / t, "ms_per_step": t * 1e3, "gpu_launches": recon.launch_count() - n0,
                     "mean_score": float(score[ok].double().mean())}
    r_full.close()
    r_short.close()
    print(json.dumps({"metric": "events/s: contracting grid alone vs a shorter grid followed by continuous refinement",
                      "value": out["grid_then_refine"]["events_per_s"], "unit": "events/s", "n_gpus": 1,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": out["grid_then_refine"]["ms_per_step"],
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32 grid + f64 refinement",
                      "data": "synthetic",
                      "config": {"workload": cfg.name + " grid + refinement", "events_per_step_per_gpu": E,
                                 "grid_iters": args.grid_iters, "refine_steps": args.refine_steps,
                                 "grid_iters_of_the_config": cfg.n_iter},
                      "results": out, "speedup_vs_grid_only": out["grid_then_refine"]["events_per_s"] / out["grid_only"]["events_per_s"]}),
          flush=True)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json config 1..5 of the headline (default 5 = the largest single-GPU config: "
                         "16 M events as 8 batches of 2 M); 6, 7, 8 = the XY / Sliced / Composite LRF workloads")
    ap.add_argument("--no-cycle", action="store_true", help="skip the response-reconstruction cycle entries")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config entries of the other configs")
    ap.add_argument("--per-config-cpu-seconds", type=float, default=5.0)
    ap.add_argument("--events", type=int, default=None, help="events per step per GPU (default: the config's batch)")
    ap.add_argument("--grid-nodes", type=int, default=None, help="kernel studies: nodes per axis instead of the config's")
    ap.add_argument("--method", type=int, default=None, choices=[0, 1, 2],
                    help="kernel studies: scoring method instead of the config's (0 Poisson ML, 1 chi-square, 2 sum-ratio LS)")
    ap.add_argument("--resident", type=int, default=None, help="distinct resident batches to rotate through")
    ap.add_argument("--e2e-chunk", type=int, default=1 << 18)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--ref-step-seconds", type=float, default=4.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--grid-iters", type=int, default=5, help="--workload refine: grid iterations before the refinement")
    ap.add_argument("--refine-steps", type=int, default=6, help="--workload refine: Levenberg-Marquardt steps")
    ap.add_argument("--workload", default="reconstruct", choices=["reconstruct", "fit", "cycle", "peak", "refine"],
                    help="fit = time the LRF calculation instead (secondary; not the BASELINE metric)")
    args = ap.parse_args(argv)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = max(args.warmup, 1)
    if args.workload == "fit":
        return run_fit(args)
    if args.workload == "cycle":
        return run_cycle(args)
    if args.workload == "peak":
        return run_peak(args)
    if args.workload == "refine":
        return run_refine(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
