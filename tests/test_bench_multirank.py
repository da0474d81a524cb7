"""N > 1 host logic of bench.py on CPU: two gloo ranks (world_size 2, 127.0.0.1).

The path has no exchange step (events are independent): ranks are replicas
with distinct seeded batches, and only the timing is reduced.  This covers that bookkeeping: distinct
sub-streams per rank, max-over-ranks time, summed event count, rank 0 alone printing, and the reference
arm running on rank 0 only."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import torch, torch.distributed as dist
    import bench
    rank, local, world = bench.dist_env()
    dist.init_process_group("gloo")
    dev = torch.device("cpu")
    local_ms = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    total_ms = bench.max_over_ranks(local_ms, dist, dev)
    events = bench.sum_over_ranks(1000.0 * (rank + 1), dist, dev)
    seeds = [bench.rank_seed_batch(rank, j, 3) for j in range(3)]
    order = [bench.rank_batch(rank, s, 3) for s in range(6)]
    gathered = [None] * world
    dist.all_gather_object(gathered, seeds)
    if rank == 0:
        print(json.dumps({"total_ms": total_ms, "events": events, "seeds": gathered, "order": order}))
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def _launch(code_or_args, env_extra=None, world=2):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        env.update(env_extra or {})
        procs.append(subprocess.Popen([sys.executable] + code_or_args, env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    return outs


def test_two_rank_timing_and_sharding_bookkeeping():
    outs = _launch(["-c", WORKER])
    assert outs[1][0].strip() == ""                                   # only rank 0 prints
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["total_ms"] == 15.0                                    # max over ranks
    assert res["events"] == 3000.0                                    # whole-job aggregate
    flat = [s for per_rank in res["seeds"] for s in per_rank]
    assert len(set(flat)) == len(flat) == 6                           # ranks never share a sub-stream
    assert sorted(set(res["order"])) == [0, 1, 2]                     # resident batches rotate


def test_reference_arm_runs_on_rank_zero_only():
    outs = _launch(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1",
                    "--config", "1", "--ref-step-seconds", "0.3"])
    assert outs[1][0].strip() == ""
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
