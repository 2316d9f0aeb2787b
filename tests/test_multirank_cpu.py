"""The N > 1 path of bench.py on CPU: world_size 2 over gloo.  The hot path itself does not shard
("replicas only"), so what N > 1 adds is the reduction of the per-rank device
times (max over ranks) and the whole-job aggregate; both are exercised here with two processes."""
import os

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times = [10.0 + rank, 30.0 - 5 * rank]            # rank 1 is slower on the first, rank 0 on the second
    red = bench.max_over_ranks(times, torch.device("cpu"), world)
    dist.barrier()
    if rank == 0:
        out.put(red)
    dist.destroy_process_group()


def test_max_over_ranks_two_processes():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    red = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert red == [11.0, 30.0]


def test_single_rank_is_identity_and_aggregate_scales_with_replicas():
    assert bench.max_over_ranks([1.5, 2.5], torch.device("cpu"), 1) == [1.5, 2.5]
    one = bench.whole_job_value(1, 5.5e12, 4.4)
    assert abs(one - 1250.0) < 1e-9
    assert bench.whole_job_value(8, 5.5e12, 4.4) == 8 * one      # weak scaling: same time, 8x the work


def test_ulysses_plan_is_deterministic_and_balances():
    # bench.py --mode ulysses: every rank derives the same head order from the same costs (no exchange needed),
    # and the greedy schedule never makes the max / mean load worse than the index order
    import numpy as np
    cost = [int(c) for c in np.random.default_rng(77).uniform(0.10, 0.40, 40) * 131072]
    for ranks in (1, 2, 4, 8):
        order, plan = bench.ulysses_plan(cost, ranks)
        assert sorted(order) == list(range(40))
        assert bench.ulysses_plan(cost, ranks)[0] == order
        assert plan["imbalance_max_over_avg_after"] <= plan["imbalance_max_over_avg_before"] + 1e-12
        assert plan["imbalance_max_over_avg_after"] >= 1.0 - 1e-12
    assert bench.ulysses_plan(cost, 1)[0] == list(range(40))          # one rank: a no-op (Table 4)
    assert bench.ulysses_plan(cost, 8)[1]["imbalance_max_over_avg_after"] < 1.06


def test_reference_arm_prints_the_contract_line():
    # bench.py --impl reference: the oracle on the host cores, one JSON line with the base contract's keys
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--workload", "cfg1"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
              "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in line, k
    assert line["impl"] == "reference" and line["dtype"] == "f64" and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
