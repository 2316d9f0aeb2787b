"""Head-level scheduling (appendix A): oracle pins, the library's host function against
the oracle (no GPU needed: it is host code), and a world_size-2 gloo run of the partition."""
import heapq
import itertools
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2606_25040_b200 import binding as B


def unconstrained_lpt(cost, n_ranks):
    """Textbook LPT with a heap (no capacity), an independent routine."""
    heap = [(0, r) for r in range(n_ranks)]
    for c in sorted(cost, reverse=True):
        l, r = heapq.heappop(heap)
        heapq.heappush(heap, (l + c, r))
    return sorted(l for l, _ in heap)


def brute_force_best_makespan(cost, n_ranks, cap):
    best = None
    for assign in itertools.product(range(n_ranks), repeat=len(cost)):
        if max(np.bincount(assign, minlength=n_ranks)) > cap:
            continue
        m = max(sum(c for c, a in zip(cost, assign) if a == r) for r in range(n_ranks))
        best = m if best is None else min(best, m)
    return best


def test_oracle_partition_is_valid_and_balanced():
    g = np.random.default_rng(0)
    for H, G in ((40, 8), (40, 4), (40, 2), (40, 1), (7, 3), (5, 8)):
        cost = g.integers(100, 60000, H)
        mine, load = oracle.schedule_heads(cost, G)
        cap = -(-H // G)
        assert sorted(h for m in mine for h in m) == list(range(H))          # every head exactly once
        assert all(len(m) <= cap for m in mine)
        assert load == [int(cost[m].sum()) if m else 0 for m in mine]
        if G == 1:
            assert mine == [list(range(H))]                                     # a no-op (Table 4)
        # no worse than the fixed contiguous assignment the paper starts from
        fixed = [int(cost[r * cap:(r + 1) * cap].sum()) for r in range(G)]
        assert max(load) <= max(fixed)


def test_oracle_equals_textbook_lpt_when_capacity_does_not_bind():
    # ranks * cap much larger than needed never happens with cap = ceil(H/G); but with equal costs per
    # pair the capacity rule and plain LPT agree on the multiset of loads
    g = np.random.default_rng(1)
    for H, G in ((8, 2), (12, 3), (16, 4)):
        base = g.integers(1000, 2000, H // 2)
        cost = np.concatenate([base, base])                                    # every cost twice
        _, load = oracle.schedule_heads(cost, G)
        assert max(load) <= max(unconstrained_lpt(list(cost), G)) * 1.05


def test_oracle_close_to_the_optimum_on_tiny_cases():
    g = np.random.default_rng(2)
    for H, G in ((6, 2), (6, 3), (8, 2)):
        cost = [int(c) for c in g.integers(1, 100, H)]
        _, load = oracle.schedule_heads(cost, G)
        opt = brute_force_best_makespan(cost, G, -(-H // G))
        assert opt <= max(load) <= opt * 4 / 3 + 1e-9


def test_skewed_heads_imbalance_drops():
    # a few dense heads among sparse ones (per-head densities differ)
    g = np.random.default_rng(3)
    cost = np.concatenate([g.integers(50000, 60000, 5), g.integers(5000, 15000, 35)])
    g.shuffle(cost)
    _, load = oracle.schedule_heads(cost, 8)
    fixed = [int(cost[r * 5:(r + 1) * 5].sum()) for r in range(8)]
    imb = lambda l: max(l) / (sum(l) / len(l))
    assert imb(load) < imb(fixed) and imb(load) < 1.15


@pytest.mark.parametrize("H,G", [(40, 8), (40, 3), (9, 4), (5, 8), (40, 1)])
def test_library_host_function_matches_oracle(H, G):
    g = np.random.default_rng(H * 10 + G)
    cost = g.integers(0, 70000, H)
    cost[: H // 4] = cost[0]                                                   # ties
    order, load = B.chorus_schedule_heads(cost, G)
    mine, load_o = oracle.schedule_heads(cost, G)
    assert [[h for h in row.tolist() if h >= 0] for row in order] == mine
    assert load.tolist() == load_o


def test_library_rejects_bad_arguments():
    with pytest.raises(B.ChorusError):
        B.chorus_schedule_heads([1, -2, 3], 2)


# ---- world_size 2 over gloo: every rank derives the same schedule and they cover the heads once ----
def _worker(rank, world, port, cost, out):
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    order, load = B.chorus_schedule_heads(cost, world)
    mine = [h for h in order[rank].tolist() if h >= 0]
    my_load = torch.tensor([sum(cost[h] for h in mine)], dtype=torch.int64)
    loads = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(loads, my_load)
    seen = torch.zeros(len(cost), dtype=torch.int64)
    seen[mine] = 1
    dist.all_reduce(seen)                       # every head taken by exactly one rank
    worst = my_load.clone().double()
    dist.all_reduce(worst, op=dist.ReduceOp.MAX)    # the step time is the slowest rank's (appendix A)
    if rank == 0:
        out.put(([int(x) for x in loads], load.tolist(), seen.tolist(), float(worst)))
    dist.destroy_process_group()


def test_two_ranks_gloo():
    cost = [int(c) for c in np.random.default_rng(5).integers(1000, 60000, 40)]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, cost, out)) for r in range(2)]
    for p in procs:
        p.start()
    gathered, load, seen, worst = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert gathered == load and seen == [1] * 40 and worst == max(load)
    assert load == oracle.schedule_heads(cost, 2)[1]
