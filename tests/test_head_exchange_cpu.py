"""CPU tests of the head exchange (appendix A): pins of the oracle's gather / scatter copies, and the
exchange functions of paper_2606_25040_b200.ulysses over a 2-rank gloo group, composed here with the oracle's copies
(the all-to-all, its split sizes for unequal shards and the views are the product's; the CUDA copies around them are
tested on the GPU in test_gpu_head_exchange.py and, with two ranks over NCCL, in test_gpu_ulysses_nccl.py)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle


def test_gather_scatter_definitions():
    n, H, d, P = 3, 4, 2, 2
    X = np.arange(n * H * d, dtype=np.int32).reshape(n, H, d)
    order = [2, 0, 3, 1]                            # rank 0 gets heads 2, 0; rank 1 gets 3, 1
    g = oracle.gather_heads(X, order, P)
    assert g.shape == (P, n, H // P, d)
    # written out by hand: chunk 1, token 2, slot 0 is head 3 of token 2
    assert np.array_equal(g[1, 2, 0], X[2, 3]) and np.array_equal(g[0, 1, 1], X[1, 0])
    assert np.array_equal(g, np.stack([X[:, [2, 0]], X[:, [3, 1]]]))          # numpy fancy indexing
    assert np.array_equal(oracle.scatter_heads(g, order), X)                    # inverse
    assert np.array_equal(oracle.gather_heads(X, list(range(H)), 1)[0], X)      # one rank, identity order


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_25040_b200 import ulysses
        oks = []
        for N in (12, 13):                                                          # equal and unequal shards
            H, d = 6, 4
            g = np.random.default_rng(0)
            X = g.standard_normal((N, H, d)).astype(np.float32)                     # the global tensor
            order = [4, 1, 3, 0, 5, 2]                                              # rank 0: 4, 1, 3; rank 1: 0, 5, 2
            bounds = ulysses.shard_bounds(N, world)
            lo, hi = bounds[rank], bounds[rank + 1]
            slots = H // world
            # the local copies are the oracle's here (no GPU); the exchange, split sizes and views are the product's
            packed = torch.from_numpy(oracle.gather_heads(X[lo:hi].copy(), order, world))
            xh = ulysses.exchange_to_heads(packed, bounds)
            mine = order[rank * slots:(rank + 1) * slots]
            oks.append(tuple(xh.shape) == (N, slots, d) and np.array_equal(xh.numpy(), X[:, mine]))   # all tokens, my heads
            # "attention" = something per (token, head) that depends on the global token index
            oh = xh * 2.0 + torch.arange(N, dtype=torch.float32)[:, None, None]
            chunks = ulysses.exchange_to_seq(oh.contiguous(), bounds)
            back = oracle.scatter_heads(chunks.numpy(), order)
            ref = (X * 2.0 + np.arange(N, dtype=np.float32)[:, None, None])[lo:hi]
            oks.append(back.shape == (hi - lo, H, d) and np.array_equal(back, ref))
        rows = ulysses.rank_rows(order, rank, world, nq_blk=5)
        oks.append(rows == [(h, 5 * h, 5 * h + 5) for h in mine])
        oks.append(ulysses.shard_bounds(13, 2) == [0, 6, 13] and ulysses.shard_bounds(32760, 8)[1] == 4095)
        oks.append(abs(ulysses.imbalance([4, 1, 1, 1, 1, 4], [0, 1, 2, 3, 4, 5], 2) - 1.0) < 1e-12 and
                   abs(ulysses.imbalance([4, 4, 1, 1, 1, 1], [0, 1, 2, 3, 4, 5], 2) - 9 / 6) < 1e-12)
        q.put((rank, all(bool(o) for o in oks), len(oks)))
    finally:
        dist.destroy_process_group()


def test_ulysses_data_flow_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True, 7), (1, True, 7)]
