"""CPU tests of the head exchange (appendix A): pins of the oracle's gather / scatter copies, and the
data flow of paper_2606_25040_b200.ulysses over a 2-rank gloo group with the oracle's copies in place of the CUDA
kernels (the exchange logic, chunk order and views are the product's; no GPU here)."""
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
        N, H, d = 12, 6, 4
        g = np.random.default_rng(0)
        X = g.standard_normal((N, H, d)).astype(np.float32)                     # the global tensor
        order = [4, 1, 3, 0, 5, 2]                                              # rank 0: 4, 1, 3; rank 1: 0, 5, 2
        n_loc, slots = N // world, H // world
        x_loc = torch.from_numpy(X[rank * n_loc:(rank + 1) * n_loc].copy())[None]
        gather = lambda x, o, P: torch.from_numpy(oracle.gather_heads(x.numpy(), o, P))

        def scatter(chunks, o, out):
            out.copy_(torch.from_numpy(oracle.scatter_heads(chunks.numpy(), o)))

        xh = ulysses.seq_to_heads(x_loc, order, _gather=gather)
        mine = order[rank * slots:(rank + 1) * slots]
        ok1 = xh.shape == (1, N, slots, d) and np.array_equal(xh[0].numpy(), X[:, mine])   # all tokens, my heads
        # "attention" = something per (token, head) that depends on the global token index
        oh = xh * 2.0 + torch.arange(N, dtype=torch.float32)[None, :, None, None]
        back = ulysses.heads_to_seq(oh.contiguous(), order, _scatter=scatter)
        ref = (X * 2.0 + np.arange(N, dtype=np.float32)[:, None, None])[rank * n_loc:(rank + 1) * n_loc]
        ok2 = back.shape == (1, n_loc, H, d) and np.array_equal(back[0].numpy(), ref)
        rows = ulysses.rank_rows(order, rank, world, nq_blk=5)
        ok3 = rows == [(h, 5 * h, 5 * h + 5) for h in mine]
        q.put((rank, bool(ok1), bool(ok2), bool(ok3)))
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
    assert res == [(0, True, True, True), (1, True, True, True)]
