"""Two ranks over NCCL (appendix A): seq_to_heads -> chorus_block_sparse_attn_fwd ->
heads_to_seq with the CUDA copies and the real all-to-all, every rank's slice of O against the fp64 oracle.
Needs two GPUs: self-skips on the one-GPU pool (there the same functions run with one rank in
test_gpu_head_exchange.py, and the two-rank exchange over gloo in test_head_exchange_cpu.py)."""
import os
import socket

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        import oracle
        from paper_2606_25040_b200 import binding as B
        from paper_2606_25040_b200 import ulysses
        from paper_2606_25040_b200 import workloads as W
        # N = 3121 on purpose: unequal shards (1560 / 1561 tokens), ragged last blocks
        cfg = W.AttnConfig("ux2", H=8, frames=1, hp=1, wp=3121, density=0.3, data_seed=3, mask_seed=4)
        Q, K, V = W.qkv_bits(cfg)
        g = np.random.default_rng(1)
        keep = g.random((cfg.H, cfg.nq, cfg.nk)) < (0.1 + 0.1 * np.arange(cfg.H))[:, None, None]   # uneven heads
        keep[:, :, 0] = True
        bm = W.pack_bits(keep)
        to = lambda x: torch.from_numpy(np.ascontiguousarray(x).view(np.int16)).view(torch.bfloat16).to(dev)
        dm = torch.from_numpy(bm[None].view(np.int32)).to(dev)
        rp, _ = B.chorus_mask_to_index(dm, cfg.nk)
        cost = B.chorus_head_costs(rp, cfg.H, cfg.nq)
        order = B.chorus_schedule_heads(cost.cpu(), world)[0].reshape(-1).tolist()
        bounds = ulysses.shard_bounds(cfg.N, world)
        lo, hi = bounds[rank], bounds[rank + 1]
        qh, kh, vh = (ulysses.seq_to_heads(to(x[:, lo:hi]), order, cfg.N) for x in (Q, K, V))
        slots = cfg.H // world
        mine = order[rank * slots:(rank + 1) * slots]
        ok_in = np.array_equal(qh[0].cpu().view(torch.int16).numpy().view(np.uint16), Q[0][:, mine])
        rp2, ci2 = B.chorus_mask_to_index(torch.from_numpy(bm[mine][None].view(np.int32)).to(dev), cfg.nk)
        oh = B.chorus_block_sparse_attn_fwd(qh.contiguous(), kh.contiguous(), vh.contiguous(), rp2, ci2, cfg.scale)
        back = ulysses.heads_to_seq(oh, order)                       # [1][hi - lo][H][d]
        torch.cuda.synchronize()
        items = np.array([(0, h, qb) for h in range(cfg.H) for qb in range(cfg.nq)], np.int32)
        ref = oracle.scatter_items(oracle.block_sparse_attn(Q, K, V, bm, cfg.scale, items=items), items, cfg.N, cfg.H)
        err = np.abs(back.float().cpu().numpy().astype(np.float64) - ref[:, lo:hi])
        q.put((rank, bool(ok_in), tuple(back.shape) == (1, hi - lo, cfg.H, cfg.d), float(err.max()), float(err.mean())))
    finally:
        dist.destroy_process_group()


def test_ulysses_attention_two_ranks_nccl():
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (the pool gives one): multi-rank path unmeasured on hardware, DESIGN.md section 8")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ok_in, ok_shape, mx, mean in res:
        assert ok_in and ok_shape, rank
        assert mx <= 2e-2 and mean <= 2e-3, (rank, mx, mean)        # north_star's BF16 tolerance
