"""GPU parity for the head exchange (appendix A): chorus_gather_heads / chorus_scatter_heads bit-exact
against the oracle's copies, and the one-rank round trip of paper_2606_25040_b200.ulysses around the attention
kernel: heads permuted by the greedy schedule, attention on the permuted heads, heads put back == the direct call,
bit for bit."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import dbf16, dev, dmask
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import ulysses
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n,H,d,P,dtype", [(37, 8, 128, 1, np.uint16), (37, 8, 128, 2, np.uint16), (100, 40, 128, 8, np.uint16),
                                           (5, 6, 128, 3, np.uint8), (64, 4, 16, 4, np.float32)])
def test_gather_scatter_bit_exact(n, H, d, P, dtype):
    g = np.random.default_rng(n + H + P)
    X = g.integers(0, 250, size=(n, H, d)).astype(dtype)
    order = g.permutation(H).astype(np.int32)
    tX = torch.from_numpy(X.view(np.int16) if dtype == np.uint16 else X).to(dev())
    packed = B.chorus_gather_heads(tX, order, P)
    torch.cuda.synchronize()
    ref = oracle.gather_heads(X, order, P)
    got = packed.cpu().numpy()
    assert np.array_equal(got.view(dtype) if dtype == np.uint16 else got, ref)
    back = torch.full_like(tX, 7)
    B.chorus_scatter_heads(packed, order, back)
    torch.cuda.synchronize()
    assert torch.equal(back, tX)
    # a head-major storage seen as [n][H][d] (stride_h > stride_n), as the attention call accepts it
    if n:
        hm = tX.permute(1, 0, 2).contiguous().permute(1, 0, 2)
        assert hm.stride(1) > hm.stride(0)
        assert torch.equal(B.chorus_gather_heads(hm, order, P), packed)
        out = torch.empty((H, n, d), dtype=tX.dtype, device=dev()).permute(1, 0, 2)
        B.chorus_scatter_heads(packed, order, out)
        torch.cuda.synchronize()
        assert torch.equal(out.contiguous(), tX)


def test_argument_validation():
    X = torch.zeros((4, 6, 128), dtype=torch.bfloat16, device=dev())
    for order, P in (([0, 1, 2, 3, 4, 4], 2), ([0, 1, 2, 3, 4, 6], 2), ([0, 1, 2, 3, 4, 5], 4)):
        with pytest.raises(B.ChorusError):
            B.chorus_gather_heads(X, order, P)
    with pytest.raises(B.ChorusError):          # rows must be multiples of 16 bytes
        B.chorus_gather_heads(torch.zeros((4, 6, 4), dtype=torch.bfloat16, device=dev()), [0, 1, 2, 3, 4, 5], 2)


def test_scheduled_round_trip_around_the_attention_kernel_one_rank():
    cfg = W.AttnConfig("ux", H=8, frames=2, hp=16, wp=40, density=0.3, data_seed=3, mask_seed=4)
    Q, K, V = W.qkv_bits(cfg)
    g = np.random.default_rng(1)
    keep = g.random((cfg.H, cfg.nq, cfg.nk)) < (0.1 + 0.1 * np.arange(cfg.H))[:, None, None]   # uneven heads
    keep[:, :, 0] = True
    bm = W.pack_bits(keep)
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    direct = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale)
    # the schedule for 4 ranks, flattened: a permutation of the heads (H % ranks == 0)
    cost = B.chorus_head_costs(rp, cfg.H, cfg.nq)
    order, load = B.chorus_schedule_heads(cost.cpu(), 4)
    order = order.reshape(-1).tolist()
    assert sorted(order) == list(range(cfg.H)) and order != list(range(cfg.H))
    # one rank: the "exchange" is the head permutation alone
    qh, kh, vh = (ulysses.seq_to_heads(x, order, cfg.N) for x in (q, k, v))
    assert np.array_equal(qh[0].cpu().view(torch.int16).numpy().view(np.uint16), Q[0][:, order])
    rp2, ci2 = B.chorus_mask_to_index(dmask(bm[order][None]), cfg.nk)      # the masks follow their heads
    oh = B.chorus_block_sparse_attn_fwd(qh, kh, vh, rp2, ci2, cfg.scale)
    back = ulysses.heads_to_seq(oh, order)
    torch.cuda.synchronize()
    assert torch.equal(back, direct)
