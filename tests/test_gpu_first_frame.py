"""GPU parity: chorus_block_sparse_attn_fwd_first_frame (eq. (1), first-frame key
enhancement fused into the attention kernel) vs the fp64 oracle on the same input bytes, in BF16, FP16 and
FP8; same tolerances as the plain call."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import (BF16_MAX, BF16_MEAN, BF16_RELFRO, FP8_COS, FP8_MAX, all_items, dbf16, dmask,
                        err_stats, gather_items)
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


def small_case(hp, wp, frames, seed):
    cfg = W.AttnConfig("ff", H=3, frames=frames, hp=hp, wp=wp, density=0.5, data_seed=seed, mask_seed=7)
    Q, K, V = W.qkv_bits(cfg)
    g = np.random.default_rng(seed)
    keep = g.random((cfg.H, cfg.nq, cfg.nk)) < 0.5
    keep[:, :, cfg.nk - 1] = True      # the ragged last key block
    keep[0] = True                     # head 0: dense
    keep[1, :, : (hp * wp) // 64 + 1] = (np.arange((hp * wp) // 64 + 1) % 2 == 0)   # first frame every other block
    keep[2, 0, :] = False              # an empty row
    return cfg, Q, K, V, W.pack_bits(keep)


# n_first = hp * wp tokens: 330 and 1560 straddle a 64-key tile (and fall inside a pair), 512 ends on a pair
@pytest.mark.parametrize("hp,wp,frames,beta", [(10, 33, 3, 1.3), (16, 32, 3, 0.6), (30, 52, 2, 1.15), (3, 43, 5, 2.0)])
def test_bf16_first_frame_scaling_matches_oracle(hp, wp, frames, beta):
    cfg, Q, K, V, bm = small_case(hp, wp, frames, seed=hp + wp)
    n0 = hp * wp
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    lse = torch.empty((1, cfg.H, cfg.N), dtype=torch.float32, device=rp.device)
    O = B.chorus_block_sparse_attn_fwd(dbf16(Q), dbf16(K), dbf16(V), rp, ci, cfg.scale, lse=lse,
                                       n_first=n0, beta=beta)
    torch.cuda.synchronize()
    items = all_items(cfg.H, cfg.nq)
    ref, ref_lse = oracle.block_sparse_attn(Q, K, V, bm, cfg.scale, items=np.asarray(items, np.int32),
                                            n_first=n0, beta=beta, return_lse=True)
    got = gather_items(O.float().cpu().numpy().astype(np.float64), items, cfg.N)
    mx, mean, relfro, _ = err_stats(got, ref)
    assert mx <= BF16_MAX and mean <= BF16_MEAN and relfro <= BF16_RELFRO, (mx, mean, relfro)
    # and it is not the unscaled result
    plain = oracle.block_sparse_attn(Q, K, V, bm, cfg.scale, items=np.asarray(items, np.int32))
    assert np.abs(plain - ref).max() > 10 * BF16_MAX
    gl = lse.cpu().numpy()
    for t, (b, h, qb) in enumerate(items):
        lo, hi = qb * 128, min(cfg.N, qb * 128 + 128)
        r = ref_lse[t, : hi - lo]
        fin = np.isfinite(r)
        assert np.array_equal(np.isfinite(gl[b, h, lo:hi]), fin)
        assert not fin.any() or np.abs(gl[b, h, lo:hi][fin] - r[fin]).max() <= 2e-3


def test_degenerate_arguments_run_the_plain_kernel_bit_for_bit():
    cfg, Q, K, V, bm = small_case(10, 33, 3, seed=5)
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    plain = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale)
    a = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, n_first=330, beta=1.0)
    b = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, n_first=0, beta=2.0)
    # n_first >= N: every score scaled == the plain kernel with scale * beta (beta a power of two: exact)
    c = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, n_first=10 ** 9, beta=2.0)
    d = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale * 2.0)
    torch.cuda.synchronize()
    assert torch.equal(a, plain) and torch.equal(b, plain) and torch.equal(c, d)
    for bad in (dict(n_first=-1, beta=2.0), dict(n_first=5, beta=0.0), dict(n_first=5, beta=-1.0),
                dict(n_first=5, beta=float("inf")), dict(n_first=5, beta=float("nan"))):
        with pytest.raises(B.ChorusError):
            B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, **bad)


def test_fp16_first_frame_scaling_matches_oracle():
    cfg, Q, K, V, bm = small_case(10, 33, 3, seed=9)
    to16 = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).to(torch.float16)
    q, k, v = (to16(x) for x in (Q, K, V))
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    O = B.chorus_block_sparse_attn_fwd(q.cuda(), k.cuda(), v.cuda(), rp, ci, cfg.scale, n_first=330, beta=1.25)
    torch.cuda.synchronize()
    items = all_items(cfg.H, cfg.nq)
    ref = oracle.block_sparse_attn(q.numpy(), k.numpy(), v.numpy(), bm, cfg.scale,
                                   items=np.asarray(items, np.int32), n_first=330, beta=1.25)
    mx, mean, _, _ = err_stats(gather_items(O.float().cpu().numpy().astype(np.float64), items, cfg.N), ref)
    assert mx <= BF16_MAX and mean <= BF16_MEAN, (mx, mean)


@pytest.mark.parametrize("hp,wp,frames,beta", [(10, 33, 3, 1.3), (16, 32, 3, 1.5)])
def test_fp8_first_frame_scaling_matches_oracle(hp, wp, frames, beta):
    cfg, Q, K, V, bm = small_case(hp, wp, frames, seed=hp)
    n0 = hp * wp
    qz = B.chorus_quantize_fp8(dbf16(Q), dbf16(K), dbf16(V))
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    O = B.chorus_block_sparse_attn_fwd(qz[0], qz[1], qz[2], rp, ci, cfg.scale, dtype=B.CHORUS_FP8_E4M3,
                                       fp8_scales=qz[3:], n_first=n0, beta=beta)
    torch.cuda.synchronize()
    q8, k8, v8, qs, ks, vs = (t.cpu().numpy() for t in qz)
    items = all_items(cfg.H, cfg.nq)
    ref = oracle.block_sparse_attn(q8.view(np.uint8), k8.view(np.uint8), v8.view(np.uint8), bm, cfg.scale,
                                   items=np.asarray(items, np.int32), fp8_scales=(qs, ks, vs),
                                   n_first=n0, beta=beta)
    mx, _, _, cos = err_stats(gather_items(O.float().cpu().numpy().astype(np.float64), items, cfg.N), ref)
    assert mx <= FP8_MAX and cos >= FP8_COS, (mx, cos)


def test_cfg2_full_size_sampled_blocks_with_first_frame_scaling():
    """480p layer in the bench's launch configuration, n_first = 1560 (tile 24 straddles it)."""
    cfg = W.CFG2
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    n0, beta = 30 * 52, 1.2
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    O = B.chorus_block_sparse_attn_fwd(dbf16(Q), dbf16(K), dbf16(V), rp, ci, cfg.scale, n_first=n0, beta=beta)
    torch.cuda.synchronize()
    g = np.random.default_rng(3)
    items = sorted({(0, int(h), int(q)) for h, q in zip(g.integers(0, cfg.H, 10), g.integers(0, cfg.nq, 10))}
                   | {(0, 0, 0), (0, cfg.H - 1, cfg.nq - 1)})
    ref = oracle.block_sparse_attn(Q, K, V, bm, cfg.scale, items=np.asarray(items, np.int32), n_first=n0, beta=beta)
    mx, mean, relfro, _ = err_stats(gather_items(O.float().cpu().numpy().astype(np.float64), items, cfg.N), ref)
    assert mx <= BF16_MAX and mean <= BF16_MEAN and relfro <= BF16_RELFRO, (mx, mean, relfro)
