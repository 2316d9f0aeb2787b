"""GPU parity for masks in the paper's own 64 x 128 block geometry (R26):
chorus_mask_to_index_64x128 bit-exact against the oracle, chorus_block_sparse_attn_fwd_64x128 against the fp64
oracle that reads the 64 x 128 bitmask itself (never the index), BF16 / FP16 / FP8, usual tolerances."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import BF16_MAX, BF16_MEAN, BF16_RELFRO, FP8_COS, FP8_MAX, dbf16, dev, dmask, err_stats
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu
SCALE = 1.0 / np.sqrt(128.0)


def random_mask(L, H, N, rho, seed):
    nq64, nk128 = (N + 63) // 64, (N + 127) // 128
    g = np.random.default_rng(seed)
    keep = g.random((L, H, nq64, nk128)) < rho
    bm = W.pack_bits(keep)
    if nk128 % 32:
        bm[..., -1] |= np.uint32((0xFFFFFFFF << (nk128 % 32)) & 0xFFFFFFFF)   # garbage pad bits
    return keep, bm


@pytest.mark.parametrize("L,H,N,rho", [(1, 1, 64, 1.0), (2, 3, 65, 0.5), (1, 2, 129, 0.5), (2, 2, 4200, 0.3),
                                       (1, 3, 8256, 0.1), (3, 2, 2049, 0.7), (1, 40, 32760, 0.25),
                                       (8, 40, 32760, 0.12), (7, 40, 32767, 0.6)])   # >= 2^20 tile-mask words: 4 per thread
def test_decode_64x128_bit_exact(L, H, N, rho):
    keep, bm = random_mask(L, H, N, rho, seed=N + L)
    rp_o, ci_o = oracle.mask_to_index_64x128(bm, N)
    rp, ci = B.chorus_mask_to_index_64x128(dmask(bm), N)
    torch.cuda.synchronize()
    assert np.array_equal(rp.cpu().numpy(), rp_o)
    assert np.array_equal(ci.cpu().numpy().view(np.uint32)[: len(ci_o)], ci_o)
    # count only, and a capacity smaller than the entry count: nothing beyond it is touched
    rp2, none = B.chorus_mask_to_index_64x128(dmask(bm), N, count_only=True)
    assert none is None and np.array_equal(rp2.cpu().numpy(), rp_o)
    if len(ci_o) > 10:
        cap = len(ci_o) // 2
        buf = torch.full((len(ci_o),), -7, dtype=torch.int32, device=dev())
        B.chorus_mask_to_index_64x128(dmask(bm), N, col_idx=buf[:cap])
        torch.cuda.synchronize()
        got = buf.cpu().numpy()
        assert np.array_equal(got[:cap].view(np.uint32), ci_o[:cap]) and np.all(got[cap:] == -7)


def attention_case(N, H, seed, rho=0.4):
    g = np.random.default_rng(seed)
    Q, K, V = (W.bf16_bits_from_f32(g.standard_normal((1, N, H, 128)).astype(np.float32)) for _ in range(3))
    keep, bm = random_mask(1, H, N, rho, seed)
    keep, bm = keep.copy(), None
    nq64 = keep.shape[2]
    keep[0, 0] = True                                   # head 0 dense
    if nq64 >= 2:
        keep[0, 1, 0, :] = False                        # upper half of block 0 keeps nothing, lower does
        keep[0, 1, 1, 0] = True
    if nq64 >= 4 and H > 2:
        keep[0, 2, 2:4, :] = False                      # a whole 128-row block empty
        keep[0, 2, 0] = keep[0, 2, 1]                   # both halves agree
    for qb in range(0, nq64 - 1, 2):                    # halves that share nothing in the first key blocks
        keep[0, H - 1, qb, 0] = True
        keep[0, H - 1, qb + 1, 0] = False
    bm = W.pack_bits(keep[0])
    return Q, K, V, keep[0], bm


def compare_items(O, Q, K, V, bm, N, H, fp8_scales=None, items=None):
    nq64 = (N + 63) // 64
    if items is None:
        items = [(0, h, qb) for h in range(H) for qb in range(nq64)]
    ref = oracle.block_sparse_attn(Q, K, V, bm, SCALE, items=np.asarray(items, np.int32), block=(64, 128),
                                   fp8_scales=fp8_scales)
    got = np.zeros_like(ref)
    for t, (_, h, qb) in enumerate(items):
        lo, hi = 64 * qb, min(N, 64 * qb + 64)
        got[t, : hi - lo] = O[0, lo:hi, h]
    return err_stats(got, ref), got, ref


@pytest.mark.parametrize("N,H", [(320, 3), (449, 3), (64, 2), (2100, 4)])
def test_bf16_attention_64x128_matches_oracle(N, H):
    Q, K, V, keep, bm = attention_case(N, H, seed=N)
    rp, ci = B.chorus_mask_to_index_64x128(dmask(bm[None]), N)
    lse = torch.empty((1, H, N), dtype=torch.float32, device=dev())
    O = B.chorus_block_sparse_attn_fwd(dbf16(Q), dbf16(K), dbf16(V), rp, ci, SCALE, lse=lse, geometry_64x128=True)
    torch.cuda.synchronize()
    O = O.float().cpu().numpy().astype(np.float64)
    assert not np.isnan(O).any()
    (mx, mean, relfro, _), got, ref = compare_items(O, Q, K, V, bm, N, H)
    assert mx <= BF16_MAX and mean <= BF16_MEAN and relfro <= BF16_RELFRO, (mx, mean, relfro)
    # rows whose own 64-row mask row is empty are exactly 0 and have lse = -inf
    gl = lse.cpu().numpy()
    for h in range(H):
        for qb in range(keep.shape[1]):
            lo, hi = 64 * qb, min(N, 64 * qb + 64)
            if not keep[h, qb].any():
                assert np.all(O[0, lo:hi, h] == 0) and np.all(np.isneginf(gl[0, h, lo:hi]))
            else:
                assert np.all(np.isfinite(gl[0, h, lo:hi]))


def test_halves_that_agree_give_the_plain_kernels_bits():
    """A 64 x 128 mask whose row pairs agree is a 128 x 64 mask with doubled key blocks: no flag bit is set and the
    result is the plain call's, bit for bit."""
    N, H = 1000, 2
    g = np.random.default_rng(5)
    Q, K, V = (W.bf16_bits_from_f32(g.standard_normal((1, N, H, 128)).astype(np.float32)) for _ in range(3))
    nq128, nk128, nk64 = 8, 8, 16
    k128 = g.random((H, nq128, nk128)) < 0.5
    keep64 = np.repeat(k128, 2, axis=1)                          # [H][16][8]
    plain = np.repeat(k128, 2, axis=2)[:, :, :nk64]              # [H][8][16] in the 128 x 64 geometry
    rp, ci = B.chorus_mask_to_index_64x128(dmask(W.pack_bits(keep64)[None]), N)
    rp2, ci2 = B.chorus_mask_to_index(dmask(W.pack_bits(plain)[None]), nk64)
    torch.cuda.synchronize()
    assert torch.equal(rp, rp2) and torch.equal(ci[: int(rp[-1])], ci2[: int(rp2[-1])])
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    a = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, SCALE, geometry_64x128=True)
    b = B.chorus_block_sparse_attn_fwd(q, k, v, rp2, ci2, SCALE)
    torch.cuda.synchronize()
    assert torch.equal(a, b)


def test_fp16_and_fp8_attention_64x128_match_oracle():
    N, H = 449, 3
    Q, K, V, keep, bm = attention_case(N, H, seed=77)
    rp, ci = B.chorus_mask_to_index_64x128(dmask(bm[None]), N)
    # fp16
    h16 = [dbf16(x).to(torch.float16) for x in (Q, K, V)]
    O = B.chorus_block_sparse_attn_fwd(*h16, rp, ci, SCALE, geometry_64x128=True)
    torch.cuda.synchronize()
    (mx, mean, _, _), _, _ = compare_items(O.float().cpu().numpy().astype(np.float64),
                                           *(t.cpu().numpy() for t in h16), bm, N, H)
    assert mx <= BF16_MAX and mean <= BF16_MEAN, (mx, mean)
    # fp8
    qz = B.chorus_quantize_fp8(dbf16(Q), dbf16(K), dbf16(V))
    O8 = B.chorus_block_sparse_attn_fwd(qz[0], qz[1], qz[2], rp, ci, SCALE, dtype=B.CHORUS_FP8_E4M3,
                                        fp8_scales=qz[3:], geometry_64x128=True)
    torch.cuda.synchronize()
    q8, k8, v8, qs, ks, vs = (t.cpu().numpy() for t in qz)
    (mx, _, _, cos), _, _ = compare_items(O8.float().cpu().numpy().astype(np.float64), q8, k8, v8, bm, N, H,
                                          fp8_scales=(qs, ks, vs))
    assert mx <= FP8_MAX and cos >= FP8_COS, (mx, cos)


def test_cfg2_full_size_sampled_blocks_64x128():
    """480p layer in the bench's launch configuration with a 25 % mask in the paper's geometry."""
    cfg = W.CFG2
    Q, K, V = W.qkv_bits(cfg)
    N, H = cfg.N, cfg.H
    keep, bm = random_mask(1, H, N, 0.25, seed=11)
    rp, ci = B.chorus_mask_to_index_64x128(dmask(bm), N)
    O = B.chorus_block_sparse_attn_fwd(dbf16(Q), dbf16(K), dbf16(V), rp, ci, cfg.scale, geometry_64x128=True)
    torch.cuda.synchronize()
    g = np.random.default_rng(3)
    nq64 = (N + 63) // 64
    items = sorted({(0, int(h), int(q)) for h, q in zip(g.integers(0, H, 12), g.integers(0, nq64, 12))}
                   | {(0, 0, 0), (0, H - 1, nq64 - 1)})
    (mx, mean, relfro, _), _, _ = compare_items(O.float().cpu().numpy().astype(np.float64), Q, K, V, bm[0], N, H,
                                                items=items)
    assert mx <= BF16_MAX and mean <= BF16_MEAN and relfro <= BF16_RELFRO, (mx, mean, relfro)


@pytest.mark.parametrize("N,H,scale", [(512, 2, 0.0884), (200, 1, 0.3), (1000, 3, 0.0884), (64, 1, 1.0), (449, 2, 0.5)])
def test_block_mass_64x128_matches_oracle_and_closes_the_loop(N, H, scale):
    """chorus_block_mass_64x128 (two passes and one pass with the LSE) against the oracle; then the paper-geometry
    loop on the GPU alone: mass -> top-p mask (bit-exact against the oracle on the same masses) -> 64 x 128 index
    -> attention, compared with the oracle on that mask."""
    g = np.random.default_rng(N)
    Q, K, V = (W.bf16_bits_from_f32(g.standard_normal((1, N, H, 128)).astype(np.float32)) for _ in range(3))
    scale = float(np.float32(scale))
    ref = oracle.block_mass(Q, K, scale, block=(64, 128))
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    got = B.chorus_block_mass(q, k, scale, geometry_64x128=True)
    # one pass, with the row log-sum-exp of the dense attention call
    nk64 = (N + 63) // 64
    full = torch.full((1, H, (N + 127) // 128, (nk64 + 31) // 32), -1, dtype=torch.int32, device=dev())
    rp, ci = B.chorus_mask_to_index(full, nk64)
    lse = torch.empty((1, H, N), dtype=torch.float32, device=dev())
    B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, scale, lse=lse)
    got1 = B.chorus_block_mass(q, k, scale, lse=lse, geometry_64x128=True)
    torch.cuda.synchronize()
    for m in (got, got1):
        m = m.cpu().numpy().astype(np.float64)
        assert m.shape == ref.shape
        tol = 2e-3 * np.maximum(ref, 1e-3) + 1e-5
        assert np.all(np.abs(m - ref) <= tol), float(np.abs(m - ref).max())
    bm, kept = B.chorus_mask_from_mass(got[0], 0.9, 0.1)
    torch.cuda.synchronize()
    bm_o, kept_o = oracle.mask_from_mass(got[0].cpu().numpy(), ref.shape[3], float(np.float32(0.9)), float(np.float32(0.1)))
    assert np.array_equal(bm.cpu().numpy().view(np.uint32), bm_o) and np.array_equal(kept.cpu().numpy(), kept_o)
    rp2, ci2 = B.chorus_mask_to_index_64x128(bm[None], N)
    O = B.chorus_block_sparse_attn_fwd(q, k, v, rp2, ci2, scale, geometry_64x128=True)
    torch.cuda.synchronize()
    nq64 = (N + 63) // 64
    items = [(0, h, qb) for h in range(H) for qb in range(nq64)]
    refO = oracle.block_sparse_attn(Q, K, V, bm_o, scale, items=np.asarray(items, np.int32), block=(64, 128))
    Of = O.float().cpu().numpy().astype(np.float64)
    gotO = np.zeros_like(refO)
    for t, (_, h, qb) in enumerate(items):
        lo, hi = 64 * qb, min(N, 64 * qb + 64)
        gotO[t, : hi - lo] = Of[0, lo:hi, h]
    mx, mean, _, _ = err_stats(gotO, refO)
    assert mx <= BF16_MAX and mean <= BF16_MEAN, (mx, mean)


@pytest.mark.parametrize("fp8", [False, True])
def test_64x128_geometry_with_first_frame_scaling(fp8):
    """Both variants at once, as the paper's pipeline uses them (L153 geometry, eq. (1) at L109-114): n_first = 330
    straddles a 64-key tile whose key block only one half of a 128-row block may keep."""
    N, H, n0, beta = 990, 3, 330, 1.3
    Q, K, V, keep, bm = attention_case(N, H, seed=31)
    rp, ci = B.chorus_mask_to_index_64x128(dmask(bm[None]), N)
    nq64 = (N + 63) // 64
    items = np.asarray([(0, h, qb) for h in range(H) for qb in range(nq64)], np.int32)
    if fp8:
        qz = B.chorus_quantize_fp8(dbf16(Q), dbf16(K), dbf16(V))
        O = B.chorus_block_sparse_attn_fwd(qz[0], qz[1], qz[2], rp, ci, SCALE, dtype=B.CHORUS_FP8_E4M3,
                                           fp8_scales=qz[3:], geometry_64x128=True, n_first=n0, beta=beta)
        q8, k8, v8, qs, ks, vs = (t.cpu().numpy() for t in qz)
        ref = oracle.block_sparse_attn(q8, k8, v8, bm, SCALE, items=items, block=(64, 128), fp8_scales=(qs, ks, vs),
                                       n_first=n0, beta=beta)
    else:
        O = B.chorus_block_sparse_attn_fwd(dbf16(Q), dbf16(K), dbf16(V), rp, ci, SCALE, geometry_64x128=True,
                                           n_first=n0, beta=beta)
        ref = oracle.block_sparse_attn(Q, K, V, bm, SCALE, items=items, block=(64, 128), n_first=n0, beta=beta)
    torch.cuda.synchronize()
    Of = O.float().cpu().numpy().astype(np.float64)
    got = np.zeros_like(ref)
    for t, (_, h, qb) in enumerate(items):
        lo, hi = 64 * qb, min(N, 64 * qb + 64)
        got[t, : hi - lo] = Of[0, lo:hi, h]
    mx, mean, _, cos = err_stats(got, ref)
    if fp8:
        assert mx <= FP8_MAX and cos >= FP8_COS, (mx, cos)
    else:
        assert mx <= BF16_MAX and mean <= BF16_MEAN, (mx, mean)
        plain = oracle.block_sparse_attn(Q, K, V, bm, SCALE, items=items, block=(64, 128))
        assert np.abs(plain - ref).max() > 10 * BF16_MAX          # the scaling is not a no-op here
