"""16-bit index entries (include/chorus.h): both decodes bit-exact against the oracle's 16-bit
forms, and the attention kernels on a 16-bit index bit-identical to the same call on the 32-bit index."""
import numpy as np
import pytest
import torch

import oracle
from gpu_common import dbf16, dev, dmask
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("nk,rows", [(1, 3), (33, 70), (512, 2560), (1182, 700), (2048, 100), (65536, 2)])
def test_decode_u16_bit_exact(nk, rows):
    g = np.random.default_rng(nk)
    words = (nk + 31) // 32
    bm = g.integers(0, 2**32, size=(1, 1, rows, words), dtype=np.uint64).astype(np.uint32)     # garbage pad bits
    bm &= g.integers(0, 2**32, size=bm.shape, dtype=np.uint64).astype(np.uint32)
    bm[0, 0, rows // 2] = 0xFFFFFFFF                    # a full row
    bm[0, 0, 0] = 0                                     # an empty one
    rp, ci = B.chorus_mask_to_index(dmask(bm), nk, idx16=True)
    torch.cuda.synchronize()
    rp_o, ci_o = oracle.mask_to_index_u16(bm, nk)
    assert ci.dtype == torch.uint16
    assert np.array_equal(rp.cpu().numpy(), rp_o)
    assert np.array_equal(ci.cpu().numpy().view(np.uint16)[: len(ci_o)], ci_o)


def test_decode_u16_full_size_layer_and_capacity_guard():
    cfg = W.CFG2
    bm = W.layer_mask(cfg)
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk, idx16=True)
    rp_o, ci_o = oracle.mask_to_index_u16(bm[None], cfg.nk)
    assert np.array_equal(rp.cpu().numpy(), rp_o) and np.array_equal(ci.cpu().numpy().view(np.uint16), ci_o)
    # entries beyond col_cap are never written
    buf = torch.full((1000 + 64,), 0xABCD, dtype=torch.uint16, device=dev())
    B.chorus_mask_to_index(dmask(bm[None]), cfg.nk, col_idx=buf[:1000])
    torch.cuda.synchronize()
    out = buf.cpu().numpy().view(np.uint16)
    assert np.array_equal(out[:1000], ci_o[:1000]) and np.all(out[1000:] == 0xABCD)
    with pytest.raises(B.ChorusError):                   # 65537 key blocks do not fit
        B.chorus_mask_to_index(torch.zeros((1, 1, 1, 2049), dtype=torch.int32, device=dev()), 65537, idx16=True)


@pytest.mark.parametrize("N", [200, 4680, 32760])
def test_decode_64x128_u16_bit_exact(N):
    g = np.random.default_rng(N)
    H = 2
    keep = g.random((1, H, (N + 63) // 64, (N + 127) // 128)) < 0.3
    bm = W.pack_bits(keep)
    rp, ci = B.chorus_mask_to_index_64x128(dmask(bm), N, idx16=True)
    torch.cuda.synchronize()
    rp_o, ci_o = oracle.mask_to_index_64x128_u16(bm, N)
    assert np.array_equal(rp.cpu().numpy(), rp_o)
    assert np.array_equal(ci.cpu().numpy().view(np.uint16)[: len(ci_o)], ci_o)


@pytest.mark.parametrize("dtype", ["bf16", "fp8"])
def test_attention_on_16_bit_index_is_bit_identical(dtype):
    cfg = W.scaled(W.CFG2, H=2, frames=3)               # N = 4680: ragged last blocks
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg, density=0.3)
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    kw = {}
    if dtype == "fp8":
        z = B.chorus_quantize_fp8(q, k, v)
        q, k, v = z[0], z[1], z[2]
        kw = dict(dtype=B.CHORUS_FP8_E4M3, fp8_scales=z[3:])
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    rp16, ci16 = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk, idx16=True)
    assert torch.equal(rp, rp16) and torch.equal(ci, ci16.to(torch.int32))
    O32 = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, **kw)
    O16 = B.chorus_block_sparse_attn_fwd(q, k, v, rp16, ci16, cfg.scale, **kw)
    ff = dict(n_first=cfg.hp * cfg.wp, beta=1.5)
    F32 = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, **kw, **ff)
    F16 = B.chorus_block_sparse_attn_fwd(q, k, v, rp16, ci16, cfg.scale, **kw, **ff)
    torch.cuda.synchronize()
    assert torch.equal(O32, O16) and torch.equal(F32, F16) and not torch.equal(O32, F32)
    # the paper's geometry with the flags in bits 14 / 15
    g = np.random.default_rng(3)
    keep = g.random((1, cfg.H, (cfg.N + 63) // 64, (cfg.N + 127) // 128)) < 0.3
    keep[..., 0] = True
    bm64 = dmask(W.pack_bits(keep))
    rpa, cia = B.chorus_mask_to_index_64x128(bm64, cfg.N)
    rpb, cib = B.chorus_mask_to_index_64x128(bm64, cfg.N, idx16=True)
    G32 = B.chorus_block_sparse_attn_fwd(q, k, v, rpa, cia, cfg.scale, geometry_64x128=True, **kw)
    G16 = B.chorus_block_sparse_attn_fwd(q, k, v, rpb, cib, cfg.scale, geometry_64x128=True, **kw)
    torch.cuda.synchronize()
    assert torch.equal(G32, G16)
