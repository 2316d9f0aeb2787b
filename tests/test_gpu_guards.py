"""Out-of-bounds guards: every output buffer sits between sentinel regions, and after each call the
sentinels must be intact (compute-sanitizer is closed on the GPU pool - its exact answer is quoted in DESIGN.md
section 7.5 - so the tests carry their own bounds checks).  Ragged shapes on purpose: N = 3120 has a 48-row last query block / 48-key last
key block."""
import numpy as np
import pytest
import torch

from gpu_common import dbf16, dev, dmask
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu
PAD = 4096


def guarded(shape, dtype, fill):
    """A tensor of `shape` carved out of the middle of a sentinel-filled allocation."""
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * PAD,), fill, dtype=dtype, device=dev())
    return buf, buf[PAD: PAD + n].view(shape)


def intact(buf, n, fill):
    f = torch.tensor(fill, dtype=buf.dtype, device=buf.device)
    return bool((buf[:PAD] == f).all()) and bool((buf[PAD + n:] == f).all())


def test_outputs_stay_inside_their_buffers():
    cfg = W.scaled(W.CFG2, H=2, frames=2)                 # N = 3120
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    rows = cfg.H * cfg.nq
    # decode
    rp_buf, rp = guarded((rows + 1,), torch.int32, -7)
    nnz = int(W.unpack_bits(bm, cfg.nk).sum())
    ci_buf, ci = guarded((nnz,), torch.int32, -7)
    B.chorus_mask_to_index(dmask(bm[None]), cfg.nk, row_ptr=rp, col_idx=ci)
    torch.cuda.synchronize()
    assert intact(rp_buf, rows + 1, -7) and intact(ci_buf, nnz, -7) and int(rp[-1]) == nnz
    # attention (bf16) with LSE
    n_o = cfg.N * cfg.H * cfg.d
    o_buf, O = guarded((1, cfg.N, cfg.H, cfg.d), torch.bfloat16, 777.0)
    l_buf, lse = guarded((1, cfg.H, cfg.N), torch.float32, 777.0)
    B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale, O=O, lse=lse)
    torch.cuda.synchronize()
    assert intact(o_buf, n_o, 777.0) and intact(l_buf, cfg.H * cfg.N, 777.0)
    assert not bool((O == 777.0).any()) and not bool((lse == 777.0).any())      # every valid row was written
    # quantise + fp8 attention
    outs = [guarded((1, cfg.N, cfg.H, cfg.d), torch.uint8, 0xAB) for _ in range(3)]
    nsb = (cfg.N + 127) // 128
    scs = [guarded((1, cfg.H, nsb), torch.float32, 777.0), guarded((1, cfg.H, nsb), torch.float32, 777.0),
           guarded((1, cfg.H, cfg.d), torch.float32, 777.0)]
    out = tuple(t for _, t in outs) + tuple(t for _, t in scs)
    B.chorus_quantize_fp8(q, k, v, out=out)
    o8_buf, O8 = guarded((1, cfg.N, cfg.H, cfg.d), torch.bfloat16, 777.0)
    B.chorus_block_sparse_attn_fwd(out[0], out[1], out[2], rp, ci, cfg.scale, dtype=B.CHORUS_FP8_E4M3, O=O8,
                                   fp8_scales=out[3:])
    torch.cuda.synchronize()
    assert all(intact(b, n_o, 0xAB) for b, _ in outs)
    assert intact(scs[0][0], cfg.H * nsb, 777.0) and intact(scs[1][0], cfg.H * nsb, 777.0)
    assert intact(scs[2][0], cfg.H * cfg.d, 777.0) and intact(o8_buf, n_o, 777.0)
    # mask construction
    m_buf, mass = guarded((1, cfg.H, cfg.nq, cfg.nk), torch.float32, 777.0)
    B.chorus_block_mass(q, k, cfg.scale, mass=mass)
    b_buf, bits = guarded((cfg.H, cfg.nq, cfg.words), torch.int32, -7)
    k_buf, kept = guarded((cfg.H, cfg.nq), torch.int32, -7)
    B.chorus_mask_from_mass(mass[0], 0.9, 0.1, bitmask=bits, kept=kept)
    c_buf, cov = guarded((cfg.H,), torch.float32, 777.0)
    B.chorus_mask_coverage(mass[0], bits, cfg.nk, coverage=cov)
    h_buf, cost = guarded((cfg.H,), torch.int64, -7)
    B.chorus_head_costs(rp, cfg.H, cfg.nq, cost=cost)
    torch.cuda.synchronize()
    assert intact(m_buf, rows * cfg.nk, 777.0) and intact(b_buf, rows * cfg.words, -7)
    assert intact(k_buf, rows, -7) and intact(c_buf, cfg.H, 777.0) and intact(h_buf, cfg.H, -7)
    assert not bool((mass == 777.0).any()) and bool((cov >= 0.9 - 1e-5).all())
    # visit refresh and retrieval
    g = np.random.default_rng(0)
    mset = W.pack_bits(g.random((9, 2, 3, 45)) < 0.2)
    v_buf, vm = guarded(mset.shape, torch.int32, -7)
    vm.copy_(torch.from_numpy(mset.view(np.int32)))
    B.chorus_visit_refresh(vm, 45, group=8)
    bank = torch.randn((50, 256), device=dev())
    outs3 = [guarded((1,), torch.int32, -7), guarded((1,), torch.float32, 777.0), guarded((1,), torch.int32, -7)]
    B.chorus_retrieve_top1(bank, bank[7].clone(), 0.4, out=tuple(t for _, t in outs3))
    torch.cuda.synchronize()
    assert intact(v_buf, mset.size, -7)
    assert intact(outs3[0][0], 1, -7) and intact(outs3[1][0], 1, 777.0) and intact(outs3[2][0], 1, -7)
    assert int(outs3[0][1]) == 7
