"""GPU parity: chorus_block_sparse_attn_fwd (BF16) vs the fp64 oracle on the same input bytes.
Tolerances are BASELINE.json north_star's (max|err| <= 2e-2, mean|err| <= 2e-3), plus the tighter
internal gates of SURVEY §8 c-5, plus closed-form probes that need no oracle run."""
import numpy as np
import pytest
import torch

from gpu_common import (BF16_MAX, BF16_MAX_TIGHT, BF16_MEAN, BF16_RELFRO, all_items, dbf16, dmask,
                        err_stats, gather_items, gpu_attention, oracle_items, report, sample_items,
                        stratified_items)
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

pytestmark = pytest.mark.gpu


def weighted_abs_v(Q, K, V, bm, cfg, items, scale):
    """A[i, c] = sum_j w_ij |v_jc| over the retained keys, in numpy fp64 straight from the definition (independent of
    the oracle and of the kernel).  The kernel feeds bf16-rounded weights to P V and divides by the fp32 sum of the
    unrounded ones, so a weight's rounding (relative 2^-9) reaches the output as 2^-9 w_ij |v_jc|: averaged away over
    thousands of comparable keys, but not on a row that a single key dominates (cfg4's x8 rows), where A ~ |O|."""
    keep = W.unpack_bits(bm, cfg.nk)
    f = lambda b: W.f32_from_bf16_bits(b).astype(np.float64)
    out = np.zeros((len(items), 128, 128))
    for t, (b, h, qb) in enumerate(items):
        lo, hi = qb * 128, min(cfg.N, qb * 128 + 128)
        idx = np.concatenate([np.arange(kb * 64, min(cfg.N, kb * 64 + 64)) for kb in np.nonzero(keep[h, qb])[0]])
        sc = scale * (f(Q[b, lo:hi, h]) @ f(K[b, idx, h]).T)
        w = np.exp(sc - sc.max(axis=1, keepdims=True))
        w /= w.sum(axis=1, keepdims=True)
        out[t, : hi - lo] = w @ np.abs(f(V[b, idx, h]))
    return out


def compare(cfg, Q, K, V, bm, items, scale=None, tight=True, stress=False):
    scale = cfg.scale if scale is None else scale
    O = gpu_attention(Q, K, V, bm, cfg.nk, scale)
    assert not np.isnan(O).any()
    ref = oracle_items(Q, K, V, bm, scale, items)
    got = gather_items(O, items, cfg.N)
    mx, mean, relfro, cos = err_stats(got, ref)
    if stress:
        # x8 rows give outputs of magnitude ~25, where the bf16 OUTPUT format alone rounds by up to
        # 2^-8 |O| ~ 0.1, and a row dominated by one key carries the bf16 rounding of that one weight
        # un-averaged (2^-9 A, A = sum_j w_ij |v_jc| ~ |O| there).  north_star's absolute 2e-2 is stated
        # for N(0,1) inputs, so it is applied to the error in excess of these two roundings, both
        # computed here from the definitions.
        err = np.abs(got - ref)
        A = weighted_abs_v(Q, K, V, bm, cfg, items, scale)
        tol = BF16_MAX + 2.0 ** -8 * np.abs(ref) + 2.0 ** -9 * A
        assert np.all(err <= tol), (mx, float((err - tol).max()))
        assert mean <= BF16_MEAN and relfro <= BF16_RELFRO, (mean, relfro)
        # how far this is from the PLAIN north_star bound: count and size of the elements beyond 2e-2, and
        # every one of them must sit where one bf16 output rounding (up to 2^-8 |ref|) alone exceeds 1e-2
        over = err > BF16_MAX
        assert np.all(2.0 ** -8 * np.abs(ref[over]) > 1e-2), float(np.abs(ref[over]).min())
        report("bf16_stress_" + cfg.name, items=len(items), elements=int(err.size), over_plain_bound=int(over.sum()),
               max_abs=mx, mean_abs=mean, relfro=relfro, max_err_over_tol=float((err / tol).max()),
               over_output_rounding_alone=int((err > BF16_MAX + 2.0 ** -8 * np.abs(ref)).sum()),
               min_abs_ref_where_over=float(np.abs(ref[over]).min()) if over.any() else None,
               max_err_over_bf16_ulp_of_ref=float((err[over] / (2.0 ** -8 * np.abs(ref[over]))).max()) if over.any() else None)
        return O
    assert mx <= BF16_MAX and mean <= BF16_MEAN, (mx, mean)
    if tight:
        assert mx <= BF16_MAX_TIGHT and relfro <= BF16_RELFRO, (mx, relfro)
    return O


def test_cfg1_all_rows():
    cfg = W.CFG1
    Q, K, V = W.qkv_bits(cfg)
    compare(cfg, Q, K, V, W.layer_mask(cfg), all_items(cfg.H, cfg.nq))


@pytest.mark.parametrize("N_hp_wp", [(10, 33), (3, 43), (1, 100), (17, 31)])
def test_ragged_shapes_and_edge_masks(N_hp_wp):
    hp, wp = N_hp_wp
    cfg = W.AttnConfig("r", H=3, frames=1, hp=hp, wp=wp, density=0.5, data_seed=20 + hp, mask_seed=5)
    Q, K, V = W.qkv_bits(cfg)
    g = np.random.default_rng(hp)
    keep = g.random((cfg.H, cfg.nq, cfg.nk)) < 0.5
    keep[:, :, cfg.nk - 1] = True           # ragged last key block always kept
    keep[0] = True                          # head 0: full mask == dense attention
    keep[1, 0, :] = False                   # an empty row: O = 0
    keep[2] = False
    keep[2, :, 0] = True                    # head 2: single kept block
    O = compare(cfg, Q, K, V, W.pack_bits(keep), all_items(cfg.H, cfg.nq))
    assert np.all(O[0, :min(128, cfg.N), 1] == 0.0)


def test_strided_bhnd_layout():
    cfg = W.AttnConfig("s", H=2, frames=1, hp=8, wp=40, density=0.5, data_seed=31, mask_seed=5)
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    tq, tk, tv = (dbf16(x).permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3) for x in (Q, K, V))
    assert tq.stride(2) > tq.stride(1)
    Oh = torch.empty((1, cfg.H, cfg.N, 128), dtype=torch.bfloat16, device=tq.device).permute(0, 2, 1, 3)
    B.chorus_block_sparse_attn_fwd(tq, tk, tv, rp, ci, cfg.scale, O=Oh)
    O2 = B.chorus_block_sparse_attn_fwd(dbf16(Q), dbf16(K), dbf16(V), rp, ci, cfg.scale)
    torch.cuda.synchronize()
    assert torch.equal(Oh.contiguous(), O2)


def test_batch_dimension():
    cfg = W.AttnConfig("b", H=2, frames=1, hp=8, wp=25, density=0.5, data_seed=32, mask_seed=5, B=2)
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    O = gpu_attention(Q, K, V, bm, cfg.nk, cfg.scale)
    for b in range(2):
        items = all_items(cfg.H, cfg.nq)
        ref = oracle_items(Q[b:b + 1], K[b:b + 1], V[b:b + 1], bm, cfg.scale, items)
        mx, mean, _, _ = err_stats(gather_items(O[b:b + 1], items, cfg.N), ref)
        assert mx <= BF16_MAX_TIGHT and mean <= BF16_MEAN


def _probe_inputs(cfg, seed):
    g = np.random.default_rng(seed)
    K = W.bf16_bits_from_f32(g.standard_normal((1, cfg.N, cfg.H, 128)).astype(np.float32))
    v = np.zeros((1, cfg.N, cfg.H, 128), np.float32)
    n = np.arange(cfg.N)
    v[0, n, :, (n // 64) % 128] = 1.0
    return K, W.bf16_bits_from_f32(v)


def q_zero_expected(keep_h, N):
    nq, nk = keep_h.shape
    valid = np.minimum(64, N - 64 * np.arange(nk)).astype(np.float64)
    out = np.zeros((nq, 128))
    for qb in range(nq):
        cnt = np.zeros(128)
        np.add.at(cnt, np.nonzero(keep_h[qb])[0] % 128, valid[keep_h[qb]])
        out[qb] = cnt / cnt.sum()
    return out


@pytest.mark.parametrize("cfg", [W.scaled(W.CFG2, H=2), W.scaled(W.CFG4, H=1)], ids=["480p", "720p"])
def test_q_zero_probe_full_size(cfg):
    # Q = 0 => uniform weights; with V[j, c] = [(j // 64) % 128 == c] the output counts kept valid
    # keys per block index: computable from the mask in integers at FULL size, no oracle run.
    K, V = _probe_inputs(cfg, 1)
    Q = np.zeros_like(K)
    bm = W.layer_mask(cfg)
    keep = W.unpack_bits(bm, cfg.nk)
    O = gpu_attention(Q, K, V, bm, cfg.nk, cfg.scale)
    for h in range(cfg.H):
        exp = q_zero_expected(keep[h], cfg.N)
        got = O[0, :, h]
        ref = np.repeat(exp, 128, axis=0)[: cfg.N]
        assert np.abs(got - ref).max() <= 2.0 ** -8 * ref.max() + 1e-6


def test_spike_and_pruned_block_probe():
    cfg = W.scaled(W.CFG2, H=1, frames=3)        # N = 4680: nq 37, nk 74 (tail 72 rows / 8 keys)
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg, density=0.3)
    keep = W.unpack_bits(bm, cfg.nk)[0]
    qf = W.f32_from_bf16_bits(Q).astype(np.float64)
    K2 = K.copy()
    rows = [5, 1000, cfg.N - 1]
    targets = []
    for n_spike, i in enumerate(rows):
        qb = i // 128
        kept = np.nonzero(keep[qb])[0]
        kb = kept[-1] if i == cfg.N - 1 else kept[len(kept) // 2]
        if i == cfg.N - 1:
            keep[qb, cfg.nk - 1] = True
            kb = cfg.nk - 1                      # spike inside the ragged last key block
        j = min(64 * kb + 3 + 7 * n_spike, cfg.N - 1)   # distinct keys even if rows share kb
        q = qf[0, i, 0]
        K2[0, j, 0] = W.bf16_bits_from_f32((60.0 / cfg.scale * q / (q @ q)).astype(np.float32))
        targets.append((i, j))
    bm = W.pack_bits(keep[None])
    # a huge key/value in a PRUNED block must have no influence at all
    qb0 = 20
    pruned = np.nonzero(~keep[qb0])[0][0]
    K3, V3 = K2.copy(), V.copy()
    K3[0, 64 * pruned:64 * pruned + 64] = 0x4700
    V3[0, 64 * pruned:64 * pruned + 64] = 0x4700
    O2 = gpu_attention(Q, K2, V, bm, cfg.nk, cfg.scale)
    O3 = gpu_attention(Q, K3, V3, bm, cfg.nk, cfg.scale)
    vf = W.f32_from_bf16_bits(V).astype(np.float64)
    for i, j in targets:
        assert np.abs(O2[0, i, 0] - vf[0, j, 0]).max() <= 2.0 ** -8 * np.abs(vf[0, j, 0]).max() + 1e-3
    sl = slice(128 * qb0, 128 * qb0 + 128)
    assert np.array_equal(O2[0, sl], O3[0, sl])


def test_cfg2_480p_sampled_blocks_full_size():
    # full 480p shape in the launch configuration bench.py times; oracle on sampled (h, qb) items
    cfg = W.CFG2
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    # all 40 heads x 8 query blocks each (first and last always): 320 of the 10 240 items
    items = stratified_items(cfg.H, cfg.nq, 8, seed=0)
    compare(cfg, Q, K, V, bm, items)


def test_cfg4_720p_stress_rows_sampled_blocks():
    cfg = W.scaled(W.CFG4, H=4)
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    items = stratified_items(cfg.H, cfg.nq, 6, seed=1)       # 24 of the 2364 items of these four heads
    compare(cfg, Q, K, V, bm, items, stress=True)


def test_density_sweep_one_head():
    cfg = W.scaled(W.CFG2, H=1, frames=5)
    Q, K, V = W.qkv_bits(cfg)
    for rho in (0.05, 0.10, 0.50, 1.0):
        bm = W.layer_mask(cfg, density=rho)
        items = sample_items(1, cfg.nq, 3, seed=int(rho * 100), always=[(0, 0, cfg.nq - 1)])
        compare(cfg, Q, K, V, bm, items)


def _fp16_inputs(cfg, seed):
    g = np.random.default_rng(seed)
    return tuple(g.standard_normal((cfg.B, cfg.N, cfg.H, cfg.d)).astype(np.float16) for _ in range(3))


@pytest.mark.parametrize("cfg,n_items", [(W.CFG1, None), (W.scaled(W.CFG2, H=2), 6)], ids=["cfg1", "480p-2heads"])
def test_fp16_path_matches_oracle(cfg, n_items):
    # dtype CHORUS_FP16 (the non-quantised path is fp16): fp16 Q/K/V, fp16 O
    Q, K, V = _fp16_inputs(cfg, 77)
    bm = W.layer_mask(cfg)
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    t = lambda x: torch.from_numpy(x).to("cuda:0")
    O = B.chorus_block_sparse_attn_fwd(t(Q), t(K), t(V), rp, ci, cfg.scale)
    torch.cuda.synchronize()
    assert O.dtype == torch.float16
    O = O.float().cpu().numpy().astype(np.float64)
    items = all_items(cfg.H, cfg.nq) if n_items is None else sample_items(cfg.H, cfg.nq, n_items, seed=3,
                                                                          always=[(0, cfg.H - 1, cfg.nq - 1)])
    ref = oracle_items(Q, K, V, bm, cfg.scale, items)
    mx, mean, relfro, _ = err_stats(gather_items(O, items, cfg.N), ref)
    assert mx <= BF16_MAX and mean <= BF16_MEAN, (mx, mean)
    assert mx <= BF16_MAX_TIGHT and relfro <= BF16_RELFRO, (mx, relfro)


def test_tail_probe_padded_allocation_does_not_leak():
    # K / V live in an allocation padded beyond N whose extra rows hold huge
    # values and NaNs; the kernel sees N through the shape only.  Nothing of the padding may leak:
    # the result must be bit-identical to the run on an unpadded copy.
    cfg = W.scaled(W.CFG2, H=2, frames=2)            # N = 3120: last key block 48 keys, last q block 48 rows
    Q, K, V = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    rp, ci = B.chorus_mask_to_index(dmask(bm[None]), cfg.nk)
    q, k, v = dbf16(Q), dbf16(K), dbf16(V)
    O_ref = B.chorus_block_sparse_attn_fwd(q, k, v, rp, ci, cfg.scale)
    pad = 256
    def padded(t, fill):
        buf = torch.full((1, cfg.N + pad, cfg.H, cfg.d), fill, dtype=torch.bfloat16, device=t.device)
        buf[:, : cfg.N] = t
        return buf[:, : cfg.N]                        # a view: same strides, the padding sits right behind it
    O_pad = B.chorus_block_sparse_attn_fwd(padded(q, 3e4), padded(k, float("nan")), padded(v, -3e38), rp, ci,
                                           cfg.scale)
    torch.cuda.synchronize()
    assert not torch.isnan(O_pad.float()).any()
    assert torch.equal(O_ref, O_pad)
