"""Pins for oracle.block_sparse_attn.  CPU only; every reference routine here is
independent of oracle/ (numpy fp64 / long double in tests/helpers.py, closed forms, a hand-derived
golden fixture)."""
import os

import numpy as np
import pytest

import oracle
from helpers import (BK, BQ, bits_to_f64, brute_force_masked_attention,
                     dense_softmax_attention, random_keep, random_qkv_bits)
from paper_2606_25040_b200 import workloads as W

SCALE = 1.0 / np.sqrt(128.0)
HERE = os.path.dirname(os.path.abspath(__file__))


def run_oracle(Q, K, V, keep, scale=SCALE, **kw):
    N, H = Q.shape[1], Q.shape[2]
    nq = (N + BQ - 1) // BQ
    items = np.array([(0, h, qb) for h in range(H) for qb in range(nq)], np.int32)
    out = oracle.block_sparse_attn(Q, K, V, W.pack_bits(keep), scale, items=items, **kw)
    if isinstance(out, tuple):
        return oracle.scatter_items(out[0], items, N, H), out[1]
    return oracle.scatter_items(out, items, N, H)


def test_full_mask_equals_dense_attention():
    N, H = 320, 2                      # nq = 3 (ragged: 64 rows), nk = 5
    Q, K, V = random_qkv_bits(N, H, seed=1)
    keep = np.ones((H, 3, 5), bool)
    O = run_oracle(Q, K, V, keep)
    for h in range(H):
        ref = dense_softmax_attention(bits_to_f64(Q[0, :, h]), bits_to_f64(K[0, :, h]),
                                      bits_to_f64(V[0, :, h]), SCALE)
        np.testing.assert_allclose(O[0, :, h], ref, rtol=0, atol=1e-12)


def test_diagonal_mask_equals_per_window_local_attention():
    # reading R4: the diagonal of query block qb is key blocks {2qb, 2qb+1} = its own 128 tokens
    N, H = 512, 1
    Q, K, V = random_qkv_bits(N, H, seed=2)
    keep = np.zeros((H, 4, 8), bool)
    for qb in range(4):
        keep[:, qb, 2 * qb] = keep[:, qb, 2 * qb + 1] = True
    O = run_oracle(Q, K, V, keep)
    q, k, v = (bits_to_f64(x[0, :, 0]) for x in (Q, K, V))
    for qb in range(4):
        sl = slice(128 * qb, 128 * qb + 128)
        np.testing.assert_allclose(O[0, sl, 0], dense_softmax_attention(q[sl], k[sl], v[sl], SCALE),
                                   rtol=0, atol=1e-12)


def test_single_kept_block_equals_that_blocks_attention():
    N, H = 384, 1
    Q, K, V = random_qkv_bits(N, H, seed=3)
    keep = np.zeros((H, 3, 6), bool)
    picks = [4, 0, 3]
    for qb, kb in enumerate(picks):
        keep[0, qb, kb] = True
    O = run_oracle(Q, K, V, keep)
    q, k, v = (bits_to_f64(x[0, :, 0]) for x in (Q, K, V))
    for qb, kb in enumerate(picks):
        qs, ks = slice(128 * qb, 128 * qb + 128), slice(64 * kb, 64 * kb + 64)
        np.testing.assert_allclose(O[0, qs, 0], dense_softmax_attention(q[qs], k[ks], v[ks], SCALE),
                                   rtol=0, atol=1e-12)


@pytest.mark.parametrize("N,seed", [(256, 0), (200, 1), (130, 2)])
def test_brute_force_tiny(N, seed):
    H = 2
    nq, nk = (N + 127) // 128, (N + 63) // 64
    Q, K, V = random_qkv_bits(N, H, seed=10 + seed)
    keep = random_keep(H, nq, nk, 0.5, seed)
    O = run_oracle(Q, K, V, keep, scale=0.3)
    for h in range(H):
        ref = brute_force_masked_attention(bits_to_f64(Q[0, :, h]), bits_to_f64(K[0, :, h]),
                                           bits_to_f64(V[0, :, h]), keep[h], 0.3, N)
        np.testing.assert_allclose(O[0, :, h], ref, rtol=0, atol=1e-12)


def test_weights_sum_to_one_and_convex_hull():
    N, H = 448, 2
    Q, K, V = random_qkv_bits(N, H, seed=4)
    keep = random_keep(H, 4, 7, 0.4, 4)
    O, ws = run_oracle(Q, K, V, keep, return_weight_sum=True)
    valid = np.zeros((H * 4, 128), bool)
    for h in range(H):
        for qb in range(4):
            valid[h * 4 + qb, : min(128, N - 128 * qb)] = True
    np.testing.assert_allclose(ws[valid], 1.0, rtol=0, atol=1e-12)
    assert np.all(ws[~valid] == 0.0)
    v = bits_to_f64(V)
    for h in range(H):
        for qb in range(4):
            toks = np.concatenate([np.arange(64 * kb, min(N, 64 * kb + 64))
                                   for kb in np.nonzero(keep[h, qb])[0]])
            lo, hi = v[0, toks, h].min(axis=0), v[0, toks, h].max(axis=0)
            rows = O[0, 128 * qb:min(N, 128 * qb + 128), h]
            assert np.all(rows >= lo - 1e-12) and np.all(rows <= hi + 1e-12)
    # V == 1 everywhere  =>  O == 1 exactly up to rounding (a dropped or doubled weight breaks it)
    ones = np.full_like(V, 0x3F80)
    O1 = run_oracle(Q, K, ones, keep)
    np.testing.assert_allclose(O1[0, :, :, :], 1.0, rtol=0, atol=1e-12)


def test_empty_row_gives_zero():
    N, H = 256, 1
    Q, K, V = random_qkv_bits(N, H, seed=5)
    keep = np.zeros((H, 2, 4), bool)
    keep[0, 1, 2] = True                     # query block 0 keeps nothing (reading R7)
    O = run_oracle(Q, K, V, keep)
    assert np.all(O[0, :128] == 0.0) and np.any(O[0, 128:] != 0.0)


def test_permutation_invariance():
    N, H = 256, 1
    Q, K, V = random_qkv_bits(N, H, seed=6)
    keep = np.array([[[1, 0, 1, 1], [0, 1, 1, 0]]], bool)
    O = run_oracle(Q, K, V, keep)
    g = np.random.default_rng(0)
    # (a) permute keys inside key block 2
    perm = np.arange(N)
    perm[128:192] = 128 + g.permutation(64)
    O2 = run_oracle(Q, K[:, perm].copy(), V[:, perm].copy(), keep)
    np.testing.assert_allclose(O2, O, rtol=0, atol=1e-13)
    # (b) permute whole key blocks together with the mask columns
    bperm = np.array([2, 0, 3, 1])
    tperm = np.concatenate([np.arange(64 * b, 64 * b + 64) for b in bperm])
    O3 = run_oracle(Q, K[:, tperm].copy(), V[:, tperm].copy(), keep[:, :, bperm])
    np.testing.assert_allclose(O3, O, rtol=0, atol=1e-13)


def test_padded_tail_equals_hand_masked_problem():
    # N = 200 (nq 2, nk 4: tail 72 rows / 8 keys) must equal dense attention over the first 200
    # keys only, whatever the mask says about the (non-existent) keys 200..255.
    N, H = 200, 1
    Q, K, V = random_qkv_bits(N, H, seed=7)
    keep = np.ones((H, 2, 4), bool)
    O = run_oracle(Q, K, V, keep)
    q, k, v = (bits_to_f64(x[0, :, 0]) for x in (Q, K, V))
    np.testing.assert_allclose(O[0, :, 0], dense_softmax_attention(q, k, v, SCALE), rtol=0, atol=1e-12)
    # the same 200 tokens inside a 256-token buffer whose extra keys are huge but masked out by
    # hand: pruning key block 3 and comparing rows that only see blocks 0..2
    keep3 = np.ones((H, 2, 4), bool)
    keep3[:, :, 3] = False
    O3 = run_oracle(Q, K, V, keep3)
    np.testing.assert_allclose(O3[0, :, 0], dense_softmax_attention(q, k[:192], v[:192], SCALE),
                               rtol=0, atol=1e-12)


def test_q_zero_probe_closed_form():
    # Q = 0 => uniform weights => O[i, c] = (# valid kept keys whose block index = c mod 128) / |J(i)|
    # with V[j, c] = 1 iff (j // 64) % 128 == c
    N, H = 1000, 1
    nq, nk = 8, 16
    Q = np.zeros((1, N, H, 128), np.uint16)
    _, K, _ = random_qkv_bits(N, H, seed=8)
    v = np.zeros((1, N, H, 128), np.float32)
    v[0, np.arange(N), 0, (np.arange(N) // 64) % 128] = 1.0
    V = W.bf16_bits_from_f32(v)
    keep = random_keep(H, nq, nk, 0.4, 8)
    keep[0, :, 15] = True                      # ragged last key block (40 valid keys)
    O = run_oracle(Q, K, V, keep)
    for qb in range(nq):
        counts = np.zeros(128)
        for kb in np.nonzero(keep[0, qb])[0]:
            counts[kb % 128] += min(64, N - 64 * kb)
        expect = counts / counts.sum()
        rows = O[0, 128 * qb:min(N, 128 * qb + 128), 0]
        np.testing.assert_allclose(rows, np.tile(expect, (rows.shape[0], 1)), rtol=0, atol=1e-14)


def test_spike_probe_and_pruned_block_has_no_influence():
    N, H = 512, 1
    Q, K, V = random_qkv_bits(N, H, seed=9)
    keep = np.ones((H, 4, 8), bool)
    keep[0, 0, 5] = False
    base = run_oracle(Q, K, V, keep)
    # huge keys/values in the pruned block 5 must not change query block 0 at all
    K2, V2 = K.copy(), V.copy()
    K2[0, 320:384] = 0x4700            # bf16 32768.0
    V2[0, 320:384] = 0x4700
    out = run_oracle(Q, K2, V2, keep)
    assert np.array_equal(out[0, :128], base[0, :128])
    assert not np.array_equal(out[0, 128:], base[0, 128:])
    # spike: make key j* align with query i so that its score dominates => O[i] = V[j*]
    i, jstar = 7, 77
    q = bits_to_f64(Q[0, i, 0])
    kspike = (60.0 / SCALE) * q / (q @ q)
    K3 = K.copy()
    K3[0, jstar, 0] = W.bf16_bits_from_f32(kspike.astype(np.float32))
    out = run_oracle(Q, K3, V, keep)
    np.testing.assert_allclose(out[0, i, 0], bits_to_f64(V[0, jstar, 0]), rtol=0, atol=1e-12)


def test_golden_two_level_closed_form():
    # hand-derived fixture, see tests/golden/attn_two_level_closed_form.txt
    N, H, d = 192, 1, 128
    q = np.zeros((1, N, H, d), np.float32); q[..., 0] = 1.0
    k = np.zeros((1, N, H, d), np.float32); k[0, :16, 0, 0] = 1.0; k[0, 128:, 0, 0] = 1.0
    v = np.zeros((1, N, H, d), np.float32)
    v[0, :16, 0, 0] = 1; v[0, 16:64, 0, 1] = 1; v[0, 64:128, 0, 2] = 1; v[0, 128:, 0, 3] = 1
    keep = np.array([[[1, 1, 0], [1, 0, 1]]], bool)
    O = run_oracle(*(W.bf16_bits_from_f32(x) for x in (q, k, v)), keep, scale=1.0)
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "attn_two_level_closed_form.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 8
    for qb, c, val in rows:
        qb, c, val = int(qb), int(c), float(val)
        blk = O[0, 128 * qb:min(N, 128 * qb + 128), 0, c]
        np.testing.assert_allclose(blk, val, rtol=0, atol=1e-14)
    assert np.all(O[0, :, 0, 4:] == 0.0)


def test_strided_layout_bhnd_matches_bnhd():
    # the ABI passes strides; [B,H,N,d] storage must give the same result as [B,N,H,d]
    N, H = 256, 2
    Q, K, V = random_qkv_bits(N, H, seed=11)
    keep = random_keep(H, 2, 4, 0.6, 11)
    O = run_oracle(Q, K, V, keep)
    tq, tk, tv = (np.ascontiguousarray(x.transpose(0, 2, 1, 3)).transpose(0, 2, 1, 3) for x in (Q, K, V))
    assert tq.strides != Q.strides
    O2 = run_oracle(tq, tk, tv, keep)
    assert np.array_equal(O, O2)


def test_row_log_sum_exp_matches_scipy():
    # full mask: lse_i = logsumexp_j(scale * q_i . k_j) over all keys (a library routine);
    # a pruned mask: the same over the retained keys only; empty row: -inf
    from scipy.special import logsumexp
    N, H, scale = 200, 2, 0.11
    Q, K, V = random_qkv_bits(N, H, seed=21)
    nq, nk = 2, 4
    q, k = bits_to_f64(Q), bits_to_f64(K)
    keep = np.ones((H, nq, nk), dtype=bool)
    keep[1, 0, 1:3] = False
    keep[1, 1, :] = False                                     # an empty query-block row
    items = np.array([(0, h, qb) for h in range(H) for qb in range(nq)], np.int32)
    _, lse = oracle.block_sparse_attn(Q, K, V, W.pack_bits(keep), scale, items=items, return_lse=True)
    for t, (_, h, qb) in enumerate(items):
        rows = range(qb * 128, min(N, qb * 128 + 128))
        cols = np.repeat(keep[h, qb], 64)[:N]
        for r, i in enumerate(rows):
            s = scale * (k[0, cols, h] @ q[0, i, h])
            want = logsumexp(s) if cols.any() else -np.inf
            assert (lse[t, r] == want) if not cols.any() else abs(lse[t, r] - want) < 1e-12
        assert np.all(np.isneginf(lse[t, len(rows):]))        # rows beyond N


def test_fp16_input_conversion_matches_numpy_for_every_bit_pattern():
    bits = np.arange(65536, dtype=np.uint16)
    want = bits.view(np.float16).astype(np.float64)
    got = np.array([oracle.f16_to_double(int(b)) for b in bits])
    nan = np.isnan(want)
    assert np.array_equal(np.isnan(got), nan) and np.array_equal(got[~nan], want[~nan])


def test_fp16_attention_equals_dense_numpy():
    # the paper's non-quantised path is fp16: same definition, fp16 input bytes
    N, H, scale = 200, 2, 0.1
    g = np.random.default_rng(4)
    Q, K, V = (g.standard_normal((1, N, H, 128)).astype(np.float16) for _ in range(3))
    full = W.pack_bits(np.ones((H, 2, 4), dtype=bool))
    items = np.array([(0, h, qb) for h in range(H) for qb in range(2)], np.int32)
    out = oracle.scatter_items(oracle.block_sparse_attn(Q, K, V, full, scale, items=items), items, N, H)
    for h in range(H):
        ref = dense_softmax_attention(Q[0, :, h].astype(np.float64), K[0, :, h].astype(np.float64),
                                      V[0, :, h].astype(np.float64), scale)
        assert np.allclose(out[0, :, h], ref, rtol=1e-12, atol=1e-14)


def test_first_frame_key_scaling_equals_dense_attention_on_scaled_keys():
    """PAPER.md:L109-114 eq. (1): K[:, 0:N0] <- beta K[:, 0:N0], Q and V unchanged.  Pinned against numpy dense
    attention on keys scaled by hand (N0 inside a key block, a non-representable beta), against a closed form
    (uniform values: O unchanged; q = 0: weights unchanged), and the degenerate cases beta = 1 and N0 = 0."""
    N, H, n0, beta = 320, 2, 100, 1.37          # n0 = 100 straddles key block 1 (64..127)
    Q, K, V = random_qkv_bits(N, H, seed=41)
    keep = np.ones((H, 3, 5), bool)
    O, lse = run_oracle(Q, K, V, keep, n_first=n0, beta=beta, return_lse=True)
    from scipy.special import logsumexp
    for h in range(H):
        q, k, v = (bits_to_f64(x[0, :, h]) for x in (Q, K, V))
        k2 = k.copy()
        k2[:n0] *= beta
        np.testing.assert_allclose(O[0, :, h], dense_softmax_attention(q, k2, v, SCALE), rtol=0, atol=1e-12)
        ref_lse = logsumexp((q @ k2.T) * SCALE, axis=1)
        got = lse.reshape(H, 3, BQ)[h].reshape(-1)[:N]
        np.testing.assert_allclose(got, ref_lse, rtol=0, atol=1e-12)
    # beta = 1 and n_first = 0 are the plain call, bit for bit
    plain = run_oracle(Q, K, V, keep)
    assert np.array_equal(run_oracle(Q, K, V, keep, n_first=n0, beta=1.0), plain)
    assert np.array_equal(run_oracle(Q, K, V, keep, n_first=0, beta=3.0), plain)
    # it moves weight TOWARDS the first frame when the scores there are positive: with K = Q = const > 0
    # every score is c; scaled columns get beta c: weight of the first n0 keys = n0 e^{beta c} / (...)
    one = np.full((1, N, 1, 128), 0x3F80, np.uint16)            # bf16 1.0
    Vb = np.zeros((1, N, 1, 128), np.uint16)
    Vb[0, :n0] = 0x3F80                                          # V = 1 on the first frame, 0 elsewhere
    O1 = run_oracle(one, one, Vb, np.ones((1, 3, 5), bool), scale=1.0 / 128.0, n_first=n0, beta=2.0)
    w = n0 * np.exp(2.0) / (n0 * np.exp(2.0) + (N - n0) * np.exp(1.0))
    np.testing.assert_allclose(O1[0, :, 0], w, rtol=1e-13)


def test_first_frame_key_scaling_only_touches_kept_first_frame_blocks():
    # a pruned first-frame block has no influence, scaled or not; a kept block beyond N0 is not scaled
    N, H, n0 = 384, 1, 128
    Q, K, V = random_qkv_bits(N, H, seed=43)
    keep = np.zeros((H, 3, 6), bool)
    keep[0, :, 3] = keep[0, :, 5] = True                         # only blocks beyond the first frame
    assert np.array_equal(run_oracle(Q, K, V, keep, n_first=n0, beta=4.0), run_oracle(Q, K, V, keep))
    keep[0, :, 1] = True                                         # one first-frame block
    a = run_oracle(Q, K, V, keep, n_first=n0, beta=4.0)
    K2 = K.copy()
    K2[0, 64:128] = (bits_to_f64(K[0, 64:128]) * 4.0).astype(np.float32).view(np.uint32).__rshift__(16).astype(np.uint16)
    np.testing.assert_allclose(a, run_oracle(Q, K2, V, keep), rtol=0, atol=1e-13)   # x4 is exact in bf16
