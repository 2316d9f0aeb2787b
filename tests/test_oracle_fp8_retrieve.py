"""Pins for oracle.quantize_fp8, the e4m3 conversions, the FP8 attention path and retrieval."""
import numpy as np
import torch

import oracle
from helpers import bits_to_f64, dense_softmax_attention, random_keep, random_qkv_bits
from paper_2606_25040_b200 import workloads as W


def test_e4m3_decode_matches_torch_for_all_codes():
    codes = np.arange(256, dtype=np.uint8)
    ref = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    mine = np.array([oracle.e4m3_to_double(int(c)) for c in codes])
    nan = np.isnan(ref)
    assert np.array_equal(nan, np.isnan(mine)) and nan.sum() == 2       # 0x7F, 0xFF
    assert np.array_equal(ref[~nan], mine[~nan])
    assert mine[0x7E] == 448.0 and mine[0x01] == 2.0 ** -9


def test_e4m3_encode_matches_torch_rne_in_range_and_saturates():
    g = np.random.default_rng(0)
    x = np.concatenate([g.uniform(-448, 448, 20000), g.normal(0, 1, 20000), g.normal(0, 0.01, 5000),
                        # exact ties between neighbouring codes
                        np.array([0.0, 1.0625, 1.1875, 3.25, 3.75, 416 + 16, 2.0 ** -10, 3 * 2.0 ** -10])
                        ]).astype(np.float32)
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    mine = np.array([oracle.float_to_e4m3(float(v)) for v in x], np.uint8)
    # +0 / -0 of tiny values: compare decoded values and codes
    assert np.array_equal(ref, mine)
    assert oracle.float_to_e4m3(1e9) == 0x7E and oracle.float_to_e4m3(-460.0) == 0xFE
    assert oracle.float_to_e4m3(463.9) == 0x7E


def test_quantize_scales_and_error_bound():
    N, H = 300, 2
    Q, K, V = random_qkv_bits(N, H, seed=20)
    q8, k8, v8, qs, ks, vs = oracle.quantize_fp8(Q, K, V)
    dec = np.vectorize(oracle.e4m3_to_double)
    for X, X8, S, kind in ((Q, q8, qs, "blk"), (K, k8, ks, "blk"), (V, v8, vs, "ch")):
        x = bits_to_f64(X)
        for h in range(H):
            if kind == "blk":
                for blk in range(3):
                    sl = slice(128 * blk, min(N, 128 * blk + 128))
                    amax = np.abs(x[0, sl, h]).max()
                    s = float(S[0, h, blk])
                    assert s * 448.0 >= amax * (1 - 1e-6) and abs(s - amax / 448.0) <= 1e-6 * s
                    deq = dec(X8[0, sl, h]) * s
                    err = np.abs(deq - x[0, sl, h])
                    normal = np.abs(x[0, sl, h]) >= s * 2.0 ** -6     # e4m3 normal range
                    assert np.all(err[normal] <= 2.0 ** -4 * np.abs(x[0, sl, h])[normal] * (1 + 1e-6))
                    assert np.all(err <= s * 2.0 ** -10 + 2.0 ** -4 * np.abs(x[0, sl, h]) + 1e-12)
            else:
                amax = np.abs(x[0, :, h]).max(axis=0)
                s = S[0, h].astype(np.float64)
                assert np.all(s * 448.0 >= amax * (1 - 1e-6))
                deq = dec(X8[0, :, h]) * s[None, :]
                assert np.all(np.abs(deq - x[0, :, h]) <= 2.0 ** -4 * np.abs(x[0, :, h]) + s * 2.0 ** -10 + 1e-12)


def test_quantize_codes_match_torch_cast_of_the_same_fp32_quotient():
    # independent library routine: torch's fp32 division + float8_e4m3fn cast (RNE)
    N, H = 256, 1
    Q, K, V = random_qkv_bits(N, H, seed=21)
    q8, k8, v8, qs, ks, vs = oracle.quantize_fp8(Q, K, V)
    x = torch.from_numpy(W.f32_from_bf16_bits(K))                    # [1][N][H][d] fp32
    for blk in range(2):
        sl = slice(128 * blk, 128 * blk + 128)
        amax = x[0, sl, 0].abs().max()
        s = torch.clamp(amax, min=1e-12) / 448.0
        assert float(s) == float(ks[0, 0, blk])
        ref = (x[0, sl, 0] / s).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
        assert np.array_equal(ref, k8[0, sl, 0])
    xv = torch.from_numpy(W.f32_from_bf16_bits(V))
    sv = torch.clamp(xv[0, :, 0].abs().amax(dim=0), min=1e-12) / 448.0
    assert np.array_equal(sv.numpy(), vs[0, 0])
    refv = (xv[0, :, 0] / sv[None, :]).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(refv, v8[0, :, 0])


def test_quantize_exact_round_trip_of_zero_and_amax():
    N, H, d = 128, 1, 128
    x = np.zeros((1, N, H, d), np.float32)
    x[0, ::3, 0, ::5] = 3.5
    x[0, 1::7, 0, 1::4] = -3.5
    X = W.bf16_bits_from_f32(x)
    q8, k8, v8, qs, ks, vs = oracle.quantize_fp8(X, X, X)
    dec = np.vectorize(oracle.e4m3_to_double)
    np.testing.assert_array_equal(dec(q8) * qs[0, 0, 0], x.astype(np.float64))
    assert set(np.unique(q8)) == {0x00, 0x7E, 0xFE}


def test_fp8_attention_is_the_same_routine_on_dequantised_values():
    N, H = 320, 2
    Q, K, V = random_qkv_bits(N, H, seed=22)
    q8, k8, v8, qs, ks, vs = oracle.quantize_fp8(Q, K, V)
    keep = random_keep(H, 3, 5, 0.6, 22)
    items = np.array([(0, h, qb) for h in range(H) for qb in range(3)], np.int32)
    out = oracle.block_sparse_attn(q8, k8, v8, W.pack_bits(keep), 0.09, items=items,
                                   fp8_scales=(qs, ks, vs))
    O = oracle.scatter_items(out, items, N, H)
    dec = np.vectorize(oracle.e4m3_to_double)
    rep = np.repeat
    for h in range(H):
        qd = dec(q8[0, :, h]) * rep(qs[0, h], 128)[:N, None]
        kd = dec(k8[0, :, h]) * rep(ks[0, h], 128)[:N, None]
        vd = dec(v8[0, :, h]) * vs[0, h][None, :]
        for qb in range(3):
            rows = slice(128 * qb, min(N, 128 * qb + 128))
            toks = np.concatenate([np.arange(64 * kb, min(N, 64 * kb + 64))
                                   for kb in np.nonzero(keep[h, qb])[0]])
            ref = dense_softmax_attention(qd[rows], kd[toks], vd[toks], 0.09)
            np.testing.assert_allclose(O[0, rows, h], ref, rtol=0, atol=1e-12)
    # and it is close to the unquantised result (sanity on the scale plumbing, not a tolerance claim)
    outb = oracle.block_sparse_attn(Q, K, V, W.pack_bits(keep), 0.09, items=items)
    assert np.abs(out - outb).max() < 0.15


def test_retrieval_planted_neighbour_and_miss():
    cfg = W.BankConfig(entries=64, dim=256)
    bank = W.embeddings(cfg)
    np.testing.assert_allclose(np.linalg.norm(bank.astype(np.float64), axis=1), 1.0, atol=1e-6)
    for target in (0, 17, 63):
        q = W.query_embedding(cfg, bank, target)
        idx, sim, hit = oracle.retrieve_top1(bank, q, cfg.tau)
        sims = bank.astype(np.float64) @ q.astype(np.float64)
        assert idx == target == int(np.argmax(sims)) and hit and abs(sim - sims[target]) < 1e-12
        assert sim > 0.9
    q = W.query_embedding(cfg, bank, None)
    idx, sim, hit = oracle.retrieve_top1(bank, q, cfg.tau)
    sims = bank.astype(np.float64) @ q.astype(np.float64)
    assert idx == int(np.argmax(sims)) and not hit and sim < cfg.tau
    # ties -> lowest index
    bank2 = np.vstack([bank[:5], bank[2:3], bank[5:]])
    idx, _, _ = oracle.retrieve_top1(bank2, bank[2], 0.4)
    assert idx == 2
