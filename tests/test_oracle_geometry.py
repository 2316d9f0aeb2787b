"""Pins for the oracle in the paper's own block geometry, 64 query rows x 128 keys (R26):
oracle.block_sparse_attn(block=(64, 128)) against numpy with a token-level keep matrix built by hand, and
oracle.mask_to_index_64x128 against a brute-force restatement and against the attention semantics it must
preserve.  CPU only; nothing here comes from the CUDA path."""
import numpy as np
import pytest

import oracle
from helpers import bits_to_f64, dense_softmax_attention, random_qkv_bits
from paper_2606_25040_b200 import workloads as W

SCALE = 1.0 / np.sqrt(128.0)


def masked_attention(q, k, v, tok_keep, scale):
    """softmax over the kept keys of each row, from a token-level bool matrix (numpy fp64)."""
    s = scale * (q @ k.T)
    s = np.where(tok_keep, s, -np.inf)
    out = np.zeros_like(q)
    for i in range(q.shape[0]):
        if tok_keep[i].any():
            p = np.exp(s[i] - s[i].max())
            out[i] = (p / p.sum()) @ v
    return out


@pytest.mark.parametrize("N,seed", [(320, 1), (200, 2), (449, 3)])
def test_attention_64x128_equals_token_level_masked_softmax(N, seed):
    H = 2
    Q, K, V = random_qkv_bits(N, H, seed=seed)
    nq64, nk128 = (N + 63) // 64, (N + 127) // 128
    g = np.random.default_rng(seed)
    keep = g.random((H, nq64, nk128)) < 0.5
    keep[0] = True                                  # head 0 dense
    keep[1, 1, :] = False                           # an empty 64-row block
    items = np.array([(0, h, qb) for h in range(H) for qb in range(nq64)], np.int32)
    out = oracle.block_sparse_attn(Q, K, V, W.pack_bits(keep), SCALE, items=items, block=(64, 128))
    assert out.shape == (len(items), 64, 128)
    for t, (_, h, qb) in enumerate(items):
        q, k, v = (bits_to_f64(x[0, :, h]) for x in (Q, K, V))
        tok = np.repeat(np.repeat(keep[h], 64, axis=0), 128, axis=1)[:N, :N]
        ref = masked_attention(q, k, v, tok, SCALE)
        lo, hi = 64 * qb, min(N, 64 * qb + 64)
        np.testing.assert_allclose(out[t, : hi - lo], ref[lo:hi], rtol=0, atol=1e-12)
        assert np.all(out[t, hi - lo:] == 0)
    # head 0 = dense attention
    np.testing.assert_allclose(out[0, :64], dense_softmax_attention(
        bits_to_f64(Q[0, :64, 0]), bits_to_f64(K[0, :, 0]), bits_to_f64(V[0, :, 0]), SCALE), rtol=0, atol=1e-12)


def brute_index(keep, N):
    """keep bool [L][H][nq64][nk128] -> (row_ptr, entries) by the definition in DESIGN.md R26."""
    L, H, nq64, nk128 = keep.shape
    rp, ent = [0], []
    for l in range(L):
        for h in range(H):
            for qb in range((N + 127) // 128):
                up = keep[l, h, 2 * qb]
                lo = keep[l, h, 2 * qb + 1] if 2 * qb + 1 < nq64 else np.zeros(nk128, bool)
                for kb in range(nk128):
                    if up[kb] or lo[kb]:
                        for t in (2 * kb, 2 * kb + 1):
                            if 64 * t < N:
                                ent.append(t | (0 if up[kb] else 1 << 30) | (0 if lo[kb] else 1 << 31))
                rp.append(len(ent))
    return np.array(rp, np.int32), np.array(ent, np.uint32)


@pytest.mark.parametrize("N", [64, 65, 128, 129, 192, 193, 320, 4200])
def test_decode_64x128_matches_brute_force_and_round_trips(N):
    L, H = 2, 3
    nq64, nk128 = (N + 63) // 64, (N + 127) // 128
    g = np.random.default_rng(N)
    keep = g.random((L, H, nq64, nk128)) < 0.4
    keep[0, 0] = True
    keep[1, 2] = False
    bm = W.pack_bits(keep)
    if nk128 % 32:
        bm[..., -1] |= np.uint32((0xFFFFFFFF << (nk128 % 32)) & 0xFFFFFFFF)    # garbage pad bits are ignored
    rp, ci = oracle.mask_to_index_64x128(bm, N)
    rp_b, ci_b = brute_index(keep, N)
    assert np.array_equal(rp, rp_b) and np.array_equal(ci, ci_b)
    # round trip: the kept (token row, key) set that the index describes is the mask's
    nq128 = (N + 127) // 128
    for l in range(L):
        for h in range(H):
            tok = np.zeros((N, N), bool)
            for qb in range(nq128):
                r = (l * H + h) * nq128 + qb
                for e in ci[rp[r]:rp[r + 1]]:
                    t = int(e & 0x3FFFFFFF)
                    ks = slice(64 * t, min(N, 64 * t + 64))
                    if not (e >> 30) & 1:
                        tok[128 * qb: min(N, 128 * qb + 64), ks] = True
                    if not (e >> 31) & 1:
                        tok[128 * qb + 64: min(N, 128 * qb + 128), ks] = True
                tiles = ci[rp[r]:rp[r + 1]] & 0x3FFFFFFF
                assert np.all(np.diff(tiles.astype(np.int64)) > 0)           # ascending, no duplicates
            ref = np.repeat(np.repeat(keep[l, h], 64, axis=0), 128, axis=1)[:N, :N]
            assert np.array_equal(tok, ref)


def test_block_mass_64x128_equals_numpy_softmax_summed_per_block():
    """oracle.block_mass(block=(64, 128)) against numpy: the dense softmax matrix summed over 64-row x 128-key
    blocks; it is also the 128 x 64 result regrouped where both geometries tile evenly."""
    N, H = 449, 2
    Q, K, _ = random_qkv_bits(N, H, seed=12)
    m = oracle.block_mass(Q, K, SCALE, block=(64, 128))
    nq64, nk128 = (N + 63) // 64, (N + 127) // 128
    assert m.shape == (1, H, nq64, nk128)
    for h in range(H):
        q, k = bits_to_f64(Q[0, :, h]), bits_to_f64(K[0, :, h])
        s = SCALE * (q @ k.T)
        p = np.exp(s - s.max(axis=1, keepdims=True))
        p /= p.sum(axis=1, keepdims=True)
        ref = np.zeros((nq64, nk128))
        for i in range(N):
            for kb in range(nk128):
                ref[i // 64, kb] += p[i, 128 * kb: 128 * kb + 128].sum()
        np.testing.assert_allclose(m[0, h], ref, rtol=0, atol=1e-12)
        np.testing.assert_allclose(m[0, h].sum(axis=1), np.minimum(64, N - 64 * np.arange(nq64)), rtol=1e-12)
    # token-level consistency of the two geometries: both sum to the same 128 x 128 super-blocks
    m2 = oracle.block_mass(Q, K, SCALE)                              # [1][H][4][8]
    a = m[0, :, : 2 * (nq64 // 2)].reshape(H, nq64 // 2, 2, nk128).sum(axis=2)
    b = np.pad(m2[0], ((0, 0), (0, 0), (0, 2 * nk128 - m2.shape[3]))).reshape(H, m2.shape[2], nk128, 2).sum(axis=3)
    np.testing.assert_allclose(a, b[:, : nq64 // 2], rtol=0, atol=1e-12)


def test_decode_64x128_golden_hand_worked_example():
    """tests/golden/decode_64x128.txt: derived by hand from the definition (R26), not by any program."""
    import os
    vals = {}
    for line in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "decode_64x128.txt")):
        if not line.startswith("#") and line.strip():
            k, *v = line.split()
            vals[k] = [int(x) for x in v]
    N = vals["N"][0]
    bm = np.array(vals["mask_rows"], np.uint32).reshape(1, 1, 4, 1)       # one word per mask row: bit kb
    rp, ci = oracle.mask_to_index_64x128(bm, N)
    assert rp.tolist() == vals["row_ptr"] and ci.tolist() == vals["col_idx"]
