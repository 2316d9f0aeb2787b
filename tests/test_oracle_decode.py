"""Pins for oracle.mask_to_index (SURVEY §8 c-4 'decode').  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2606_25040_b200 import workloads as W


def brute_force(bm, nk):
    """Per-bit Python loop written independently of the oracle."""
    L, H, nq, words = bm.shape
    row_ptr, cols = [0], []
    for l in range(L):
        for h in range(H):
            for qb in range(nq):
                for kb in range(nk):
                    w = int(bm[l, h, qb, kb // 32])
                    if (w >> (kb % 32)) & 1:
                        cols.append(kb)
                row_ptr.append(len(cols))
    return np.array(row_ptr, np.int32), np.array(cols, np.int32)


@pytest.mark.parametrize("nk", [1, 31, 32, 33, 64, 65, 100])
def test_brute_force_and_pad_bits(nk):
    g = np.random.default_rng(nk)
    L, H, nq = 2, 3, 5
    words = (nk + 31) // 32
    bm = g.integers(0, 2**32, size=(L, H, nq, words), dtype=np.uint64).astype(np.uint32)  # garbage pad bits
    rp, ci = oracle.mask_to_index(bm, nk)
    rp2, ci2 = brute_force(bm, nk)
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
    # total popcount over valid bits, computed a third way
    assert rp[-1] == W.unpack_bits(bm, nk).sum()
    # pad bits are ignored: clearing them changes nothing
    clean = W.pack_bits(W.unpack_bits(bm, nk))
    rp3, ci3 = oracle.mask_to_index(clean, nk)
    assert np.array_equal(rp, rp3) and np.array_equal(ci, ci3)


def test_round_trip_and_ascending():
    nk = 1182  # cfg4's key-block count: 37 words, 30 valid bits in the last one
    g = np.random.default_rng(7)
    keep = g.random((1, 2, 9, nk)) < 0.15
    bm = W.pack_bits(keep)
    rp, ci = oracle.mask_to_index(bm, nk)
    rebuilt = np.zeros_like(keep).reshape(-1, nk)
    for r in range(rebuilt.shape[0]):
        row = ci[rp[r]:rp[r + 1]]
        assert np.all(np.diff(row) > 0)           # strictly ascending => unique output
        rebuilt[r, row] = True
    assert np.array_equal(rebuilt.reshape(keep.shape), keep)


def test_full_and_empty():
    nk, nq = 70, 4
    full = np.full((1, 1, nq, 3), 0xFFFFFFFF, dtype=np.uint32)
    rp, ci = oracle.mask_to_index(full, nk)
    assert np.array_equal(rp, np.arange(nq + 1) * nk)
    assert np.array_equal(ci.reshape(nq, nk), np.tile(np.arange(nk), (nq, 1)))
    empty = np.zeros((1, 1, nq, 3), dtype=np.uint32)
    rp, ci = oracle.mask_to_index(empty, nk)
    assert np.all(rp == 0) and ci.size == 0


def test_count_only_matches():
    cfg = W.CFG1
    bm = W.layer_mask(cfg)[None]
    rp, ci = oracle.mask_to_index(bm, cfg.nk)
    rp2, none = oracle.mask_to_index(bm, cfg.nk, count_only=True)
    assert none is None and np.array_equal(rp, rp2)
    assert rp[-1] == cfg.H * cfg.nq * 32          # cfg1: exactly 32 kept blocks per row


def test_visit_refresh_every_pair_visited_once_per_group():
    # PAPER.md:L93 (1): after the refresh every (h, q, k) pair is touched at least once per
    # group of 8 layers, and only the last layer of each complete group is changed.
    nk, nq, H, L = 45, 3, 2, 19
    g = np.random.default_rng(3)
    keep = g.random((L, H, nq, nk)) < 0.2
    bm = W.pack_bits(keep)
    out = W.unpack_bits(oracle.visit_refresh(bm, nk, group=8), nk)
    for grp in range(L // 8):
        sl = slice(8 * grp, 8 * grp + 8)
        assert out[sl].any(axis=0).all()
        assert np.array_equal(out[8 * grp:8 * grp + 7], keep[8 * grp:8 * grp + 7])
        expect_last = keep[8 * grp + 7] | ~keep[8 * grp:8 * grp + 7].any(axis=0)
        assert np.array_equal(out[8 * grp + 7], expect_last)
    assert np.array_equal(out[16:], keep[16:])    # trailing partial group untouched


# ---- 16-bit entries -------------------------------------------------------------------
@pytest.mark.parametrize("nk", [1, 33, 100, 512, 1182, 65536])
def test_u16_form_against_an_independent_loop_and_the_32_bit_form(nk):
    g = np.random.default_rng(nk + 1)
    L, H, nq = (1, 1, 2) if nk == 65536 else (2, 2, 3)
    words = (nk + 31) // 32
    bm = g.integers(0, 2**32, size=(L, H, nq, words), dtype=np.uint64).astype(np.uint32)  # garbage pad bits
    bm &= g.integers(0, 2**32, size=bm.shape, dtype=np.uint64).astype(np.uint32)
    rp, ci = oracle.mask_to_index_u16(bm, nk)
    assert ci.dtype == np.uint16
    # independent per-bit loop (numpy unpack, written here)
    keep = W.unpack_bits(bm, nk).reshape(-1, nk)
    want = np.concatenate([np.nonzero(r)[0] for r in keep]) if keep.any() else np.zeros(0, np.int64)
    assert np.array_equal(ci.astype(np.int64), want)
    assert np.array_equal(rp, np.concatenate([[0], np.cumsum(keep.sum(axis=1))]).astype(np.int32))
    rp32, ci32 = oracle.mask_to_index(bm, nk)
    assert np.array_equal(rp, rp32) and np.array_equal(ci.astype(np.int32), ci32)
    if nk == 65536:
        assert int(ci.max()) <= 65535 and keep[:, 65535].any() == (65535 in ci)


def test_u16_forms_refuse_what_does_not_fit():
    bm = np.zeros((1, 1, 1, (65537 + 31) // 32), np.uint32)
    with pytest.raises(ValueError):
        oracle.mask_to_index_u16(bm, 65537)
    N = 64 * 16385                                      # 16385 tiles: one more than 14 bits hold
    bm64 = np.zeros((1, 1, (N + 63) // 64, ((N + 127) // 128 + 31) // 32), np.uint32)
    with pytest.raises(ValueError):
        oracle.mask_to_index_64x128_u16(bm64, N)


@pytest.mark.parametrize("N", [64, 200, 1000, 4680])
def test_u16_form_of_the_64x128_decode(N):
    g = np.random.default_rng(N)
    nq64, nk128 = (N + 63) // 64, (N + 127) // 128
    keep = g.random((1, 2, nq64, nk128)) < 0.4
    bm = W.pack_bits(keep)
    rp, ci = oracle.mask_to_index_64x128_u16(bm, N)
    rp32, ci32 = oracle.mask_to_index_64x128(bm, N)
    assert np.array_equal(rp, rp32)
    # same tiles, flags moved from bits 30 / 31 to bits 14 / 15
    assert np.array_equal(ci & 0x3FFF, (ci32 & 0x3FFFFFFF).astype(np.uint16))
    assert np.array_equal((ci >> 14) & 1, ((ci32 >> 30) & 1).astype(np.uint16))
    assert np.array_equal((ci >> 15) & 1, ((ci32 >> 31) & 1).astype(np.uint16))
    # and an independent statement of one row: upper / lower mask rows of 128-row block 0 of head 1
    up, lo = keep[0, 1, 0], (keep[0, 1, 1] if nq64 > 1 else np.zeros(nk128, bool))
    row = ci[rp[(N + 127) // 128]: rp[(N + 127) // 128 + 1]]
    want = [t | (0 if up[t // 2] else 1 << 14) | (0 if lo[t // 2] else 1 << 15)
            for t in range((N + 63) // 64) if up[t // 2] or lo[t // 2]]
    assert list(map(int, row)) == want
