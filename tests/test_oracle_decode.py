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
