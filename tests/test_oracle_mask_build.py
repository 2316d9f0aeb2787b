"""Pins of the oracle's mask-construction functions (PAPER.md:L73, L81, L93 (2), L153; R21-R23)
against things other than the oracle itself: numpy's dense softmax, exact rational arithmetic on tiny
rows, closed forms, invariants, and a hand-worked row in tests/golden/."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from helpers import bits_to_f64, random_qkv_bits
from paper_2606_25040_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---- block mass ------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [256, 200, 333])
def test_block_mass_equals_numpy_dense_softmax_summed_per_block(N):
    H, scale = 2, 0.09
    Q, K, _ = random_qkv_bits(N, H, seed=N)
    got = oracle.block_mass(Q, K, scale)
    nq, nk = (N + 127) // 128, (N + 63) // 64
    q, k = bits_to_f64(Q), bits_to_f64(K)
    for h in range(H):
        s = scale * (q[0, :, h] @ k[0, :, h].T)
        p = np.exp(s - s.max(axis=1, keepdims=True))
        p /= p.sum(axis=1, keepdims=True)
        ref = np.zeros((nq, nk))
        for i in range(N):
            for kb in range(nk):
                ref[i // 128, kb] += p[i, kb * 64: kb * 64 + 64].sum()
        assert np.allclose(got[0, h], ref, rtol=1e-12, atol=1e-14)
        # every valid query row carries exactly one unit of mass
        rows = np.minimum(128, N - 128 * np.arange(nq))
        assert np.allclose(got[0, h].sum(axis=1), rows, rtol=1e-12)


def test_block_mass_uniform_attention_closed_form():
    # Q = 0: every key gets 1/N of every row => mass[qb][kb] = rows(qb) * keys(kb) / N
    N, H = 200, 1
    _, K, _ = random_qkv_bits(N, H, seed=1)
    Q = np.zeros_like(K)
    got = oracle.block_mass(Q, K, 1.0)[0, 0]
    rows = np.array([128, 72], dtype=np.float64)
    keys = np.array([64, 64, 64, 8], dtype=np.float64)
    assert np.allclose(got, rows[:, None] * keys[None, :] / N, rtol=1e-13)


# ---- top-p with a top-k floor ----------------------------------------------------------------------
def exact_top_p(mass_row, top_p, min_top_k):
    """The rule of DESIGN.md R22 in exact rational arithmetic (an independent restatement)."""
    nk = len(mass_row)
    q = [int(Fraction(float(m)) * 2 ** 24) for m in mass_row]          # floor for m >= 0
    order = sorted(range(nk), key=lambda k: (-q[k], k))
    total = sum(q)
    target = Fraction(top_p) * total
    n_p, acc = 0, 0
    if total > 0:
        while n_p < nk and acc < target:
            acc += q[order[n_p]]
            n_p += 1
    # the floor is DEFINED through the double product (0.1 * 70 is 7 blocks, not 8: R22)
    n_floor = min(nk, max(0, math.ceil(min_top_k * nk)))
    n = max(n_p, n_floor)
    return sorted(order[:n])


@pytest.mark.parametrize("nk", [1, 5, 31, 32, 33, 64, 70])
def test_mask_from_mass_matches_exact_rational_rule(nk):
    g = np.random.default_rng(nk)
    for top_p, k_min in ((0.95, 0.1), (0.9, 0.0), (0.5, 0.25), (1.0, 0.0), (0.0, 0.0)):
        mass = (g.random((6, nk)) ** 4).astype(np.float32)      # peaked rows
        mass[1] = 0.0                                            # a row without mass
        mass[2, : nk // 2] = mass[2, 0]                          # ties: broken by index
        bm, kept = oracle.mask_from_mass(mass, nk, top_p, k_min)
        keep = W.unpack_bits(bm, nk)
        for r in range(6):
            want = exact_top_p(mass[r], top_p, k_min)
            assert list(np.nonzero(keep[r])[0]) == want, (nk, top_p, k_min, r)
            assert kept[r] == len(want)
        # pad bits stay clear
        if nk % 32:
            assert not (bm[:, -1] >> np.uint32(nk % 32)).any()


def test_mask_from_mass_properties():
    g = np.random.default_rng(7)
    nk, p, k_min = 64, 0.9, 0.1
    mass = (g.random((50, nk)) ** 6).astype(np.float32)
    bm, kept = oracle.mask_from_mass(mass, nk, p, k_min)
    keep = W.unpack_bits(bm, nk)
    m64 = np.floor(mass.astype(np.float64) * 2 ** 24)
    for r in range(50):
        tot, inside = m64[r].sum(), m64[r][keep[r]].sum()
        assert inside >= np.ceil(p * tot)                        # reaches the mass fraction ...
        assert kept[r] >= int(np.ceil(k_min * nk))               # ... and the floor
        # every kept block is at least as heavy as every dropped one
        if keep[r].any() and (~keep[r]).any():
            assert m64[r][keep[r]].min() >= m64[r][~keep[r]].max()
        # minimality: without its lightest block the prefix is below the target (unless the floor binds)
        if kept[r] > int(np.ceil(k_min * nk)):
            assert inside - m64[r][keep[r]].min() < np.ceil(p * tot)
    # the floor alone: top_p = 0 keeps exactly ceil(k_min * nk) heaviest blocks
    bm0, kept0 = oracle.mask_from_mass(mass, nk, 0.0, 0.25)
    assert (kept0 == 16).all()
    # top_p = 1 keeps every block that has any mass
    bm1, kept1 = oracle.mask_from_mass(mass, nk, 1.0, 0.0)
    assert (kept1 == (m64 > 0).sum(axis=1)).all()


def test_mask_from_mass_golden_row():
    # tests/golden/top_p_row.txt: a row worked out by hand (see the file)
    rows = [l.split("#")[0].split() for l in open(os.path.join(GOLDEN, "top_p_row.txt"))
            if l.strip() and not l.startswith("#")]
    mass = np.array([[float(x) for x in rows[0]]], dtype=np.float32)
    top_p, k_min = float(rows[1][0]), float(rows[1][1])
    want = [int(x) for x in rows[2]]
    bm, kept = oracle.mask_from_mass(mass, mass.shape[1], top_p, k_min)
    assert list(np.nonzero(W.unpack_bits(bm, mass.shape[1])[0])[0]) == want and kept[0] == len(want)


# ---- coverage --------------------------------------------------------------------------------------
def test_coverage_matches_numpy_and_bounds():
    g = np.random.default_rng(3)
    H, nq, nk = 3, 4, 45
    mass = (g.random((H, nq, nk)) ** 3).astype(np.float32)
    keep = g.random((H, nq, nk)) < 0.3
    cov = oracle.mask_coverage(mass, W.pack_bits(keep), nk)
    ref = (mass.astype(np.float64) * keep).sum(axis=(1, 2)) / mass.astype(np.float64).sum(axis=(1, 2))
    assert np.allclose(cov, ref, rtol=1e-13)
    assert np.allclose(oracle.mask_coverage(mass, W.pack_bits(np.ones_like(keep)), nk), 1.0)
    assert np.allclose(oracle.mask_coverage(mass, W.pack_bits(np.zeros_like(keep)), nk), 0.0)
    # a top-p mask covers at least p of the (quantised) mass of every row, hence of every head
    bm, _ = oracle.mask_from_mass(mass, nk, 0.9, 0.0)
    assert (oracle.mask_coverage(mass, bm, nk) >= 0.9 - 1e-6).all()


def test_true_top_p_mask_of_a_dense_pass_end_to_end():
    # the true-top-p mask selects blocks of the dense attention until they cover p
    N, H, scale = 512, 2, 0.3
    Q, K, _ = random_qkv_bits(N, H, seed=5)
    mass = oracle.block_mass(Q, K, scale)[0].astype(np.float32)
    nk = 8
    bm, kept = oracle.mask_from_mass(mass, nk, 0.9, 0.0)
    cov = oracle.mask_coverage(mass, bm, nk)
    assert (cov >= 0.9 - 1e-6).all() and (kept <= nk).all() and (kept >= 1).all()


def test_reused_mask_coverage_grows_with_request_similarity():
    # PAPER.md:L73 (Observation 1, Fig. 4): a true-top-p mask taken from a similar request "still
    # preserves most of the target's attention mass", and "the coverage grows monotonically as the input
    # conditions of the two requests become more similar".  Synthetic stand-in: block-clustered requests
    # that share all but a fraction of their block structure (workloads.clustered_request).
    N, H, nk, scale = 1024, 2, 16, 1 / np.sqrt(128)
    Qs, Ks = W.clustered_request(N, H, 0.0, noise_seed=100)
    src_mass = oracle.block_mass(Qs, Ks, scale)[0].astype(np.float32)
    src_mask, kept = oracle.mask_from_mass(src_mass, nk, 0.9, 0.1)
    assert kept.mean() / nk < 0.5                                  # a genuinely sparse mask
    assert (oracle.mask_coverage(src_mass, src_mask, nk) >= 0.9 - 1e-6).all()
    cov = []
    for f in (0.0, 0.1, 0.25, 0.5, 1.0):
        Qt, Kt = W.clustered_request(N, H, f, noise_seed=200)
        tgt_mass = oracle.block_mass(Qt, Kt, scale)[0].astype(np.float32)
        cov.append(oracle.mask_coverage(tgt_mass, src_mask, nk).mean())
    assert cov[0] >= 0.9                                           # same scene, fresh noise: like its own mask
    assert all(a > b for a, b in zip(cov, cov[1:]))                # monotone in similarity
    assert cov[-1] < 0.7                                           # an unrelated request loses a third of the mass
