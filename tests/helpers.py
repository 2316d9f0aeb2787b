"""Independent reference routines used ONLY to pin the oracle (numpy, fp64 / long double).

Nothing here calls oracle/ or the CUDA path; these are the textbook definitions the oracle's
special cases must reduce to.
"""
from __future__ import annotations

import numpy as np

from paper_2606_25040_b200 import workloads as W

BQ, BK = 128, 64


def bits_to_f64(bits: np.ndarray) -> np.ndarray:
    return W.f32_from_bf16_bits(bits).astype(np.float64)


def dense_softmax_attention(q, k, v, scale):
    """Textbook softmax(q k^T * scale) v in fp64 (no mask logic at all)."""
    s = scale * (q @ k.T)
    s = s - s.max(axis=-1, keepdims=True)
    p = np.exp(s)
    return (p / p.sum(axis=-1, keepdims=True)) @ v


def brute_force_masked_attention(q, k, v, keep_blocks, scale, N):
    """Second, deliberately different formulation: materialise the full N x N score matrix in
    long double with -inf at masked positions, two-pass softmax.  keep_blocks: bool [nq][nk]."""
    ld = np.longdouble
    s = (scale * (q.astype(ld) @ k.astype(ld).T)).astype(ld)
    tok_keep = np.repeat(np.repeat(keep_blocks, BQ, axis=0), BK, axis=1)[:N, :N]
    s = np.where(tok_keep, s, -np.inf)
    out = np.zeros((N, v.shape[1]), dtype=ld)
    for i in range(N):
        if not tok_keep[i].any():
            continue
        m = s[i].max()
        p = np.exp(s[i] - m)
        out[i] = (p[:, None] * v.astype(ld)).sum(axis=0) / p.sum()
    return out.astype(np.float64)


def random_qkv_bits(N, H, d=128, seed=0, B=1):
    g = np.random.default_rng(seed)
    return tuple(W.bf16_bits_from_f32(g.standard_normal((B, N, H, d)).astype(np.float32))
                 for _ in range(3))


def random_keep(H, nq, nk, density, seed, force_diag=True):
    g = np.random.default_rng(seed)
    keep = g.random((H, nq, nk)) < density
    if force_diag:
        for qb in range(nq):
            keep[:, qb, min(2 * qb, nk - 1)] = True
    return keep
