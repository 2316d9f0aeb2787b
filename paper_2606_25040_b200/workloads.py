"""Seeded synthetic workloads shared by the CUDA path's tests/bench and by the oracle's tests.

This module holds NONE of the method's arithmetic: it only draws inputs (Gaussian Q/K/V rounded to
bf16, structured block masks, unit-norm embeddings) with the shapes and structure of the paper's
Wan2.2-I2V workload as fixed by BASELINE.json `configs` (DESIGN.md §4 gives the
recipe).  The inputs STAND IN for the paper's COCO-2017 / service-prompt requests, which are not
available; nothing here reproduces any dataset item.

Everything is generated on the host with numpy's counter-based Philox generator, so the same seed
gives the same bytes on every machine; both the oracle and the GPU read those bytes.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BQ, BK, HEAD_DIM = 128, 64, 128


@dataclass(frozen=True)
class AttnConfig:
    """One attention-layer workload (BASELINE.json configs[0..3])."""
    name: str
    H: int
    frames: int
    hp: int          # latent patch rows per frame
    wp: int          # latent patch cols per frame
    density: float
    data_seed: int
    mask_seed: int
    band: str = "spatiotemporal"   # "fixed8" for cfg1
    stress_rows: float = 0.0       # fraction of token rows scaled x8 (cfg4)
    B: int = 1
    d: int = HEAD_DIM

    @property
    def tokens_per_frame(self) -> int:
        return self.hp * self.wp

    @property
    def N(self) -> int:
        return self.frames * self.hp * self.wp

    @property
    def nq(self) -> int:
        return (self.N + BQ - 1) // BQ

    @property
    def nk(self) -> int:
        return (self.N + BK - 1) // BK

    @property
    def words(self) -> int:
        return (self.nk + 31) // 32

    @property
    def scale(self) -> float:
        return 1.0 / float(np.sqrt(self.d))


# BASELINE.json configs[0]: tiny, 4 latent frames x 32x32, 50 % density, width-8 band.
CFG1 = AttnConfig("cfg1_tiny", H=2, frames=4, hp=32, wp=32, density=0.50, data_seed=0,
                  mask_seed=1000, band="fixed8")
# configs[1]/[2]: Wan-2.2-14B-shaped 480p layer, 21 x 30 x 52 = 32760 tokens, 25 % density.
CFG2 = AttnConfig("cfg2_480p", H=40, frames=21, hp=30, wp=52, density=0.25, data_seed=1,
                  mask_seed=2000)
# configs[3]: 720p layer, 21 x 45 x 80 = 75600 tokens, 15 % density, 1 % of rows x8.
CFG4 = AttnConfig("cfg4_720p", H=40, frames=21, hp=45, wp=80, density=0.15, data_seed=2,
                  mask_seed=3000, stress_rows=0.01)


def scaled(cfg: AttnConfig, **kw) -> AttnConfig:
    """A copy of cfg with some fields replaced (fewer heads / frames for fast tests)."""
    d = {f: getattr(cfg, f) for f in cfg.__dataclass_fields__}
    d.update(kw)
    return AttnConfig(**d)


# ------------------------------------------------------------------------------------------------
# Q / K / V
# ------------------------------------------------------------------------------------------------
def _rng(seed: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def bf16_bits_from_f32(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit patterns (uint16), round-to-nearest-even.  Input generation only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounded = u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))
    return (rounded >> np.uint32(16)).astype(np.uint16)


def f32_from_bf16_bits(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def qkv_bits(cfg: AttnConfig, heads: int | None = None):
    """Q, K, V ~ N(0,1) as bf16 bit patterns, uint16 [B][N][H][d]; cfg.stress_rows of the token
    rows of each tensor and head are multiplied by 8 before rounding (BASELINE.json configs[3])."""
    H = cfg.H if heads is None else heads
    out = []
    for t in range(3):
        g = _rng(cfg.data_seed, t)
        x = g.standard_normal((cfg.B, cfg.N, H, cfg.d), dtype=np.float32)
        if cfg.stress_rows > 0:
            sel = _rng(cfg.data_seed, 10 + t).random((cfg.B, cfg.N, H)) < cfg.stress_rows
            x *= np.where(sel, np.float32(8.0), np.float32(1.0))[..., None]
        out.append(bf16_bits_from_f32(x))
    return tuple(out)


# ------------------------------------------------------------------------------------------------
# block masks
# ------------------------------------------------------------------------------------------------
def pack_bits(keep: np.ndarray) -> np.ndarray:
    """bool [..., nk] -> uint32 [..., ceil(nk/32)], key block kb = bit (kb & 31) of word kb >> 5."""
    nk = keep.shape[-1]
    words = (nk + 31) // 32
    padded = np.zeros(keep.shape[:-1] + (words * 32,), dtype=np.uint8)
    padded[..., :nk] = keep
    by = np.packbits(padded, axis=-1, bitorder="little")
    return np.ascontiguousarray(by).view(np.uint32).reshape(keep.shape[:-1] + (words,))


def unpack_bits(words: np.ndarray, nk: int) -> np.ndarray:
    by = np.ascontiguousarray(words, dtype=np.uint32).view(np.uint8)
    bits = np.unpackbits(by, axis=-1, bitorder="little")
    return bits[..., :nk].astype(bool)


def head_mask(nq: int, nk: int, tokens_per_frame: int, density: float, seed: int,
              band: str = "spatiotemporal", jitter: bool = False) -> np.ndarray:
    """Keep-matrix bool [nq][nk] of one head (DESIGN.md §4 mask recipe).

    Per-row budget b = max(2, round(density*nk)) kept blocks, chosen in this priority order:
    the diagonal {2qb, 2qb+1}; all frame-0 key blocks; a band (cfg1: the fixed width-8 band
    2qb-3..2qb+4; otherwise same-position blocks of the same and adjacent frames, nearest first)
    up to a per-head structural quota; then a seeded uniform random fill.  density >= 1 gives the
    all-ones mask.  Every row has exactly b kept blocks unless jitter is set.
    """
    if density >= 1.0:
        return np.ones((nq, nk), dtype=bool)
    g = _rng(seed, 0)
    b = max(2, int(round(density * nk)))
    sigma = g.uniform(0.5, 0.8)
    qb = np.arange(nq)[:, None]
    kb = np.arange(nk)[None, :]
    INF = np.float64(1e18)
    score = np.full((nq, nk), INF)
    # band candidates (lowest priority of the structural part)
    if band == "fixed8":
        inband = (kb >= 2 * qb - 3) & (kb <= 2 * qb + 4)
        score = np.where(inband, 2.0 + np.abs(kb - (2 * qb + 0.5)) / nk, score)
        n_f0 = (tokens_per_frame + BK - 1) // BK
        quota_min = None
    else:
        n_f0 = (tokens_per_frame + BK - 1) // BK
        order = 0
        rows = np.arange(nq)
        max_delta = b  # more than enough candidates
        for di in range(2 * max_delta + 1):
            delta = 0 if di == 0 else ((di + 1) // 2) * (-1 if di % 2 == 1 else 1)
            for df in (0, -1, 1):
                cand = 2 * rows + int(round(df * tokens_per_frame / BK)) + delta
                ok = (cand >= 0) & (cand < nk)
                r_ok, c_ok = rows[ok], cand[ok]
                np.minimum.at(score, (r_ok, c_ok), 2.0 + order)
                order += 1
        quota_min = None
    # frame-0 blocks (all of them; truncated from the high end only if the budget is too small)
    f0 = kb < n_f0
    score = np.where(f0, 1.0 + kb / (nk + 1.0), score)
    # diagonal
    diag = (kb == 2 * qb) | (kb == 2 * qb + 1)
    score = np.where(diag, 0.0, score)

    n_forced = (diag | f0).sum(axis=1)                       # |D u F0| per row
    if band == "fixed8":
        quota = np.minimum(b, (score < INF).sum(axis=1))     # whole band + frame 0 + diagonal
    else:
        quota = np.minimum(b, np.maximum(int(round(sigma * b)), n_forced))
    row_budget = np.full(nq, b)
    if jitter:
        row_budget = np.clip(np.round(b * g.uniform(0.7, 1.3, size=nq)).astype(int), 2, nk)
        quota = np.minimum(quota, row_budget)
    rank = np.argsort(np.argsort(score, axis=1, kind="stable"), axis=1, kind="stable")
    structural = (rank < quota[:, None]) & (score < INF)
    rnd = g.random((nq, nk))
    final = np.where(structural, -1.0, rnd)
    frank = np.argsort(np.argsort(final, axis=1, kind="stable"), axis=1, kind="stable")
    keep = frank < row_budget[:, None]
    return keep


def layer_mask(cfg: AttnConfig, heads: int | None = None, density: float | None = None,
               seed: int | None = None, jitter: bool = False) -> np.ndarray:
    """Packed uint32 [H][nq][words] block mask of one layer; the pattern differs per head."""
    H = cfg.H if heads is None else heads
    rho = cfg.density if density is None else density
    s0 = cfg.mask_seed if seed is None else seed
    keep = np.stack([head_mask(cfg.nq, cfg.nk, cfg.tokens_per_frame, rho, s0 + h, cfg.band, jitter)
                     for h in range(H)])
    return pack_bits(keep)


def mask_density(words: np.ndarray, nk: int) -> float:
    keep = unpack_bits(words, nk)
    return float(keep.mean())


# ------------------------------------------------------------------------------------------------
# cfg5: mask bank + request embeddings (BASELINE.json configs[4])
# ------------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class BankConfig:
    name: str = "cfg5_reuse_step"
    entries: int = 1024
    dim: int = 4096
    layers: int = 40
    attn: AttnConfig = field(default_factory=lambda: CFG2)
    bank_seed: int = 4
    query_seed: int = 5
    tau: float = 0.4
    rho_lo: float = 0.10
    rho_hi: float = 0.40


CFG5 = BankConfig()


def embeddings(cfg: BankConfig) -> np.ndarray:
    """Unit-norm fp32 request embeddings [entries][dim]."""
    e = _rng(cfg.bank_seed, 0).standard_normal((cfg.entries, cfg.dim), dtype=np.float32)
    e /= np.linalg.norm(e.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
    return np.ascontiguousarray(e, dtype=np.float32)


def query_embedding(cfg: BankConfig, bank: np.ndarray, target: int | None, noise: float = 0.3):
    """A request embedding close to bank[target] (cos ~ 0.96), or an unrelated one (target=None,
    max cos ~ 0.06 < tau: the cache-miss case of PAPER.md:L87)."""
    g = _rng(cfg.query_seed, 0 if target is None else 1 + target)
    v = g.standard_normal(cfg.dim, dtype=np.float32)
    if target is not None:
        v = bank[target] + np.float32(noise) * v / np.float32(np.sqrt(cfg.dim))
    v = v / np.float32(np.linalg.norm(v.astype(np.float64)))
    return np.ascontiguousarray(v, dtype=np.float32)


def bank_entry_densities(cfg: BankConfig, entry: int, layers: int | None = None,
                         heads: int | None = None) -> np.ndarray:
    """Per-(layer, head) density ~ U[rho_lo, rho_hi] of one stored mask set (the
    sparsity level differs per head)."""
    L = cfg.layers if layers is None else layers
    H = cfg.attn.H if heads is None else heads
    return _rng(cfg.bank_seed, 1000 + entry).uniform(cfg.rho_lo, cfg.rho_hi, size=(L, H))


def bank_entry_masks(cfg: BankConfig, entry: int, layers: int | None = None,
                     heads: int | None = None) -> np.ndarray:
    """Structured mask set of one bank entry: uint32 [L][H][nq][words]."""
    L = cfg.layers if layers is None else layers
    H = cfg.attn.H if heads is None else heads
    rho = bank_entry_densities(cfg, entry, L, H)
    a = cfg.attn
    out = np.zeros((L, H, a.nq, a.words), dtype=np.uint32)
    for l in range(L):
        for h in range(H):
            keep = head_mask(a.nq, a.nk, a.tokens_per_frame, float(rho[l, h]),
                             cfg.bank_seed * 1_000_003 + entry * 4099 + l * 64 + h, a.band)
            out[l, h] = pack_bits(keep)
    return out


def hash_fill_masks(shape_rows: int, words: int, nk: int, density: float, seed: int) -> np.ndarray:
    """Unstructured Bernoulli(density) mask rows (decoy bank entries), diagonal bit not forced."""
    g = _rng(seed, 7)
    keep = g.random((shape_rows, nk)) < density
    return pack_bits(keep).reshape(shape_rows, words)


# ------------------------------------------------------------------------------------------------
# "similar requests" for the mask-construction path (Observation 1 / Fig. 4)
# ------------------------------------------------------------------------------------------------
def clustered_request(N: int, H: int, reassigned: float, noise_seed: int, structure_seed: int = 1,
                      clusters: int = 8, strength: float = 0.7, d: int = 128):
    """Q, K bf16 bits [1][N][H][d] whose attention is block-structured: every 64-token block belongs to
    one of `clusters` clusters (per head), and a token's q and k are strength * its cluster's centre
    plus N(0,1) noise, so that a query attends mostly to the key blocks of its own cluster.  Two
    requests with the same structure_seed share centres and block assignment except for a fraction
    `reassigned` of the blocks, which is what "similarity" means here: reassigned = 0 is the same
    scene with fresh noise, 1 an unrelated one.  Stands in for the paper's similar I2V requests; no
    arithmetic of the method lives here."""
    g = _rng(structure_seed, 11)
    centres = g.standard_normal((H, clusters, d))
    assign = g.integers(0, clusters, size=(H, (N + 63) // 64))
    g2 = _rng(noise_seed, 12)
    flip = g2.random(assign.shape) < reassigned
    assign = np.where(flip, g2.integers(0, clusters, size=assign.shape), assign)
    Q = np.empty((1, N, H, d), dtype=np.float32)
    K = np.empty((1, N, H, d), dtype=np.float32)
    for h in range(H):
        c = np.repeat(assign[h], 64)[:N]
        Q[0, :, h] = strength * centres[h, c] + g2.standard_normal((N, d))
        K[0, :, h] = strength * centres[h, c] + g2.standard_normal((N, d))
    return bf16_bits_from_f32(Q), bf16_bits_from_f32(K)
