"""Shared helpers of the GPU parity tests (they call the CUDA path through the C ABI binding and
compare with the oracle on the same seeded input bytes)."""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2606_25040_b200 import binding as B
from paper_2606_25040_b200 import workloads as W

# BASELINE.json north_star tolerances
BF16_MAX, BF16_MEAN = 2e-2, 2e-3
FP8_MAX, FP8_COS = 8e-2, 0.995
# tighter internal gates: bf16 output rounding is ~2^-9 |O|
BF16_MAX_TIGHT, BF16_RELFRO = 6e-3, 5e-3


def dev():
    return torch.device("cuda:0")


def dmask(bm: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(bm).view(np.int32)).to(dev())


def dbf16(bits: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).to(dev())


def gpu_attention(Qb, Kb, Vb, bm_layer, nk, scale):
    """bf16 path through the ABI: decode then attention.  Returns float64 numpy [B][N][H][d]."""
    rp, ci = B.chorus_mask_to_index(dmask(bm_layer[None]), nk)
    O = B.chorus_block_sparse_attn_fwd(dbf16(Qb), dbf16(Kb), dbf16(Vb), rp, ci, scale)
    torch.cuda.synchronize()
    return O.float().cpu().numpy().astype(np.float64)


def oracle_items(Q, K, V, bm_layer, scale, items, fp8_scales=None):
    return oracle.block_sparse_attn(Q, K, V, bm_layer, scale, items=np.asarray(items, np.int32),
                                    fp8_scales=fp8_scales)


def gather_items(O, items, N):
    """dense [1][N][H][d] -> [n_items][128][d] (rows beyond N zero)."""
    out = np.zeros((len(items), 128, O.shape[3]))
    for t, (b, h, qb) in enumerate(items):
        lo, hi = qb * 128, min(N, qb * 128 + 128)
        out[t, : hi - lo] = O[b, lo:hi, h]
    return out


def all_items(H, nq):
    return [(0, h, qb) for h in range(H) for qb in range(nq)]


def sample_items(H, nq, n, seed, always=()):
    g = np.random.default_rng(seed)
    picks = {(0, int(h), int(q)) for h, q in zip(g.integers(0, H, n), g.integers(0, nq, n))}
    picks |= set(always)
    return sorted(picks)


def stratified_items(H, nq, per_head, seed):
    """per_head (head, query-block) items in EVERY head: the first and the last (ragged) query block always,
    the rest drawn without replacement."""
    g = np.random.default_rng(seed)
    out = []
    for h in range(H):
        mid = g.choice(np.arange(1, nq - 1), size=min(per_head - 2, max(nq - 2, 0)), replace=False) if nq > 2 else []
        out += [(0, h, 0)] + [(0, h, int(q)) for q in sorted(mid)] + ([(0, h, nq - 1)] if nq > 1 else [])
    return out


def report(name, **kv):
    """Append measured parity figures to gpurun_out/parity_report.jsonl (scratch; the figures that matter are
    quoted in DESIGN.md section 5) and print them."""
    import json
    import os
    d = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    os.makedirs(d, exist_ok=True)
    line = json.dumps({"test": name, **kv})
    print(line)
    with open(os.path.join(d, "parity_report.jsonl"), "a") as f:
        f.write(line + "\n")


def err_stats(got, ref):
    e = np.abs(got - ref)
    relfro = np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-30)
    cos = float((got * ref).sum() / max(np.linalg.norm(got) * np.linalg.norm(ref), 1e-30))
    return float(e.max()), float(e.mean()), float(relfro), cos
