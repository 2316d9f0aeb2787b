"""Timing of the mask-construction calls (the historical request's side) on a 480p layer.

    python -m paper_2606_25040_b200.bench_mask_build [--heads H] [--iters K]

Prints one JSON line: chorus_block_mass (two passes, and one pass with the attention kernel's LSE),
chorus_mask_from_mass, chorus_mask_coverage, with the MUFU roofline of the block-mass kernel
(2 N^2 H exponentials in two passes, N^2 H in one; peak = SMs x 16 /clk x SM clock).
bench.py stays the headline benchmark; this one covers the "next" row f-2.
"""
from __future__ import annotations

import argparse
import json
import statistics

import torch

from . import binding as B
from . import workloads as W


def _time(fn, iters):
    fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(iters):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return statistics.median(ts)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--heads", type=int, default=40)
    ap.add_argument("--iters", type=int, default=5)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device (no CPU fallback)")
    dev = torch.device("cuda:0")
    cfg = W.scaled(W.CFG2, H=args.heads)
    g = torch.Generator(device=dev)
    g.manual_seed(0)
    Q, K, V = (torch.randn((1, cfg.N, cfg.H, cfg.d), device=dev, generator=g).to(torch.bfloat16) for _ in range(3))
    # the dense attention call of the historical request, with its LSE output
    full = torch.full((1, cfg.H, cfg.nq, cfg.words), -1, dtype=torch.int32, device=dev)
    rp, ci = B.chorus_mask_to_index(full, cfg.nk)
    lse = torch.empty((1, cfg.H, cfg.N), dtype=torch.float32, device=dev)
    O = torch.empty_like(Q)
    mass = torch.empty((1, cfg.H, cfg.nq, cfg.nk), dtype=torch.float32, device=dev)
    # two rounds, the second one reported: the first kernels of a process run at boost clocks
    for _ in range(2):
        t_attn = _time(lambda: B.chorus_block_sparse_attn_fwd(Q, K, V, rp, ci, cfg.scale, O=O, lse=lse), args.iters)
        t2 = _time(lambda: B.chorus_block_mass(Q, K, cfg.scale, mass=mass), args.iters)
        t1 = _time(lambda: B.chorus_block_mass(Q, K, cfg.scale, mass=mass, lse=lse), args.iters)
    bm = torch.empty((cfg.H, cfg.nq, cfg.words), dtype=torch.int32, device=dev)
    kept = torch.empty((cfg.H, cfg.nq), dtype=torch.int32, device=dev)
    t_sel = _time(lambda: B.chorus_mask_from_mass(mass[0], 0.9, 0.1, bitmask=bm, kept=kept), args.iters)
    cov = torch.empty(cfg.H, dtype=torch.float32, device=dev)
    t_cov = _time(lambda: B.chorus_mask_coverage(mass[0], bm, cfg.nk, coverage=cov), args.iters)
    props = torch.cuda.get_device_properties(dev)
    exps = float(cfg.N) * cfg.N * cfg.H
    peak = props.multi_processor_count * 16 * 1.8e9       # exp/s at ~1.8 GHz under load
    print(json.dumps({
        "workload": cfg.name, "H": cfg.H, "N": cfg.N,
        "dense_attention_with_lse_ms": t_attn,
        "block_mass_two_pass_ms": t2, "block_mass_one_pass_ms": t1,
        "block_mass_one_pass_TFLOPs": 2.0 * exps * cfg.d / (t1 * 1e-3) / 1e12,
        "roofline": {"kernel": "block_mass (one pass)", "bound": "alu", "unit": "Gexp/s",
                     "achieved": exps / (t1 * 1e-3) / 1e9, "peak": peak / 1e9,
                     "frac": exps / (t1 * 1e-3) / peak},
        "mask_from_mass_ms": t_sel, "mask_coverage_ms": t_cov,
        "kept_blocks_mean": float(kept.float().mean()), "coverage_mean": float(cov.mean()),
    }))


if __name__ == "__main__":
    main()
