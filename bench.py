#!/usr/bin/env python
"""bench.py — headline benchmark of the Chorus II sparsity-reuse hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl chorus|reference]
                    [--workload cfg2|cfg1|cfg4] [--mode replicas|ulysses] [--no-fp8] [--no-extras]

One "step" = one pass of the hot path over one attention layer's inputs (BASELINE.json configs[1]:
480p Wan-2.2-14B-shaped layer, H=40, N=32760, d=128, 25 % density block masks):
    chorus_mask_to_index (stored bitmask -> CSR)  ->  chorus_block_sparse_attn_fwd (BF16)
    -> chorus_quantize_fp8 -> chorus_block_sparse_attn_fwd (FP8)         [--no-fp8 leaves this leg out]
Metric: effective TFLOP/s on kept tiles, FLOPs = 4*N^2*d*H*density per attention call
(BASELINE.json north_star).  Prints ONE JSON line (rank 0).

Besides the timed step the line carries, outside the timed region (rank 0, N = 1): `parity` (the CPU oracle's
sampled items compared element-wise with what the GPU just computed), `cpu_baseline`, `density_sweep`
(5/10/25/50/100 % on one layer, 100 % against the dense roofline), `cfg4` (the 720p layer) and `extras`
(first-frame scaling, the paper's 64 x 128 geometry, mask construction; --no-extras leaves them out).

Multi-GPU (torchrun).  --mode replicas (default): the path has no exchange step (one GPU per attention call,
north_star), so N ranks run N independent replicas; `value` is the aggregate ("weak").  --mode ulysses: the
paper's own multi-GPU scheme (appendix A): tokens sharded over the ranks, heads re-partitioned by
the greedy schedule, all-to-all in and out around the per-rank attention; total work fixed ("strong").

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the
same workload on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "block-sparse attn effective TFLOPS (kept tiles) @480p"
UNIT = "TFLOP/s"
# BASELINE.json north_star tolerances
BF16_MAX, BF16_MEAN, FP8_MAX, FP8_COS = 2e-2, 2e-3, 8e-2, 0.995


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16": d["bf16_tflops"],
                "bf16_sustained": d.get("bf16_tflops_sustained"), "sm_max_mhz": d.get("sm_max_mhz", 1965.0),
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def get_cfg(name):
    from paper_2606_25040_b200 import workloads as W
    return {"cfg1": W.CFG1, "cfg2": W.CFG2, "cfg4": W.CFG4}[name]


def attn_flops(cfg, density):
    return 4.0 * cfg.N * cfg.N * cfg.d * cfg.H * density


# --------------------------------------------------------------------------------------------------
# clock sampling during the timed region
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: NVML every 2 ms when the
    nvidia_ml_py binding is there (the timed region is only ~0.2 s), else `nvidia-smi` every 0.1 s."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int, uuid: str | None = None):
        self.index = index
        self.samples = []          # (sm_mhz, sm_max_mhz, [active reason names])
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            # CUDA ordinals follow CUDA_VISIBLE_DEVICES, NVML's do not: go by UUID when torch gives one
            self._h = (pynvml.nvmlDeviceGetHandleByUUID(uuid) if uuid
                       else pynvml.nvmlDeviceGetHandleByIndex(index))
            self._max = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
            self._bits = [(pynvml.nvmlClocksEventReasonHwSlowdown, "hw_slowdown"),
                          (pynvml.nvmlClocksEventReasonHwThermalSlowdown, "hw_thermal_slowdown"),
                          (pynvml.nvmlClocksEventReasonSwThermalSlowdown, "sw_thermal_slowdown"),
                          (pynvml.nvmlClocksEventReasonSwPowerCap, "sw_power_cap")]
            self._nvml = pynvml
        except Exception:
            self._nvml = None

    def _sample_once(self):
        try:
            if self._nvml is not None:
                n = self._nvml
                mhz = float(n.nvmlDeviceGetClockInfo(self._h, n.NVML_CLOCK_SM))
                mask = int(n.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                self.samples.append((mhz, self._max, [nm for bit, nm in self._bits if mask & bit]))
                return
            out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.QUERY}",
                                  "--format=csv,noheader,nounits"], capture_output=True, text=True,
                                 timeout=5).stdout.strip().splitlines()
            if out:
                f = [x.strip() for x in out[0].split(",")]
                self.samples.append((float(f[0]), float(f[1]),
                                     [n for n, v in zip(self.NAMES, f[3:]) if v.lower().startswith("active")]))
        except Exception:
            pass

    def _run(self):
        period = 0.002 if self._nvml is not None else 0.1
        while not self._stop.is_set():
            self._sample_once()
            self._stop.wait(period)

    def start(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join(timeout=10)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        reasons = sorted({n for _, _, fl in self.samples for n in fl})
        return {"sm_mhz": statistics.median(s[0] for s in self.samples),
                "sm_min_mhz": min(s[0] for s in self.samples),
                "sm_max_mhz": self.samples[0][1], "reasons": reasons, "samples": len(self.samples),
                "via": "nvml" if self._nvml is not None else "nvidia-smi"}


# --------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline + parity / --impl reference)
# --------------------------------------------------------------------------------------------------
def item_flops(cfg, bm, items):
    from paper_2606_25040_b200 import workloads as W
    keep = W.unpack_bits(bm, cfg.nk)
    valid = np.minimum(64, cfg.N - 64 * np.arange(cfg.nk))
    flops = 0.0
    for _, h, qb in items:
        rows = min(128, cfg.N - 128 * qb)
        flops += 4.0 * rows * float(valid[keep[h, qb]].sum()) * cfg.d
    return flops


def draw_items(cfg, H, n, seed):
    """n (head, query block) items: every head in turn, first and last (ragged) query block of head 0 and of the
    last head always in."""
    g = np.random.default_rng(seed)
    hs = np.arange(n) % H
    qs = g.integers(0, cfg.nq, n)
    qs[0], hs[0] = 0, 0
    if n > 1:
        qs[-1], hs[-1] = cfg.nq - 1, H - 1
    return np.stack([np.zeros(n, np.int64), hs, qs], axis=1).astype(np.int32)


def oracle_run(cfg, Q, K, V, bm, items, fp8_scales=None):
    """The oracle, as it stands, on `items`: (seconds, flops, outputs float64 [n][128][d])."""
    import oracle
    t0 = time.perf_counter()
    out = oracle.block_sparse_attn(Q, K, V, bm, cfg.scale, items=items, fp8_scales=fp8_scales)
    return time.perf_counter() - t0, item_flops(cfg, bm, items), out


def gather_gpu_items(O, items, N):
    """O: torch [1][N][H][d] on the device -> float64 numpy [n][128][d] (rows beyond N zero)."""
    out = np.zeros((len(items), 128, O.shape[3]))
    for t, (_, h, qb) in enumerate(items):
        lo, hi = int(qb) * 128, min(N, int(qb) * 128 + 128)
        out[t, : hi - lo] = O[0, lo:hi, int(h)].float().cpu().numpy()
    return out


def parity_stats(got, ref):
    e = np.abs(got - ref)
    cos = float((got * ref).sum() / max(np.linalg.norm(got) * np.linalg.norm(ref), 1e-30))
    return {"max_abs": float(e.max()), "mean_abs": float(e.mean()), "cos": cos,
            "relfro": float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-30))}


def cpu_baseline_and_parity(cfg, Qb, Kb, Vb, bm, dO, fp8_host, dO8, budget_s=9.0):
    """Time the oracle on a bounded sample of the step's own tensors (about budget_s per attention leg) and
    compare its outputs element by element with what the GPU computed for the same items."""
    import oracle
    cores = oracle.num_threads()
    H = Qb.shape[2]
    dt, _, _ = oracle_run(cfg, Qb, Kb, Vb, bm, draw_items(cfg, H, cores, 0))            # probe: one item per core
    n = int(max(cores, min(40 * cores, cores * round(budget_s / max(dt, 1e-3)))))
    items = draw_items(cfg, H, n, 1)
    dt, fl, ref = oracle_run(cfg, Qb, Kb, Vb, bm, items)
    st = parity_stats(gather_gpu_items(dO, items, cfg.N), ref)
    parity = {"items": int(n), "of": int(H * cfg.nq), "heads_covered": int(len(set(items[:, 1].tolist()))),
              "bf16": {**st, "tol": {"max_abs": BF16_MAX, "mean_abs": BF16_MEAN},
                       "pass": bool(st["max_abs"] <= BF16_MAX and st["mean_abs"] <= BF16_MEAN)}}
    seconds, flops = dt, fl
    if fp8_host is not None:
        q8, k8, v8, qs, ks, vs = fp8_host
        dt8, fl8, ref8 = oracle_run(cfg, q8, k8, v8, bm, items, fp8_scales=(qs, ks, vs))
        st8 = parity_stats(gather_gpu_items(dO8, items, cfg.N), ref8)
        parity["fp8"] = {**st8, "reference": "fp64 oracle on the dequantised codes (configs[2])",
                         "tol": {"max_abs": FP8_MAX, "cos": FP8_COS},
                         "pass": bool(st8["max_abs"] <= FP8_MAX and st8["cos"] >= FP8_COS)}
        seconds, flops = seconds + dt8, flops + fl8
    parity["pass"] = all(v["pass"] for k, v in parity.items() if isinstance(v, dict))
    base = {"value": flops / seconds / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n} (head, 128-row query block) items of {cfg.name} over all {H} heads (of {H * cfg.nq}), "
                      f"fp64, bf16 inputs{' and dequantised e4m3 inputs' if fp8_host is not None else ''}, {seconds:.1f} s",
            "seconds": seconds}
    return base, parity


def run_reference(args):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_25040_b200 import workloads as W
    import oracle
    cfg = get_cfg(args.workload)
    heads = min(cfg.H, 4)                      # the sample only touches a few heads
    sub = W.scaled(cfg, H=heads)
    Qb, Kb, Vb = W.qkv_bits(sub)
    bm = W.layer_mask(sub)
    cores = oracle.num_threads()
    # size one step at ~2.5 s of CPU work
    dt, _, _ = oracle_run(sub, Qb, Kb, Vb, bm, draw_items(sub, heads, cores, 0))
    n = int(max(1, min(16 * cores, round(cores * 2.5 / max(dt, 1e-3)))))
    for _ in range(args.warmup):
        oracle_run(sub, Qb, Kb, Vb, bm, draw_items(sub, heads, max(1, n // 4), 99))
    tot_t = tot_f = 0.0
    for s in range(args.steps):
        dt, fl, _ = oracle_run(sub, Qb, Kb, Vb, bm, draw_items(sub, heads, n, s))
        tot_t += dt
        tot_f += fl
    val = tot_f / tot_t / 1e12
    sample = f"{n} random (head, query-block) items of {cfg.name} per step, fp64 oracle"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": cfg.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# --------------------------------------------------------------------------------------------------
# multi-rank aggregation (only the timings are reduced; the ulysses mode's data path is in ulysses.py)
# --------------------------------------------------------------------------------------------------
def max_over_ranks(values, device, world):
    """Device-side times of all ranks -> the slowest rank's (the driver's contract: max over ranks)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_value(world, flops_per_rank_step, ms_per_step):
    """Aggregate TFLOP/s of `world` replicas that each do flops_per_rank_step in ms_per_step (max)."""
    return world * flops_per_rank_step / (ms_per_step * 1e-3) / 1e12


def ulysses_plan(cost, world):
    """Head -> rank plan of the ulysses mode from the per-head costs (host ints): the greedy schedule's order,
    and the max / mean load before (heads in index order) and after it."""
    from paper_2606_25040_b200 import binding as B
    from paper_2606_25040_b200 import ulysses
    H = len(cost)
    order = B.chorus_schedule_heads(cost, world)[0].reshape(-1).tolist()
    return order, {"imbalance_max_over_avg_before": ulysses.imbalance(cost, list(range(H)), world),
                   "imbalance_max_over_avg_after": ulysses.imbalance(cost, order, world)}


def median_ms(fn, stream, iters=7, warm=3):
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(iters):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        fn()
        b.record(stream)
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return statistics.median(ts)


# --------------------------------------------------------------------------------------------------
# blocks measured outside the timed region (rank 0)
# --------------------------------------------------------------------------------------------------
def density_sweep(cfg, dev, stream, dQ, dK, dV, dO, q8, dO8, peaks):
    """BASELINE.json configs[4]: one layer at 5/10/25/50/100 %; 100 % is dense attention through the same
    kernel, set against the dense roofline (all N^2 tiles at the measured cuBLAS rate)."""
    import torch
    from paper_2606_25040_b200 import binding as B
    from paper_2606_25040_b200 import workloads as W
    out = []
    for rho in (0.05, 0.10, 0.25, 0.50, 1.0):
        bms = W.layer_mask(cfg, density=rho)
        rho_real = W.mask_density(bms, cfg.nk)
        rp_, ci_ = B.chorus_mask_to_index(torch.from_numpy(bms[None].view(np.int32)).to(dev), cfg.nk)
        ent = {"density": rho_real, "flops": attn_flops(cfg, rho_real)}
        legs = [("bf16", lambda: B.chorus_block_sparse_attn_fwd(dQ, dK, dV, rp_, ci_, cfg.scale, O=dO), 1)]
        if q8 is not None:
            legs.append(("fp8", lambda: B.chorus_block_sparse_attn_fwd(q8[0], q8[1], q8[2], rp_, ci_, cfg.scale,
                                                                       dtype=B.CHORUS_FP8_E4M3, O=dO8, fp8_scales=q8[3:]), 2))
        for name, fn, mult in legs:
            ms = median_ms(fn, stream, iters=5, warm=2)
            tf = ent["flops"] / (ms * 1e-3) / 1e12
            ent[name] = {"ms": ms, "TFLOPs": tf, "frac_of_peak": tf / (peaks["bf16"] * mult)}
            if rho == 1.0:
                ent[name]["dense_roofline_ms"] = ent["flops"] / (peaks["bf16"] * mult * 1e12) * 1e3
        out.append(ent)
        del rp_, ci_
    return out


def cfg4_block(dev, stream, peaks, fp8):
    """The 720p layer (BASELINE.json configs[3]: H 40, N 75600, 15 %, 1 % of rows x8), timing only: the values are
    drawn on the device (same distribution, not workloads.py's bytes; parity of cfg4 is in tests/)."""
    import torch
    from paper_2606_25040_b200 import binding as B
    from paper_2606_25040_b200 import workloads as W
    cfg = W.CFG4
    g = torch.Generator(device=dev)
    g.manual_seed(2)
    ts = []
    for _ in range(3):
        x = torch.randn((1, cfg.N, cfg.H, cfg.d), device=dev, generator=g)
        x *= torch.where(torch.rand((1, cfg.N, cfg.H, 1), device=dev, generator=g) < 0.01, 8.0, 1.0)
        ts.append(x.to(torch.bfloat16))
        del x
    Q, K, V = ts
    O = torch.empty_like(Q)
    # 15 % Bernoulli rows with the diagonal forced: the kernels see what they see with workloads.layer_mask
    # (which takes ~25 s on the host at this size), row lengths 177 +- 12 instead of exactly 177
    keep = torch.rand((cfg.H, cfg.nq, cfg.nk), device=dev, generator=g) < cfg.density
    keep[:, torch.arange(cfg.nq), torch.clamp(2 * torch.arange(cfg.nq), max=cfg.nk - 1)] = True
    pad = cfg.words * 32 - cfg.nk
    bits = torch.nn.functional.pad(keep, (0, pad)).view(cfg.H, cfg.nq, cfg.words, 32).to(torch.int64)
    bm = (bits << torch.arange(32, device=dev)).sum(-1)
    bm = torch.where(bm >= 2 ** 31, bm - 2 ** 32, bm).to(torch.int32)[None].contiguous()
    density = float(keep.float().mean())
    rp, ci = B.chorus_mask_to_index(bm, cfg.nk)
    ws = torch.empty(max(4, B.mask_to_index_workspace_bytes(1, cfg.H, cfg.nq, cfg.nk)), dtype=torch.uint8, device=dev)
    flops = attn_flops(cfg, density)
    out = {"workload": cfg.name, "H": cfg.H, "N": cfg.N, "density": density, "flops": flops,
           "data": "device-drawn N(0,1) bf16, 1 % of rows x8, Bernoulli masks with the diagonal forced"}
    ms = median_ms(lambda: B.chorus_mask_to_index(bm, cfg.nk, row_ptr=rp, col_idx=ci, workspace=ws), stream, 5, 2)
    out["decode_ms"] = ms
    ms = median_ms(lambda: B.chorus_block_sparse_attn_fwd(Q, K, V, rp, ci, cfg.scale, O=O), stream, 5, 2)
    out["attn_bf16"] = {"ms": ms, "TFLOPs": flops / ms / 1e9, "frac_of_peak": flops / ms / 1e9 / peaks["bf16"]}
    if fp8:
        q8 = B.chorus_quantize_fp8(Q, K, V)
        out["quantize_ms"] = median_ms(lambda: B.chorus_quantize_fp8(Q, K, V, out=q8), stream, 5, 2)
        ms = median_ms(lambda: B.chorus_block_sparse_attn_fwd(q8[0], q8[1], q8[2], rp, ci, cfg.scale, dtype=B.CHORUS_FP8_E4M3,
                                                              O=O, fp8_scales=q8[3:]), stream, 5, 2)
        out["attn_fp8"] = {"ms": ms, "TFLOPs": flops / ms / 1e9, "frac_of_2x_bf16_peak": flops / ms / 1e9 / (2 * peaks["bf16"])}
    return out


def extras_block(cfg, dev, stream, dQ, dK, dV, dO, q8, dO8, rp, ci, peaks):
    """Variants of row f-4 and the mask-construction calls of row f-2 on the bench's own 480p tensors
    (median of 5 launches each after 2 warm-ups; the kernels before them have brought the part to its
    power-capped steady state)."""
    import torch
    from paper_2606_25040_b200 import binding as B
    from paper_2606_25040_b200 import workloads as W
    N, H = cfg.N, cfg.H
    out = {}
    bf16 = lambda **kw: median_ms(lambda: B.chorus_block_sparse_attn_fwd(dQ, dK, dV, rp, ci, cfg.scale, O=dO, **kw), stream, 5, 2)
    ff = dict(n_first=cfg.hp * cfg.wp, beta=1.2)
    out["plain_bf16_ms"] = bf16()
    out["first_frame_bf16_ms"] = bf16(**ff)
    if q8 is not None:
        fp8 = lambda **kw: median_ms(lambda: B.chorus_block_sparse_attn_fwd(
            q8[0], q8[1], q8[2], rp, ci, cfg.scale, O=dO8, dtype=B.CHORUS_FP8_E4M3, fp8_scales=q8[3:], **kw), stream, 5, 2)
        out["plain_fp8_ms"] = fp8()
        out["first_frame_fp8_ms"] = fp8(**ff)
    out["first_frame"] = ff
    # uneven rows (top-p-like): row budgets x U[0.7, 1.3] at the same mean density, against the uniform mask
    bmj = W.layer_mask(cfg, jitter=True)
    rpj, cij = B.chorus_mask_to_index(torch.from_numpy(bmj[None].view(np.int32)).to(dev), cfg.nk)
    msj = median_ms(lambda: B.chorus_block_sparse_attn_fwd(dQ, dK, dV, rpj, cij, cfg.scale, O=dO), stream, 5, 2)
    dj = W.mask_density(bmj, cfg.nk)
    out["jitter_mask_bf16"] = {"density": dj, "ms": msj, "TFLOPs": attn_flops(cfg, dj) / msj / 1e9,
                               "uniform_TFLOPs": attn_flops(cfg, cfg.density) / out["plain_bf16_ms"] / 1e9}
    del rpj, cij
    # the paper's geometry: 64-row x 128-key mask blocks at 25 %
    rng = np.random.default_rng(0)
    nq64, nk128 = (N + 63) // 64, (N + 127) // 128
    k_half = rng.random((H, nq64 // 2, nk128)) < 0.25
    ws = torch.empty(1 << 20, dtype=torch.uint8, device=dev)
    for name, keep in (("halves_agree", np.repeat(k_half, 2, axis=1)), ("halves_independent", rng.random((H, nq64, nk128)) < 0.25)):
        bm64 = torch.from_numpy(W.pack_bits(keep)[None].view(np.int32)).to(dev)
        rp64, ci64 = B.chorus_mask_to_index_64x128(bm64, N)
        t_dec = median_ms(lambda: B.chorus_mask_to_index_64x128(bm64, N, row_ptr=rp64, col_idx=ci64, workspace=ws), stream, 5, 2)
        t_att = median_ms(lambda: B.chorus_block_sparse_attn_fwd(dQ, dK, dV, rp64, ci64, cfg.scale, O=dO, geometry_64x128=True), stream, 5, 2)
        tiles = int(rp64[-1])
        out["geometry_64x128_" + name] = {
            "mask_density": float(keep.mean()), "tiles_computed_frac": tiles / (H * cfg.nq * cfg.nk),
            "decode_us": t_dec * 1e3, "attn_bf16_ms": t_att,
            "TFLOPs_on_computed_tiles": 4.0 * 128 * 64 * 128 * tiles / (t_att * 1e-3) / 1e12,
            "TFLOPs_on_mask_blocks": 4.0 * 64 * 128 * 128 * float(keep.sum()) / (t_att * 1e-3) / 1e12}
        del bm64, rp64, ci64
    # mask construction (the historical request's side): dense attention with its LSE, block
    # mass from that LSE in one sweep, top-p selection, coverage
    full = torch.full((1, H, cfg.nq, cfg.words), -1, dtype=torch.int32, device=dev)
    rpf, cif = B.chorus_mask_to_index(full, cfg.nk)
    lse = torch.empty((1, H, N), dtype=torch.float32, device=dev)
    mass = torch.empty((1, H, cfg.nq, cfg.nk), dtype=torch.float32, device=dev)
    t_attn = median_ms(lambda: B.chorus_block_sparse_attn_fwd(dQ, dK, dV, rpf, cif, cfg.scale, O=dO, lse=lse), stream, 3, 1)
    t1 = median_ms(lambda: B.chorus_block_mass(dQ, dK, cfg.scale, mass=mass, lse=lse), stream, 3, 1)
    bmo = torch.empty((H, cfg.nq, cfg.words), dtype=torch.int32, device=dev)
    kept = torch.empty((H, cfg.nq), dtype=torch.int32, device=dev)
    t_sel = median_ms(lambda: B.chorus_mask_from_mass(mass[0], 0.9, 0.1, bitmask=bmo, kept=kept), stream, 3, 1)
    cov = torch.empty(H, dtype=torch.float32, device=dev)
    t_cov = median_ms(lambda: B.chorus_mask_coverage(mass[0], bmo, cfg.nk, coverage=cov), stream, 3, 1)
    exps = float(N) * N * H
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = sms * 16 * peaks["sm_max_mhz"] * 1e6            # MUFU: 16 exp / clk / SM at the maximum SM clock
    out["mask_build"] = {"dense_attention_with_lse_ms": t_attn, "block_mass_given_lse_ms": t1,
                         "block_mass_over_dense_attention": t1 / t_attn,
                         "block_mass_TFLOPs": 2.0 * exps * cfg.d / (t1 * 1e-3) / 1e12,
                         "roofline": {"kernel": "block_mass (one sweep)", "bound": "alu", "unit": "Gexp/s",
                                      "achieved": exps / (t1 * 1e-3) / 1e9, "peak": peak / 1e9,
                                      "frac": exps / (t1 * 1e-3) / peak,
                                      "on_mufu": 0.625, "frac_mufu_only": 0.625 * exps / (t1 * 1e-3) / peak,
                                      "note": "all N^2 H exponentials against the MUFU rate; 3 of 8 take the "
                                              "degree-3 polynomial on the FMA pipe (frac_mufu_only counts 5 of 8)",
                                      "peak_source": "148 SMs x 16 MUFU lanes x max SM clock (DESIGN.md 6.6)"},
                         "mask_from_mass_ms": t_sel, "mask_coverage_ms": t_cov,
                         "kept_blocks_mean": float(kept.float().mean()), "coverage_mean": float(cov.mean())}
    return out


# --------------------------------------------------------------------------------------------------
# the CUDA path
# --------------------------------------------------------------------------------------------------
def run_chorus(args):
    import torch
    import torch.distributed as dist
    from paper_2606_25040_b200 import binding as B
    from paper_2606_25040_b200 import ulysses
    from paper_2606_25040_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()  # fail loudly if the extension is missing

    cfg = get_cfg(args.workload)
    peaks = load_peaks()
    uly = args.mode == "ulysses"
    Qb, Kb, Vb = W.qkv_bits(cfg)
    if uly:
        # per-head densities ~ U[0.10, 0.40] (a different sparsity level per head; configs[4])
        rho_h = np.random.default_rng(77).uniform(0.10, 0.40, cfg.H)
        bm = W.pack_bits(np.stack([W.head_mask(cfg.nq, cfg.nk, cfg.tokens_per_frame, float(rho_h[h]), cfg.mask_seed + h,
                                               cfg.band) for h in range(cfg.H)]))
    else:
        bm = W.layer_mask(cfg)
    density = W.mask_density(bm, cfg.nk)
    flops_attn = attn_flops(cfg, density)                 # whole layer, all heads

    to_bf16 = lambda x: torch.from_numpy(x.view(np.int16)).view(torch.bfloat16)
    stream = torch.cuda.current_stream()
    has_fp8 = args.fp8

    # ---- ulysses mode: this rank's token shard in, this rank's heads through the kernels, shard of O out -------
    plan = None
    if uly:
        assert cfg.H % world == 0, "ulysses mode: H must be a multiple of the number of ranks"
        keep_counts = W.unpack_bits(bm, cfg.nk).sum(axis=(1, 2))
        order, plan = ulysses_plan([int(c) for c in keep_counts], world)
        slots = cfg.H // world
        mine = order[rank * slots:(rank + 1) * slots]
        bounds = ulysses.shard_bounds(cfg.N, world)
        lo, hi = bounds[rank], bounds[rank + 1]
        xQ, xK, xV = (to_bf16(np.ascontiguousarray(x[:, lo:hi])).to(dev) for x in (Qb, Kb, Vb))
        bm_loc = np.ascontiguousarray(bm[mine])
        Hl = slots
        my_flops = attn_flops(cfg, 1.0) / cfg.H * float(W.unpack_bits(bm_loc, cfg.nk).mean()) * Hl
        row_bytes = cfg.d * 2
        plan.update({"heads_per_rank": slots, "tokens_per_rank": hi - lo,
                     "a2a_send_bytes_per_rank_per_step": int((3 + (2 if has_fp8 else 1)) * (hi - lo) * cfg.H * row_bytes * (world - 1) / world),
                     "order": order, "hardware": "measured on this run" if world > 1 else "one rank: no exchange (Table 4: a no-op)"})
        dM = torch.from_numpy(bm_loc[None].view(np.int32)).to(dev)
        if world == 1:
            dQ, dK, dV = xQ, xK, xV
    else:
        Hl = cfg.H
        my_flops = flops_attn
        hQ, hK, hV = (to_bf16(x).pin_memory() for x in (Qb, Kb, Vb))
        hM = torch.from_numpy(bm[None].view(np.int32)).pin_memory()
        dQ, dK, dV, dM = (x.to(dev) for x in (hQ, hK, hV, hM))
    rows = Hl * cfg.nq
    row_ptr = torch.empty(rows + 1, dtype=torch.int32, device=dev)
    col_idx = torch.empty(rows * cfg.nk, dtype=torch.int32, device=dev)  # upper bound: no D2H read of nnz
    ws = torch.empty(max(4, B.mask_to_index_workspace_bytes(1, Hl, cfg.nq, cfg.nk)), dtype=torch.uint8, device=dev)
    dO = torch.empty((1, cfg.N, Hl, cfg.d), dtype=torch.bfloat16, device=dev)
    dO8 = torch.empty_like(dO) if has_fp8 else None
    q8 = None
    if has_fp8:
        if uly and world > 1:                         # buffers only: the step quantises what the exchange delivers
            z = torch.zeros((1, cfg.N, Hl, cfg.d), dtype=torch.bfloat16, device=dev)
            q8 = B.chorus_quantize_fp8(z, z, z)
            del z
        else:
            q8 = B.chorus_quantize_fp8(dQ, dK, dV)

    def kernels(q, k, v, ev=None):
        B.chorus_mask_to_index(dM, cfg.nk, row_ptr=row_ptr, col_idx=col_idx, workspace=ws)
        if ev: ev[0].record(stream)
        B.chorus_block_sparse_attn_fwd(q, k, v, row_ptr, col_idx, cfg.scale, O=dO)
        if ev: ev[1].record(stream)
        if has_fp8:
            B.chorus_quantize_fp8(q, k, v, out=q8)
            if ev: ev[2].record(stream)
            B.chorus_block_sparse_attn_fwd(q8[0], q8[1], q8[2], row_ptr, col_idx, cfg.scale,
                                           dtype=B.CHORUS_FP8_E4M3, O=dO8, fp8_scales=q8[3:])
            if ev: ev[3].record(stream)

    def step(ev=None):
        if uly and world > 1:
            q, k, v = (ulysses.seq_to_heads(x, order, cfg.N) for x in (xQ, xK, xV))
            kernels(q, k, v, ev)
            ulysses.heads_to_seq(dO, order)
            if has_fp8:
                ulysses.heads_to_seq(dO8, order)
        else:
            kernels(dQ, dK, dV, ev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid)
    if rank == 0:
        sampler.start()
    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    e_start = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    e_end = torch.cuda.Event(enable_timing=True)
    B.chorus_reset_launch_count()
    for k in range(K):
        e_start[k].record(stream)
        step(evs[k])
    e_end.record(stream)
    barrier()
    launches = B.chorus_launch_count()
    clocks = sampler.stop() if rank == 0 else None     # clocks of the device-timed region only
    total_ms = e_start[0].elapsed_time(e_end)
    dec_ms = statistics.mean(e_start[k].elapsed_time(evs[k][0]) for k in range(K))   # ulysses: incl. the exchange in
    attn_ms = statistics.mean(evs[k][0].elapsed_time(evs[k][1]) for k in range(K))
    attn_ms_min = min(evs[k][0].elapsed_time(evs[k][1]) for k in range(K))
    attn_ms_median = statistics.median(evs[k][0].elapsed_time(evs[k][1]) for k in range(K))
    if has_fp8:
        quant_ms = statistics.mean(evs[k][1].elapsed_time(evs[k][2]) for k in range(K))
        attn8_ms = statistics.mean(evs[k][2].elapsed_time(evs[k][3]) for k in range(K))

    # ---- end to end through the ABI with HOST buffers (replicas mode) ---------------------------------------
    # H2D of Q, K, V and the mask, D2H of both results, per step.  The host tensors are stored head-major
    # ([B][H][N][d]; the ABI takes it through its strides), so that a group of heads is one contiguous copy: heads
    # go through in E2E_CHUNKS groups on three streams (H2D of group c+1 | kernels of group c | D2H of group c-1).
    e2e = None
    if not uly:
        E2E_CHUNKS = next(c for c in (20, 10, 8, 5, 4, 2, 1) if cfg.H % c == 0)   # small groups: short fill and drain
        hc = cfg.H // E2E_CHUNKS
        hm = lambda t: t.permute(0, 2, 1, 3).contiguous()                 # [B][N][H][d] -> [B][H][N][d]
        hQh, hKh, hVh = (hm(x).pin_memory() for x in (hQ, hK, hV))
        hOh = torch.empty_like(hQh).pin_memory()
        hO8h = torch.empty_like(hQh).pin_memory() if has_fp8 else None
        dQh, dKh, dVh = (torch.empty_like(x, device=dev) for x in (hQh, hKh, hVh))
        dOh, dO8h = torch.empty_like(dQh), torch.empty_like(dQh)
        as_bnhd = lambda t, c: t[:, c * hc:(c + 1) * hc].permute(0, 2, 1, 3)   # strided [B][N][hc][d] view
        q8c = [B.chorus_quantize_fp8(as_bnhd(dQh, 0), as_bnhd(dKh, 0), as_bnhd(dVh, 0)) for _ in range(E2E_CHUNKS)] if has_fp8 else None
        s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        ev_in = [torch.cuda.Event() for _ in range(E2E_CHUNKS)]
        ev_done = [torch.cuda.Event() for _ in range(E2E_CHUNKS)]
        ev_top, ev_mask = torch.cuda.Event(), torch.cuda.Event()
        ev_h2d = [torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)]

        def e2e_step():
            ev_top.record(stream)
            s_in.wait_event(ev_top)                 # do not run ahead of the step's start
            ev_h2d[0].record(s_in)
            # every host-to-device copy goes on s_in: a copy issued on the compute stream sits in the same
            # copy-engine queue as the Q/K/V groups and cost 2 ms per step
            with torch.cuda.stream(s_in):
                dM.copy_(hM, non_blocking=True)
                ev_mask.record(s_in)
            stream.wait_event(ev_mask)
            B.chorus_mask_to_index(dM, cfg.nk, row_ptr=row_ptr, col_idx=col_idx, workspace=ws)
            for c in range(E2E_CHUNKS):
                hs = slice(c * hc, (c + 1) * hc)
                with torch.cuda.stream(s_in):
                    s_in.wait_event(ev_done[c])     # the previous step has finished with this group's buffers
                    dQh[:, hs].copy_(hQh[:, hs], non_blocking=True)
                    dKh[:, hs].copy_(hKh[:, hs], non_blocking=True)
                    dVh[:, hs].copy_(hVh[:, hs], non_blocking=True)
                    ev_in[c].record(s_in)
                stream.wait_event(ev_in[c])
                q, k, v = as_bnhd(dQh, c), as_bnhd(dKh, c), as_bnhd(dVh, c)
                rp_c = row_ptr[c * hc * cfg.nq:(c + 1) * hc * cfg.nq + 1]
                B.chorus_block_sparse_attn_fwd(q, k, v, rp_c, col_idx, cfg.scale, O=as_bnhd(dOh, c))
                if has_fp8:
                    B.chorus_quantize_fp8(q, k, v, out=q8c[c])
                    B.chorus_block_sparse_attn_fwd(q8c[c][0], q8c[c][1], q8c[c][2], rp_c, col_idx, cfg.scale,
                                                   dtype=B.CHORUS_FP8_E4M3, O=as_bnhd(dO8h, c), fp8_scales=q8c[c][3:])
                ev_done[c].record(stream)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_done[c])
                    hOh[:, hs].copy_(dOh[:, hs], non_blocking=True)
                    if has_fp8:
                        hO8h[:, hs].copy_(dO8h[:, hs], non_blocking=True)
            ev_h2d[1].record(s_in)
            stream.wait_stream(s_out)               # the step ends when both results are in host memory
            stream.wait_stream(s_in)

        e2e_steps = max(2, min(K, 5))
        e2e_step()
        barrier()
        enc0 = B.chorus_tensor_map_encodes()
        a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        t_host = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        t_host = (time.perf_counter() - t_host) / e2e_steps * 1e3      # host time to enqueue one step
        b_.record(stream)
        barrier()
        e2e_ms = a.elapsed_time(b_) / e2e_steps
        e2e_h2d_ms = ev_h2d[0].elapsed_time(ev_h2d[1])     # the last step's host-to-device copies, first to last
        # regression check (not parity): the pipelined path must give what the single call gives
        e2e_ok = bool(torch.equal(hOh.permute(0, 2, 1, 3), dO.cpu())) if rank == 0 else True
        if has_fp8 and rank == 0:
            e2e_ok = e2e_ok and bool(torch.equal(hO8h.permute(0, 2, 1, 3), dO8.cpu()))
        e2e = {"ms_per_step": e2e_ms, "h2d_span_ms": e2e_h2d_ms, "host_enqueue_ms": t_host,
               "tensor_map_encodes_per_step": (B.chorus_tensor_map_encodes() - enc0) / e2e_steps,
               "h2d_bytes_per_step": int(3 * Qb.nbytes + bm.nbytes),
               "d2h_bytes_per_step": int(Qb.nbytes * (2 if has_fp8 else 1)),
               "results_copied_back": "O (bf16 leg)" + (" and O (fp8 leg)" if has_fp8 else ""),
               "pipeline": "%d head groups, H2D | kernels | D2H on three streams, head-major host tensors" % E2E_CHUNKS,
               "matches_single_call": e2e_ok}
        del hQh, hKh, hVh, hOh, hO8h, dQh, dKh, dVh, dOh, dO8h, q8c
    else:
        e2e_ms = total_ms / K                        # ulysses mode: the shards live on the devices; no host leg
        e2e = {"ms_per_step": e2e_ms, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
               "note": "ulysses mode: the token shards are device-resident between layers; see the replicas mode for the host-buffer leg"}

    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_ms], dev, world)
    ms_per_step = total_ms / K
    legs = 2 if has_fp8 else 1
    if uly:
        value = flops_attn * legs / (ms_per_step * 1e-3) / 1e12        # strong scaling: the layer is one job
        e2e_val = value
    else:
        value = whole_job_value(world, flops_attn * legs, ms_per_step)
        e2e_val = whole_job_value(world, flops_attn * legs, e2e_ms)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rank 0: the blocks outside the timed region, then the line ------------------------------------------
    single = world == 1 and not uly
    sweep = cfg4 = extras = None
    if single and cfg.name.startswith("cfg2"):
        sweep = density_sweep(cfg, dev, stream, dQ, dK, dV, dO, q8, dO8, peaks)
    # mask decode at the size where it is HBM-bound: a whole stored mask set (40 layers x H heads,
    # SURVEY section 8 d-4), timed alone with a flushed L2; reported beside the per-layer figure
    set_ms = set_bytes = None
    if single and cfg.name.startswith("cfg2"):
        Lset = 40
        dMs = dM.repeat(Lset, 1, 1, 1).contiguous()
        rows_s = Lset * rows
        rp_s = torch.empty(rows_s + 1, dtype=torch.int32, device=dev)
        ci_s = torch.empty(int(density * rows_s * cfg.nk) + 1024, dtype=torch.int32, device=dev)
        ws_s = torch.empty(max(4, B.mask_to_index_workspace_bytes(Lset, cfg.H, cfg.nq, cfg.nk)), dtype=torch.uint8, device=dev)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        ts = []
        for i in range(8):
            flush.zero_()
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            B.chorus_mask_to_index(dMs, cfg.nk, row_ptr=rp_s, col_idx=ci_s, workspace=ws_s)
            b_.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b_))
        set_ms = statistics.median(ts)
        set_bytes = 4 * rows_s * cfg.words + 4 * (rows_s + 1) + 4 * int(rp_s[-1].item())
        # the same set with 16-bit entries (chorus_mask_to_index_u16: half the dominant write)
        ci_s16 = torch.empty(ci_s.numel(), dtype=torch.uint16, device=dev)
        ts = []
        for i in range(8):
            flush.zero_()
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            B.chorus_mask_to_index(dMs, cfg.nk, row_ptr=rp_s, col_idx=ci_s16, workspace=ws_s)
            b_.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b_))
        set16_ms = statistics.median(ts)
        set16_bytes = 4 * rows_s * cfg.words + 4 * (rows_s + 1) + 2 * int(rp_s[-1].item())
        del ci_s16
        # one layer alone with a cold L2 (the step's own decode_ms follows an attention kernel, warm)
        ts = []
        for i in range(8):
            flush.zero_()
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            B.chorus_mask_to_index(dM, cfg.nk, row_ptr=row_ptr, col_idx=col_idx, workspace=ws)
            b_.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b_))
        layer_cold_ms = statistics.median(ts)
        del dMs, rp_s, ci_s, flush
    if single:
        # restore the step's outputs (the sweep and the decode legs overwrote dO / row_ptr) for the parity block
        kernels(dQ, dK, dV)
        torch.cuda.synchronize()
    cpu = parity = None
    if single and not args.no_cpu_baseline:
        fp8_host = tuple(t.cpu().numpy() for t in q8) if has_fp8 else None
        cpu, parity = cpu_baseline_and_parity(cfg, Qb, Kb, Vb, bm, dO, fp8_host, dO8)
    if single and args.extras and cfg.name.startswith("cfg2"):
        extras = extras_block(cfg, dev, stream, dQ, dK, dV, dO, q8, dO8, row_ptr, col_idx, peaks)
        del dQ, dK, dV, dO, dO8, q8
        torch.cuda.empty_cache()
        cfg4 = cfg4_block(dev, stream, peaks, has_fp8)

    achieved = my_flops / (attn_ms * 1e-3) / 1e12
    traffic = None
    tp = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    tj = json.load(open(tp)) if os.path.exists(tp) else {}
    traffic = tj.get(f"{cfg.name}_bf16_attn_dram_bytes_per_launch") if not uly else None
    nnz = int(round(density * cfg.H * cfg.nq * cfg.nk)) if not uly else int(W.unpack_bits(bm_loc, cfg.nk).sum())
    dec_bytes = 4 * (rows * cfg.words) + 4 * (rows + 1) + 4 * nnz
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "strong" if uly else "weak", "vs_baseline": None,
        "dtype": "bf16" + ("+fp8_e4m3" if has_fp8 else ""), "data": "synthetic",
        "config": {"workload": cfg.name, "B": cfg.B, "H": cfg.H, "N": cfg.N, "d": cfg.d,
                   "block": "128q x 64k", "density": density,
                   "multi_gpu": "ulysses: tokens sharded, heads scheduled, all-to-all in and out" if uly else "replicas only",
                   "l2": "inputs larger than L2 (Q+K+V+O = %.2f GB per step)" % (4 * Qb.nbytes / 1e9),
                   "step": "mask_to_index -> attn_fwd(bf16)" + (" -> quantize_fp8 -> attn_fwd(fp8)" if has_fp8 else "")},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": UNIT, **e2e},
        "gpu_launches": int(launches),
        "roofline": {"kernel": "attn_fwd bf16", "bound": "tensor", "achieved": achieved,
                     "peak": peaks["bf16"], "unit": "TFLOP/s", "frac": achieved / peaks["bf16"],
                     "traffic": traffic, "traffic_source": tj.get("source"),
                     "peak_source": peaks["source"] + " (burst cuBLAS bf16)",
                     "frac_of_sustained": achieved / peaks["bf16_sustained"] if peaks["bf16_sustained"] else None,
                     "frac_of_datasheet_2250": achieved / 2250.0,
                     "ms": attn_ms, "ms_min": attn_ms_min, "ms_median": attn_ms_median,
                     "flops_per_launch": my_flops},
        "breakdown": {"decode_ms": dec_ms, "decode_GBps": dec_bytes / (dec_ms * 1e-3) / 1e9,
                      "decode_frac_of_hbm": dec_bytes / (dec_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                      "attn_bf16_ms": attn_ms, "attn_bf16_TFLOPs": achieved,
                      "routing_overhead_ratio": dec_ms / (dec_ms + attn_ms)},
    }
    if set_ms is not None:
        line["breakdown"].update({"decode_set_ms": set_ms, "decode_set_bytes": set_bytes,
                                  "decode_set_GBps": set_bytes / (set_ms * 1e-3) / 1e9,
                                  "decode_set_frac_of_hbm": set_bytes / (set_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                  "decode_set": "40 layers x %d heads x %d rows, L2 flushed, median of 5" % (cfg.H, cfg.nq),
                                  "decode_layer_cold_l2_ms": layer_cold_ms,
                                  "decode_set_u16_ms": set16_ms, "decode_set_u16_bytes": set16_bytes,
                                  "decode_set_u16_frac_of_hbm": set16_bytes / (set16_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]})
    if has_fp8:
        a8 = my_flops / (attn8_ms * 1e-3) / 1e12
        line["breakdown"].update({"quantize_ms": quant_ms, "attn_fp8_ms": attn8_ms, "attn_fp8_TFLOPs": a8,
                                  "attn_fp8_frac_of_2x_bf16_peak": a8 / (2 * peaks["bf16"]),
                                  "attn_fp8_frac_of_datasheet_4500": a8 / 4500.0,
                                  "attn_fp8_plus_quantize_over_attn_bf16": (attn8_ms + quant_ms) / attn_ms,
                                  "attn_fp8_traffic": tj.get(f"{cfg.name}_fp8_attn_dram_bytes_per_launch")})
    if plan is not None:
        line["ulysses"] = plan
    if parity is not None:
        line["parity"] = parity
    if cpu is not None:
        line["cpu_baseline"] = cpu
    if sweep is not None:
        line["density_sweep"] = sweep
    if cfg4 is not None:
        line["cfg4"] = cfg4
    if extras is not None:
        line["extras"] = extras
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="chorus", choices=["chorus", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg4"])
    ap.add_argument("--mode", default="replicas", choices=["replicas", "ulysses"],
                    help="multi-GPU scheme: independent replicas (default) or the paper's Ulysses + head schedule")
    ap.add_argument("--no-fp8", dest="fp8", action="store_false", default=True,
                    help="leave the FP8 leg (quantise + FP8 attention) out of the step")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle leg (cpu_baseline and parity)")
    ap.add_argument("--no-extras", dest="extras", action="store_false", default=True,
                    help="skip the variants / mask-construction / 720p blocks measured outside the timed region")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "chorus" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_chorus(args)


if __name__ == "__main__":
    main()
