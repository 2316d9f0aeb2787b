#!/usr/bin/env python
"""bench.py — headline benchmark of the Chorus II sparsity-reuse hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl chorus|reference] [--workload cfg2|cfg1|cfg4]

One "step" = one pass of the hot path over one attention layer's inputs (BASELINE.json configs[1]:
480p Wan-2.2-14B-shaped layer, H=40, N=32760, d=128, 25 % density block masks):
    chorus_mask_to_index (stored bitmask -> CSR)  ->  chorus_block_sparse_attn_fwd (BF16)
    -> chorus_quantize_fp8 -> chorus_block_sparse_attn_fwd (FP8)         [--no-fp8 leaves this leg out]
Metric: effective TFLOP/s on kept tiles, FLOPs = 4*N^2*d*H*density per attention call
(BASELINE.json north_star).  Prints ONE JSON line (rank 0).

Multi-GPU (torchrun): the path has no exchange step (one GPU per attention call, north_star), so
N ranks run N independent replicas ("replicas only"); `value` is the aggregate.

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


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16": d["bf16_tflops"],
                "bf16_sustained": d.get("bf16_tflops_sustained"), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


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
# CPU oracle leg (cpu_baseline / --impl reference)
# --------------------------------------------------------------------------------------------------
def oracle_sample_time(cfg, Qb, Kb, Vb, bm, n_items, seed=0):
    """Time the oracle, as it stands, on n_items (head, q-block) items of the workload."""
    import oracle
    g = np.random.default_rng(seed)
    items = np.stack([np.zeros(n_items, np.int64), g.integers(0, Qb.shape[2], n_items),
                      g.integers(0, cfg.nq, n_items)], axis=1).astype(np.int32)
    keep_rows = 0
    from paper_2606_25040_b200 import workloads as W
    keep = W.unpack_bits(bm, cfg.nk)
    valid = np.minimum(64, cfg.N - 64 * np.arange(cfg.nk))
    flops = 0.0
    for _, h, qb in items:
        rows = min(128, cfg.N - 128 * qb)
        keys = float(valid[keep[h, qb]].sum())
        flops += 4.0 * rows * keys * cfg.d
        keep_rows += rows
    t0 = time.perf_counter()
    oracle.block_sparse_attn(Qb, Kb, Vb, bm, cfg.scale, items=items)
    dt = time.perf_counter() - t0
    return dt, flops, oracle.num_threads()


def cpu_baseline(cfg, Qb, Kb, Vb, bm, budget_s=15.0):
    import oracle
    cores = oracle.num_threads()
    dt, fl, _ = oracle_sample_time(cfg, Qb, Kb, Vb, bm, cores)          # probe: one item per core
    n = int(max(cores, min(64 * cores, cores * round(budget_s / max(dt, 1e-3)))))
    dt, fl, _ = oracle_sample_time(cfg, Qb, Kb, Vb, bm, n, seed=1)
    return {"value": fl / dt / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n} random (head, 128-row query block) items of {cfg.name} "
                      f"(of {Qb.shape[2] * cfg.nq}), fp64, {dt:.1f} s",
            "seconds": dt}


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
    dt, fl, _ = oracle_sample_time(sub, Qb, Kb, Vb, bm, cores)
    n = int(max(1, min(16 * cores, round(cores * 2.5 / max(dt, 1e-3)))))
    for _ in range(args.warmup):
        oracle_sample_time(sub, Qb, Kb, Vb, bm, max(1, n // 4))
    tot_t = tot_f = 0.0
    for s in range(args.steps):
        dt, fl, _ = oracle_sample_time(sub, Qb, Kb, Vb, bm, n, seed=s)
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
# multi-rank aggregation ("replicas only": no data-path collective; only the timings are reduced)
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


# --------------------------------------------------------------------------------------------------
# the CUDA path
# --------------------------------------------------------------------------------------------------
def run_chorus(args):
    import torch
    import torch.distributed as dist
    from paper_2606_25040_b200 import binding as B
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
    Qb, Kb, Vb = W.qkv_bits(cfg)
    bm = W.layer_mask(cfg)
    density = W.mask_density(bm, cfg.nk)
    flops_attn = attn_flops(cfg, density)

    to_bf16 = lambda x: torch.from_numpy(x.view(np.int16)).view(torch.bfloat16)
    hQ, hK, hV = (to_bf16(x).pin_memory() for x in (Qb, Kb, Vb))
    hM = torch.from_numpy(bm[None].view(np.int32)).pin_memory()
    hO = torch.empty((cfg.B, cfg.N, cfg.H, cfg.d), dtype=torch.bfloat16).pin_memory()
    dQ, dK, dV, dM = (x.to(dev) for x in (hQ, hK, hV, hM))
    dO = torch.empty_like(dQ)
    rows = cfg.H * cfg.nq
    row_ptr = torch.empty(rows + 1, dtype=torch.int32, device=dev)
    col_idx = torch.empty(rows * cfg.nk, dtype=torch.int32, device=dev)  # upper bound: no D2H read of nnz
    ws = torch.empty(max(4, B.mask_to_index_workspace_bytes(1, cfg.H, cfg.nq, cfg.nk)), dtype=torch.uint8, device=dev)
    has_fp8 = args.fp8
    if has_fp8:
        q8 = B.chorus_quantize_fp8(dQ, dK, dV)
        dO8 = torch.empty_like(dQ)
    stream = torch.cuda.current_stream()

    def step(ev=None):
        B.chorus_mask_to_index(dM, cfg.nk, row_ptr=row_ptr, col_idx=col_idx, workspace=ws)
        if ev: ev[0].record(stream)
        B.chorus_block_sparse_attn_fwd(dQ, dK, dV, row_ptr, col_idx, cfg.scale, O=dO)
        if ev: ev[1].record(stream)
        if has_fp8:
            B.chorus_quantize_fp8(dQ, dK, dV, out=q8)
            if ev: ev[2].record(stream)
            B.chorus_block_sparse_attn_fwd(q8[0], q8[1], q8[2], row_ptr, col_idx, cfg.scale,
                                           dtype=B.CHORUS_FP8_E4M3, O=dO8, fp8_scales=q8[3:])
            if ev: ev[3].record(stream)

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
    dec_ms = statistics.mean(e_start[k].elapsed_time(evs[k][0]) for k in range(K))
    attn_ms = statistics.mean(evs[k][0].elapsed_time(evs[k][1]) for k in range(K))
    attn_ms_min = min(evs[k][0].elapsed_time(evs[k][1]) for k in range(K))
    attn_ms_median = statistics.median(evs[k][0].elapsed_time(evs[k][1]) for k in range(K))
    if has_fp8:
        quant_ms = statistics.mean(evs[k][1].elapsed_time(evs[k][2]) for k in range(K))
        attn8_ms = statistics.mean(evs[k][2].elapsed_time(evs[k][3]) for k in range(K))

    # end-to-end through the ABI with HOST buffers: H2D of Q, K, V and the mask, D2H of O, per step.
    # The host tensors are stored head-major ([B][H][N][d]; the ABI takes it through its strides), so
    # that a group of heads is one contiguous copy: heads go through in E2E_CHUNKS groups on three
    # streams (H2D of group c+1 | the kernels of group c | D2H of group c-1).  Same bytes, same calls.
    E2E_CHUNKS = next(c for c in (20, 10, 8, 5, 4, 2, 1) if cfg.H % c == 0)   # small groups: short fill and drain
    hc = cfg.H // E2E_CHUNKS
    hm = lambda t: t.permute(0, 2, 1, 3).contiguous()                 # [B][N][H][d] -> [B][H][N][d]
    hQh, hKh, hVh = (hm(x).pin_memory() for x in (hQ, hK, hV))
    hOh = torch.empty_like(hQh).pin_memory()
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
        ev_h2d[1].record(s_in)
        stream.wait_stream(s_out)               # the step ends when its result is in host memory
        stream.wait_stream(s_in)

    e2e_steps = max(2, min(K, 5))
    e2e_step()
    barrier()
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
    # the pipelined path must give what the single call gives
    e2e_ok = bool(torch.equal(hOh.permute(0, 2, 1, 3), dO.cpu())) if rank == 0 else True

    # optional: the density sweep of BASELINE.json configs[4] (5/10/25/50/100 % on one layer; 100 % is
    # dense attention through the same kernel), outside the timed region, rank 0 only
    sweep = None
    if rank == 0 and args.sweep:
        sweep = []
        for rho in (0.05, 0.10, 0.25, 0.50, 1.0):
            bms = W.layer_mask(cfg, density=rho)
            dMs_ = torch.from_numpy(bms[None].view(np.int32)).to(dev)
            rho_real = W.mask_density(bms, cfg.nk)
            rp_, ci_ = B.chorus_mask_to_index(dMs_, cfg.nk)
            ent = {"density": rho_real, "flops": attn_flops(cfg, rho_real)}
            for name, fn in (("bf16", lambda: B.chorus_block_sparse_attn_fwd(dQ, dK, dV, rp_, ci_, cfg.scale, O=dO)),
                             ("fp8", (lambda: B.chorus_block_sparse_attn_fwd(q8[0], q8[1], q8[2], rp_, ci_, cfg.scale,
                                                                             dtype=B.CHORUS_FP8_E4M3, O=dO8, fp8_scales=q8[3:]))
                              if has_fp8 else None)):
                if fn is None:
                    continue
                for _ in range(3):
                    fn()
                torch.cuda.synchronize()
                ts = []
                for _ in range(7):
                    a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream); fn(); b_.record(stream)
                    torch.cuda.synchronize()
                    ts.append(a.elapsed_time(b_))
                ms = statistics.median(ts)
                tf = ent["flops"] / (ms * 1e-3) / 1e12
                ent[name] = {"ms": ms, "TFLOPs": tf,
                             "frac_of_peak": tf / (peaks["bf16"] * (2 if name == "fp8" else 1))}
            sweep.append(ent)
            del dMs_, rp_, ci_

    # mask decode at the size where it is HBM-bound: a whole stored mask set (40 layers x H heads,
    # SURVEY section 8 d-4), timed alone with a flushed L2; reported beside the per-layer figure
    set_ms = set_bytes = None
    if rank == 0 and cfg.name.startswith("cfg2"):
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
        del dMs, rp_s, ci_s, flush

    total_ms, e2e_ms = max_over_ranks([total_ms, e2e_ms], dev, world)
    ms_per_step = total_ms / K
    step_flops = flops_attn * (2 if has_fp8 else 1)
    value = whole_job_value(world, step_flops, ms_per_step)
    e2e_val = whole_job_value(world, step_flops, e2e_ms)

    if rank == 0:
        achieved = flops_attn / (attn_ms * 1e-3) / 1e12
        traffic = None
        tp = os.path.join(ROOT, "profiles", "roofline_traffic.json")
        if os.path.exists(tp):
            traffic = json.load(open(tp)).get(f"{cfg.name}_bf16_attn_dram_bytes_per_launch")
        nnz = int(round(density * rows * cfg.nk))
        dec_bytes = 4 * (rows * cfg.words) + 4 * (rows + 1) + 4 * nnz
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "bf16" + ("+fp8_e4m3" if has_fp8 else ""),
            "data": "synthetic",
            "config": {"workload": cfg.name, "B": cfg.B, "H": cfg.H, "N": cfg.N, "d": cfg.d,
                       "block": "128q x 64k", "density": density, "multi_gpu": "replicas only",
                       "l2": "inputs larger than L2 (Q+K+V+O = %.2f GB per step)" % (4 * Qb.nbytes / 1e9),
                       "step": "mask_to_index -> attn_fwd(bf16)" + (" -> quantize_fp8 -> attn_fwd(fp8)" if has_fp8 else "")},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_span_ms": e2e_h2d_ms, "host_enqueue_ms": t_host,
                    "h2d_bytes_per_step": int(3 * Qb.nbytes + bm.nbytes), "d2h_bytes_per_step": int(Qb.nbytes),
                    "pipeline": "%d head groups, H2D | kernels | D2H on three streams, head-major host tensors" % E2E_CHUNKS,
                    "matches_single_call": e2e_ok},
            "gpu_launches": int(launches),
            "roofline": {"kernel": "attn_fwd bf16", "bound": "tensor", "achieved": achieved,
                         "peak": peaks["bf16"], "unit": "TFLOP/s", "frac": achieved / peaks["bf16"],
                         "traffic": traffic, "peak_source": peaks["source"] + " (burst cuBLAS bf16)",
                         "frac_of_sustained": achieved / peaks["bf16_sustained"] if peaks["bf16_sustained"] else None,
                         "frac_of_datasheet_2250": achieved / 2250.0,
                         "ms": attn_ms, "ms_min": attn_ms_min, "ms_median": attn_ms_median,
                         "flops_per_launch": flops_attn},
            "breakdown": {"decode_ms": dec_ms, "decode_GBps": dec_bytes / (dec_ms * 1e-3) / 1e9,
                          "decode_frac_of_hbm": dec_bytes / (dec_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                          "attn_bf16_ms": attn_ms, "attn_bf16_TFLOPs": achieved,
                          "routing_overhead_ratio": dec_ms / (dec_ms + attn_ms)},
        }
        if set_ms is not None:
            line["breakdown"].update({"decode_set_ms": set_ms, "decode_set_bytes": set_bytes,
                                      "decode_set_GBps": set_bytes / (set_ms * 1e-3) / 1e9,
                                      "decode_set_frac_of_hbm": set_bytes / (set_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                      "decode_set": "40 layers x %d heads x %d rows, L2 flushed, median of 5" % (cfg.H, cfg.nq)})
        if sweep is not None:
            line["density_sweep"] = sweep
        if has_fp8:
            a8 = flops_attn / (attn8_ms * 1e-3) / 1e12
            line["breakdown"].update({"quantize_ms": quant_ms, "attn_fp8_ms": attn8_ms, "attn_fp8_TFLOPs": a8,
                                      "attn_fp8_frac_of_2x_bf16_peak": a8 / (2 * peaks["bf16"]),
                                      "attn_fp8_frac_of_datasheet_4500": a8 / 4500.0,
                                      "attn_fp8_traffic": json.load(open(tp)).get(f"{cfg.name}_fp8_attn_dram_bytes_per_launch")
                                      if os.path.exists(tp) else None})
        if world == 1 and not args.no_cpu_baseline:
            heads = min(cfg.H, 4)
            line["cpu_baseline"] = cpu_baseline(W.scaled(cfg, H=heads), Qb[:, :, :heads].copy(),
                                                Kb[:, :, :heads].copy(), Vb[:, :, :heads].copy(), bm[:heads])
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
    ap.add_argument("--no-fp8", dest="fp8", action="store_false", default=True,
                    help="leave the FP8 leg (quantise + FP8 attention) out of the step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="add the 5/10/25/50/100 %% density sweep of one layer to the JSON line (off by default)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "chorus" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_chorus(args)


if __name__ == "__main__":
    main()
