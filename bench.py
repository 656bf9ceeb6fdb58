#!/usr/bin/env python
"""bench.py -- throughput of the butterfly-filtering hot path on B200.

A step = one pass of the whole hot path (rows A2-A8: sliding norm, data spectra, correlation
core with fused epilogue, threshold + map) of one data segment against the whole template
bank.  Default workload = BASELINE.json configs[3], "Paper-scale bank": 2^23 templates of
L = 4096 against a 16-s segment (65536 samples at 4096 Hz), i.e. exactly the paper's unit:
one correlation = one template x one 16-s segment over all 61441 lags.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Prints ONE JSON line (rank 0).  With N > 1 (torchrun) every rank runs the same job on its own
GPU (replicas only, no collective on the data path); value = all
ranks' correlations / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import bank_grid, default_map_grid, get_config, make_data, sub_bank_indices  # noqa: E402

METRIC = "1-s template correlations/sec"
UNIT = "correlations/s"
REF_LAGS = 61441            # lags of one paper-unit correlation (16 s at 4096 Hz, L = 4096)
FFT_B = 8192                # overlap-save block of the FFT form
SM_COUNT, FP32_LANES = 148, 128


def correlations_per_step(cfg, n_templates):
    """Paper-unit correlations in one step: templates x lags / 61441 (= templates at config 4)."""
    return n_templates * cfg.n_lags / REF_LAGS


def fft_form_flops(cfg, n_templates):
    """Algorithmic flops of one launch of the FFT-form core: per template
    one template FFT + per block one spectral multiply (6 B) and one inverse FFT, each FFT
    counted 5 B log2 B."""
    V = FFT_B - cfg.L + 1
    n_blocks = (cfg.n_lags + V - 1) // V
    fft = 5 * FFT_B * int(math.log2(FFT_B))
    return n_templates * ((n_blocks + 1) * fft + n_blocks * 6 * FFT_B)


def direct_form_flops(cfg, n_templates):
    return n_templates * 2 * (2 * cfg.L * cfg.n_lags)


def max_over_ranks(value: float, world: int, device=None) -> float:
    """The slowest rank's figure (replicas run side by side: the job ends with the last rank)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_value(units_per_rank: float, steps: int, seconds: float, world: int) -> float:
    """Whole-job throughput of `world` independent replicas (replicas
    only): the units all ranks processed over the max-over-ranks time."""
    return world * units_per_rank * steps / seconds


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def host_description():
    """nproc and the CPU model string of the box the CPU baselines ran on."""
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


def time_oracle(cfg, x, f0, f1, seconds):
    """The oracle as it stands on the host cores, on a bounded sample of the workload: as many
    of the given templates (all lags) as fit in about `seconds`.  Returns (corr/s, n, s, cores)."""
    import oracle
    n0 = min(64, len(f0))         # several templates per core, so that the first timing is not noise
    t = time.perf_counter()
    oracle.correlate(x, cfg.fs_hz, cfg.L, f0[:n0], f1[:n0])
    dt0 = time.perf_counter() - t
    n = int(max(n0, min(len(f0), (seconds / max(dt0, 1e-3)) * n0)))
    t = time.perf_counter()
    oracle.correlate(x, cfg.fs_hz, cfg.L, f0[:n], f1[:n])
    dt = time.perf_counter() - t
    return correlations_per_step(cfg, n) / dt, n, dt, oracle.max_threads()


def time_oracle_fft(cfg, x, f0, f1, seconds):
    """The second reported CPU baseline: oracle/fft_variant.py, the float64 numpy
    FFT restatement of the correlation -- the paper's own algorithm (FFT-based
    correlation) on the host, as it stands (numpy's pocketfft, one thread)."""
    from oracle import fft_variant
    n0 = min(4, len(f0))
    t = time.perf_counter()
    fft_variant.correlate_fft(x, cfg.fs_hz, cfg.L, f0[:n0], f1[:n0])
    dt0 = time.perf_counter() - t
    n = int(max(n0, min(len(f0), (seconds / max(dt0, 1e-3)) * n0)))
    t = time.perf_counter()
    fft_variant.correlate_fft(x, cfg.fs_hz, cfg.L, f0[:n], f1[:n])
    dt = time.perf_counter() - t
    return correlations_per_step(cfg, n) / dt, n, dt


def run_reference(args, cfg, rank):
    """--impl reference: the float64 oracle on the box's host cores (rank 0 only)."""
    if rank != 0:
        return
    # the same process environment as the main arm's cpu_baseline leg, which runs after torch has
    # been imported (round 1 measured the oracle 1.5x slower in a process without it: the OpenMP
    # runtime behaves differently); torch does no work here
    import torch  # noqa: F401
    import oracle
    x = make_data(cfg)
    f0a, f1a = bank_grid(cfg)
    idx = sub_bank_indices(cfg, 1 << 16, seed=7, halfwidth=0, max_track=0)
    f0, f1 = f0a[idx], f1a[idx]
    # one step = a bounded sample: about 150 s of CPU work for the whole run, at most 8 s per step,
    # in whole multiples of the thread count (the oracle hands out templates one by one)
    cores = oracle.max_threads()
    n0 = 4 * cores
    t = time.perf_counter()
    oracle.correlate(x, cfg.fs_hz, cfg.L, f0[:n0], f1[:n0])
    per_template = (time.perf_counter() - t) / n0
    step_s = min(8.0, 150.0 / max(args.steps + args.warmup, 1))
    n = int(step_s / max(per_template, 1e-6)) // cores * cores
    n = max(cores, min(len(f0) // max(args.steps + args.warmup, 1), n))
    pos = 0
    for _ in range(args.warmup):
        oracle.correlate(x, cfg.fs_hz, cfg.L, f0[pos:pos + n], f1[pos:pos + n]); pos += n
    t = time.perf_counter()
    for _ in range(args.steps):
        oracle.correlate(x, cfg.fs_hz, cfg.L, f0[pos:pos + n], f1[pos:pos + n]); pos += n
    dt = time.perf_counter() - t
    value = correlations_per_step(cfg, n) * args.steps / dt
    sample = f"{n} templates x all {cfg.n_lags} lags per step, seeded stratified sample of the bank"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {cfg.index} ({cfg.name})", "templates_per_step": n,
                   "n_samples": cfg.n_samples, "L": cfg.L, "lags": cfg.n_lags},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.max_threads(),
                         "kind": "oracle", "sample": sample, **host_description()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def measure_peaks(bfly, device):
    """The unit rates the correlation kernels are bound by, measured on this box in this run
    (bfly_debug_peak; "measured by a microbenchmark on the box")."""
    ffma, _ = bfly.debug_peak(bfly.PEAK_FFMA, 0, 4000, device)
    ffma2, _ = bfly.debug_peak(bfly.PEAK_FFMA2, 0, 4000, device)
    lds, _ = bfly.debug_peak(bfly.PEAK_LDS, 0, 4000, device)
    hmma, _ = bfly.debug_peak(bfly.PEAK_HMMA, 0, 4000, device)
    l2, _ = bfly.debug_peak(bfly.PEAK_L2, 0, 2000, device)
    (umma_ss, _), _ = bfly.debug_peak(bfly.PEAK_UMMA, 1 | 4, 3000, device)
    (umma_ts, _), _ = bfly.debug_peak(bfly.PEAK_UMMA, 2 | 4, 3000, device)
    return {"ffma_tflops": ffma / 1e12, "ffma2_tflops": ffma2 / 1e12, "lds_tbs": lds / 1e12,
            "hmma_tflops": hmma / 1e12, "l2_hot_tbs": l2 / 1e12,
            "tcgen05_f16_m128n256_smem_a_flop_per_clk_sm": umma_ss,
            "tcgen05_f16_m128n256_tmem_a_flop_per_clk_sm": umma_ts,
            "how": "bfly_debug_peak (csrc/bfly_peaks.cu): one kernel per unit on every SM, CUDA events, "
                   "third of three launches"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config, 1-based")
    ap.add_argument("--form", type=int, default=0,
                    help="0 default (= 3), 1 fp32 FFT, 2 fp32 direct, 3 tensor-core FFT (mma.sync), 4 dense tcgen05, "
                         "5 FFT with the transform on tcgen05")
    ap.add_argument("--templates", type=int, default=0,
                    help="development only: first n templates of the bank (not a bench line)")
    ap.add_argument("--cpu-seconds", type=float, default=30.0)
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = get_config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_1802_01685_b200 as bfly

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- inputs (seeded, synthetic) and the persistent bank (A1)
    x = make_data(cfg)
    t0 = time.perf_counter()
    if args.templates:
        f0a, f1a = bank_grid(cfg)
        bank = bfly.make_bank(cfg.fs_hz, cfg.L, f0a[:args.templates], f1a[:args.templates], local)
    else:
        bank = bfly.make_bank_grid(cfg.fs_hz, cfg.L, cfg.f0_lo, cfg.f0_hi, cfg.n_f0,
                                   cfg.f1_lo, cfg.f1_hi, cfg.n_f1, local)
    bank_s = time.perf_counter() - t0
    T = len(bank)
    bank.reserve(cfg.n_samples)
    grid = default_map_grid(cfg)
    dev = torch.device("cuda", local)
    xd = torch.from_numpy(x).to(dev)
    rho = torch.empty(T, dtype=torch.float32, device=dev)
    arg = torch.empty(T, dtype=torch.int32, device=dev)
    m = torch.zeros((grid["n_tbins"], grid["n_fbins"]), dtype=torch.int32, device=dev)
    cnt = torch.zeros(2, dtype=torch.int64, device=dev)
    form = args.form
    chunk = cfg.chunk_samples if cfg.streaming else 0

    def step():
        if cfg.streaming:
            raise SystemExit("config 5 is a parity-test case; bench on configs 1-4")
        bfly.correlate_form(bank, form, xd, 0, None, rho, arg)
        bfly.butterfly_map(bank, rho, arg, cfg.kappa, 0, **grid, map_out=m, counters=cnt)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    m.zero_(); cnt.zero_()
    bank.set_timing(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local) if rank == 0 else None
    barrier(); torch.cuda.synchronize()
    launches0 = bfly.launch_count()
    core_ms = []
    e0.record()
    for _ in range(args.steps):
        step()
        core_ms.append(bank.core_ms())       # waits for this step's core kernel only
    e1.record()
    torch.cuda.synchronize(); barrier()
    launches = bfly.launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    bank.set_timing(False)
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, world, dev)
    corr_step = correlations_per_step(cfg, T)
    value = replicas_value(corr_step, args.steps, ms * 1e-3, world)

    # ---- e2e: the same step through bfly_search_host with HOST buffers (copies inside)
    e2e = None
    if not args.no_e2e:
        xh = torch.from_numpy(x).pin_memory()
        bfly.search_host(bank, xh, chunk, cfg.kappa, **grid)          # warm-up (allocations)
        barrier(); torch.cuda.synchronize()
        t = time.perf_counter()
        for _ in range(args.steps):
            bfly.search_host(bank, xh, chunk, cfg.kappa, **grid)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t
        dt = max_over_ranks(dt, world, dev)
        e2e = {"value": replicas_value(corr_step, args.steps, dt, world), "unit": UNIT,
               "h2d_bytes_per_step": int(x.nbytes),
               "d2h_bytes_per_step": int(T * 8 + m.numel() * 4 + 16)}

    if rank == 0:
        # ---- roofline of the dominant kernel (the correlation core), timed live above; every
        #      denominator is measured in this run by bfly_debug_peak
        core_s = float(np.median(core_ms)) * 1e-3
        is_fft = form in (0, 1, 3, 5)
        is_tc5 = form == 5
        is_tc = form in (0, 3) and cfg.L >= 256           # BFLY_TC_MIN_L (include/bfly.h)
        is_dense = form == 4
        kernel = (("c5_correlate_kernel" if is_tc5 else "tc_correlate_kernel" if is_tc else "fft_correlate_kernel") if is_fft
                  else "dense_tc_kernel" if is_dense else "direct_kernel")
        peaks = measure_peaks(bfly, local)
        mpath = os.path.join(ROOT, "MEASURED_PEAKS.json")
        driver_peaks = json.load(open(mpath)) if os.path.exists(mpath) else {}
        bf16 = driver_peaks.get("bf16_tflops_sustained", 1400.0)
        bf16_basis = ("measured sustained cuBLAS bf16 (MEASURED_PEAKS.json); fp16 operands run at the same rate"
                      if driver_peaks else "fallback 1.4 PFLOP/s sustained (B200_PROFILING.md)")
        alg_flops = fft_form_flops(cfg, T) if is_fft else direct_form_flops(cfg, T)
        fp32_peak = peaks["ffma_tflops"]
        algorithmic = {"flops_per_launch": alg_flops, "tflops": alg_flops / core_s / 1e12,
                       "fp32_fma_peak_tflops_measured": fp32_peak,
                       "ratio_to_fp32_peak": alg_flops / core_s / 1e12 / fp32_peak,
                       "basis": ("(n_blocks + 1) x 5 B log2 B + n_blocks x 6 B per template, B = 8192 "
                                 "(SURVEY 8(d)); the rate a CUDA-core FFT would need -- a yardstick, "
                                 "not the pipe this kernel runs on") if is_fft
                                else "2 quadratures x 2 L n_lags flop per template (SURVEY 8(d))"}
        traffic, traffic_src = None, None
        tpath = os.path.join(ROOT, "profiles", "dram_traffic.json")
        if os.path.exists(tpath):
            tj = json.load(open(tpath))
            per_template = tj.get(kernel + "_bytes_per_template")
            if per_template is not None:
                traffic = per_template * T
                traffic_src = tj.get(kernel + "_source")
        if is_tc:
            # what the kernel executes on its binding units: mma.sync m16n8k16 MMAs
            # (4096 flop each): 512 per block transform, 768 for G; shared-memory bytes: per block
            # X_b staged and read, G read, one exchange written and read (5 x 32 KB), per template
            # g's exchange, G written (3 x 32 KB) and the tail window
            n_blocks, n_tail = divmod(cfg.n_lags, 4096)      # tc_plan (csrc/bfly_fft_tc.cu)
            if n_tail > 4:
                n_blocks, n_tail = n_blocks + 1, 0
            mma_flops = T * (n_blocks * 512 + 768) * 4096
            smem_bytes = T * (n_blocks * 5 * 32768 + 3 * 32768 + (cfg.L * 4 * n_tail))
            t_hmma = mma_flops / (peaks["hmma_tflops"] * 1e12)
            t_smem = smem_bytes / (peaks["lds_tbs"] * 1e12)
            tight = max(t_hmma, t_smem)
            roofline = {"bound": "tensor", "kernel": kernel,
                        "achieved": mma_flops / core_s / 1e12, "peak": peaks["hmma_tflops"],
                        "unit": "TFLOP/s", "frac": mma_flops / core_s / 1e12 / peaks["hmma_tflops"],
                        "flops_per_launch": mma_flops,
                        "flops_basis": "executed: (512 n_blocks + 768) mma.sync.m16n8k16 x 4096 flop per template "
                                       "(the real-embedded radix-8/16 DFT matrices of the FFT; DESIGN.md 6.1)",
                        "peak_basis": "measured in this run (bfly_debug_peak): independent mma.sync.m16n8k16 "
                                      "f16->f32 on every SM, the pipe this kernel's MMAs run on",
                        "bounds_s": {"mma_sync": t_hmma, "shared_memory": t_smem},
                        "smem_bytes_per_launch": smem_bytes,
                        "frac_of_tightest_bound": tight / core_s,
                        "tightest_bound": "shared_memory" if t_smem >= t_hmma else "mma_sync",
                        "vs_tcgen05_rate": {"frac": mma_flops / core_s / 1e12 / bf16, "peak": bf16,
                                            "peak_basis": bf16_basis}}
        elif is_tc5:
            # executed tcgen05 flops: per pair of transforms 8 MMAs of 128 x 256 x 16 and 16 of 128 x 128 x 16;
            # per template one G pair + ceil(n_blocks / 2) block pairs
            n_blocks, n_tail = divmod(cfg.n_lags, 4096)
            if n_tail > 4:
                n_blocks += 1
            pairs = 1 + (n_blocks + 1) // 2
            mma_flops = T * pairs * (8 * 2 * 128 * 256 * 16 + 16 * 2 * 128 * 128 * 16)
            roofline = {"bound": "tensor", "kernel": kernel, "achieved": mma_flops / core_s / 1e12, "peak": bf16,
                        "unit": "TFLOP/s", "frac": mma_flops / core_s / 1e12 / bf16, "flops_per_launch": mma_flops,
                        "flops_basis": "executed: per pair of transforms 8 tcgen05.mma 128x256x16 + 16 of 128x128x16 "
                                       "(real-embedded 64-point DFT matrices; DESIGN.md 6.8)",
                        "peak_basis": bf16_basis}
        elif is_dense:
            roofline = {"bound": "tensor", "kernel": kernel, "achieved": alg_flops / core_s / 1e12,
                        "peak": bf16, "unit": "TFLOP/s", "frac": alg_flops / core_s / 1e12 / bf16,
                        "flops_per_launch": alg_flops, "flops_basis": algorithmic["basis"],
                        "peak_basis": bf16_basis}
        else:
            roofline = {"bound": "alu", "kernel": kernel, "achieved": alg_flops / core_s / 1e12,
                        "peak": fp32_peak, "unit": "TFLOP/s", "frac": alg_flops / core_s / 1e12 / fp32_peak,
                        "flops_per_launch": alg_flops, "flops_basis": algorithmic["basis"],
                        "peak_basis": "measured in this run (bfly_debug_peak): independent FFMA chains on every SM"}
        roofline.update({"traffic": traffic, "traffic_source": traffic_src,
                         "algorithmic_bytes_per_launch": T * 32,
                         "kernel_ms": core_s * 1e3, "kernel_ms_all": [float(v) for v in core_ms],
                         "kernel_share_of_step": core_s * 1e3 * args.steps / ms,
                         "algorithmic": algorithmic, "peaks_measured": peaks})
        npath = os.path.join(ROOT, "profiles", "ncu_utilisation.json")
        if os.path.exists(npath):
            roofline["ncu"] = json.load(open(npath)).get(kernel)
        f0a, f1a = bank_grid(cfg)
        # ---- the other tensor-core form beside the chosen one ("chosen by measurement"): the dense
        #      tcgen05 contraction on the first 4 waves of template tiles (cost is linear in T)
        other = None
        if is_tc and form in (0, 3) and not args.templates and not cfg.streaming:
            nd = min(T, 4 * SM_COUNT * 128)
            dbank = bfly.make_bank(cfg.fs_hz, cfg.L, f0a[:nd], f1a[:nd], local)
            dbank.reserve(cfg.n_samples)
            dbank.set_timing(True)
            dms = []
            for i in range(3):
                bfly.correlate_form(dbank, 4, xd, 0, None, rho[:nd], arg[:nd])
                if i:
                    dms.append(dbank.core_ms())
            dsec = float(np.mean(dms)) * 1e-3
            dfl = direct_form_flops(cfg, nd)
            other = {"dense_tc": {"kernel": "dense_tc_kernel", "templates": nd, "kernel_ms": dsec * 1e3,
                                  "value": correlations_per_step(cfg, nd) / dsec, "unit": UNIT,
                                  "roofline": {"bound": "tensor", "achieved": dfl / dsec / 1e12, "peak": bf16,
                                               "unit": "TFLOP/s", "frac": dfl / dsec / 1e12 / bf16,
                                               "peak_basis": bf16_basis},
                                  "note": "same rows A3-A7 as a Hankel x template contraction on tcgen05; "
                                          "109x the flops of the FFT form, hence not the default"}}
            # the FFT form with its transform on tcgen05 (BFLY_FORM_FFT_TC5), same partial bank
            dms = []
            for i in range(3):
                bfly.correlate_form(dbank, 5, xd, 0, None, rho[:nd], arg[:nd])
                if i:
                    dms.append(dbank.core_ms())
            t5s = float(np.mean(dms)) * 1e-3
            other["fft_tc5"] = {"kernel": "c5_correlate_kernel", "templates": nd, "kernel_ms": t5s * 1e3,
                                "value": correlations_per_step(cfg, nd) / t5s, "unit": UNIT,
                                "note": "the same overlap-save FFT with the length-8192 transform as 64 x 128 on "
                                        "tcgen05.mma (DFT matrices in tensor memory); measured slower than the "
                                        "mma.sync transform (DESIGN.md 10), hence not the default"}
            # several segments per launch (bfly_correlate_multi: the two detectors of PAPER.md:124, the
            # chunks of a stream): two 16-s segments through one launch against one call each
            x2 = torch.flip(xd, dims=[0]).contiguous()
            def _ms(fn, reps=3):
                fn(); torch.cuda.synchronize()
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a0.record()
                for _ in range(reps):
                    fn()
                a1.record(); torch.cuda.synchronize()
                return a0.elapsed_time(a1) / reps
            t_multi = _ms(lambda: bfly.correlate_multi(dbank, [xd, x2]))
            t_each = _ms(lambda: (bfly.correlate(dbank, xd), bfly.correlate(dbank, x2)))
            other["multi_segment"] = {"kernel": "tc_correlate_kernel<MULTI>", "templates": nd, "segments": 2,
                                      "ms_one_launch": t_multi, "ms_one_call_each": t_each,
                                      "value": 2 * correlations_per_step(cfg, nd) / (t_multi * 1e-3), "unit": UNIT,
                                      "note": "synthesis and the transform of g once per template for both segments; "
                                              "results bit-identical to one call per segment"}
            # the paper's own reduction on the same kernel: sigma by Parseval + all tails above
            # kappa sigma (bfly_tails), whole bank, kappa = 5.5 (about 1e5 hits in noise)
            bank.set_timing(True)
            tms, nh = [], 0
            for i in range(2):
                sg, hj, hl, hr, nhits = bfly.tails(bank, xd, 5.5, 1 << 22)
                if i:
                    tms.append(bank.core_ms())
                nh = int(nhits.item())
            tsec = float(np.mean(tms)) * 1e-3
            other["tails"] = {"kernel": "tc_correlate_kernel<TAILS>", "templates": T, "kappa_sigma": 5.5,
                              "kernel_ms": tsec * 1e3, "value": corr_step / tsec, "unit": UNIT, "hits": nh,
                              "note": "PAPER.md:70, 120: sigma per template by the Parseval predictor, "
                                      "every lag with rho > kappa sigma appended to a hit list"}
            bank.set_timing(False)
        # ---- the oracle beside it, on this box's host cores, on a bounded sample
        idx = sub_bank_indices(cfg, 8192, seed=7, halfwidth=0, max_track=0)
        cv, cn, cs, cores = time_oracle(cfg, x, f0a[idx], f1a[idx], args.cpu_seconds)
        fv, fn, fs_ = time_oracle_fft(cfg, x, f0a[idx], f1a[idx], min(args.cpu_seconds, 15.0))
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "f16 mma operands, f32 accumulate" if (is_tc or is_dense) else "f32", "data": "synthetic",
            "config": {"workload": f"config {cfg.index} ({cfg.name})", "templates": T,
                       "n_samples": cfg.n_samples, "L": cfg.L, "lags": cfg.n_lags,
                       "form": ("fft_tc5" if is_tc5 else "fft_tc" if is_tc else "fft") if is_fft
                               else "dense_tc" if is_dense else "direct",
                       "l2": "inputs larger than L2 (bank parameters + outputs "
                             f"{(T * 48) >> 20} MiB per step)",
                       "parallelism": "replicas" if world > 1 else "single GPU",
                       "bank_build_s": bank_s,
                       "partial_bank_dev_run": bool(args.templates)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "other_forms": other,
            "pairs_per_s": world * T * cfg.n_lags * args.steps / (ms * 1e-3),
            "direct_equiv_mac_per_s": world * T * cfg.n_lags * 2 * cfg.L * args.steps / (ms * 1e-3),
            "cpu_baseline": {"value": cv, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{cn} templates x all {cfg.n_lags} lags of config "
                                       f"{cfg.index} in {cs:.1f} s (float64 direct, OpenMP)",
                             **host_description()},
            "cpu_baseline_fft": {"value": fv, "unit": UNIT, "cores": 1, "kind": "oracle (float64 FFT variant)",
                                 "sample": f"{fn} templates x all {cfg.n_lags} lags in {fs_:.1f} s "
                                           "(oracle/fft_variant.py: numpy FFT correlation, the paper's "
                                           "algorithm, PAPER.md:70, one thread)"},
        }
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
