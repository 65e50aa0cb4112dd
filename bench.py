#!/usr/bin/env python
"""bench.py -- throughput of the batched likelihood hot path on B200 (one JSON line on stdout).

  python bench.py --gpus N --steps K --warmup W [--config 2|3|4] [--impl reference]

A "step" is one pass of the whole hot path (per-sample constants ->
fused per-bin kernel -> fixed-order combine) over one batch of B synthetic samples: one
pespace_loglike call.  The workload at N=1 is BASELINE.json configs[1] ("config 2":
B=4096 x N=262144, one LISA-like detector, (2,2) mode), the one the metric is quoted on.
With N>1 GPUs (torchrun) every rank evaluates its own batch of B samples on replicated
data -- no data-path collective -- so scaling is "weak" and `value` is the whole-job rate.

value     device-timed lnL evaluations/s, inputs resident in HBM (CUDA events, max over ranks)
e2e       the same metric through the C ABI with HOST buffers (pespace_loglike_host):
          H2D of params + data + psd and D2H of lnL inside the timed region
roofline  the dominant kernel (loglike_kernel) against the FP64 ALU peak
cpu_baseline / --impl reference   the oracle, as it stands, on the box's host cores
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2602_12011_b200 import dist as pdist          # noqa: E402
from paper_2602_12011_b200 import workloads as W         # noqa: E402

# ---- roofline constants:
# FP64 ALU peak: 148 SMs x 64 FP64 FMA lanes x 2 flop x clocks.max.sm (1965 MHz) = 37.23 TFLOP/s.
# The pespace_fp64_peak DFMA micro-benchmark measures ~36.6 TFLOP/s on this pool (reported too).
SM_COUNT, FP64_LANES_PER_SM = 148, 64
# Executed FP64 work of loglike_kernel per bin-eval, from the committed ncu profile
# (profiles/r01_*): thread-level DFMA, DMUL, DADD counts divided by B*N.  flop = 2*DFMA+DMUL+DADD.
EXEC_FP64_PER_BIN_EVAL = {
    2: {"dfma": 0.0, "dmul": 0.0, "dadd": 0.0},
    3: {"dfma": 0.0, "dmul": 0.0, "dadd": 0.0},
    4: {"dfma": 0.0, "dmul": 0.0, "dadd": 0.0},
}
# SURVEY.md 8(d) algorithmic estimate (transcendentals costed: sincos 40, cbrt 30, log 35, ...)
SURVEY_FLOP_PER_BIN_EVAL = {2: 970.0, 3: 4500.0, 4: 11200.0}
METRIC, UNIT = "lnL_evals_per_sec", "lnL/s"


def load_exec_counts():
    path = os.path.join(ROOT, "profiles", "fp64_ops_per_bin_eval.json")
    if os.path.exists(path):
        with open(path) as fh:
            for k, v in json.load(fh).items():
                if k.isdigit():
                    EXEC_FP64_PER_BIN_EVAL[int(k)] = v


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.idx)], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        rows = [r.split(",") for r in open(self.tmp.name).read().strip().splitlines() if r.strip()]
        os.unlink(self.tmp.name)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[5:9]):
                if v.strip().lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [s for s, p in zip(sm, pw) if p > 0.5 * max(pw)] or sm
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_timed(wl, n_samples, steps: int, warmup: int, target_s: float = 12.0):
    """Time the oracle, as it stands, on `n_samples` samples x all N bins per step.
    n_samples=None: sized from a one-sample-per-core calibration pass for ~target_s of wall time."""
    import oracle
    psd = wl.psd()
    data = wl.data(lambda p, fr, m: oracle.response(p, fr, m))
    cores = oracle.get_threads()
    t0 = time.perf_counter()
    oracle.loglike(wl.params[:cores], data, psd, wl.grid, wl.model)          # warm-up + calibration
    t_cal = time.perf_counter() - t0
    if n_samples is None:
        n_samples = int(min(wl.B, max(cores, cores * round(target_s / max(t_cal, 1e-3)))))
    idx = np.linspace(0, wl.B - 1, n_samples).astype(int)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.loglike(wl.params[idx], data, psd, wl.grid, wl.model)
    dt = time.perf_counter() - t0
    return n_samples * steps / dt, dt / steps, cores, n_samples


def run_reference(args):
    rank, _, world = pdist.env_world()
    if rank != 0:
        return
    wl = W.config(args.config)
    rate, sec_per_step, cores, n = oracle_timed(wl, args.ref_samples, args.steps, min(args.warmup, 1),
                                                target_s=max(2.0, 60.0 / max(1, args.steps)))
    sample = f"{n} of {wl.B} samples (evenly spaced) x all {wl.grid.N} bins per step, OpenMP over samples"
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec_per_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "bin_evals_per_sec": rate * wl.grid.N,
        "config": workload_config(wl, args, l2="n/a (CPU)"),
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(wl, args, l2):
    return {"workload": f"config{args.config}: B={wl.B} x N={wl.grid.N}, {len(wl.model.detectors)} detector(s) "
                        f"[{', '.join(d.name for d in wl.model.detectors)}], mode_mask={wl.model.mode_mask}, "
                        f"TDI {wl.model.detectors[0].tdi_gen / 10:.1f}, f0={wl.grid.f0} Hz, df=1/(30 d)",
            "B_per_gpu": wl.B, "N_bins": wl.grid.N, "n_det": len(wl.model.detectors),
            "mode_mask": wl.model.mode_mask, "parallelism": f"sample-sharded x{args.gpus} (no data-path collective)",
            "l2": l2}


def run_ours(args):
    import torch
    from paper_2602_12011_b200 import binding as P      # fails loudly if libpespace.so is missing

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle timing)")
    rank, local_rank, world = pdist.init("nccl")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    load_exec_counts()

    # ---- inputs: synthetic, seeded; the injection comes from this library's own response call
    n_batches = 4
    wls = [W.config(args.config, param_seed=pdist.rank_seed(1000 + i, rank)) for i in range(n_batches)]
    wl = wls[0]
    B, N = wl.B, wl.grid.N
    freqs_d = torch.from_numpy(wl.grid.freqs()).to(device)

    def gpu_response(p, fr, m):
        return P.response(torch.from_numpy(np.ascontiguousarray(p)).to(device), freqs_d, m).cpu().numpy()

    data_h = np.ascontiguousarray(wl.data(gpu_response))
    psd_h = np.ascontiguousarray(wl.psd())
    lik = P.Likelihood(torch.from_numpy(data_h).to(device), torch.from_numpy(psd_h).to(device), wl.grid, wl.model, B)
    params_d = [torch.from_numpy(w.params).to(device) for w in wls]
    out_d = torch.empty(B, dtype=torch.float64, device=device)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)   # > 126 MB L2

    def step(i):
        flush.zero_()
        lik(params_d[i % n_batches], out_d)

    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()

    # ---- timed region: exactly K steps, device events, barrier + sync on both sides
    sampler = ClockSampler(local_rank)
    sampler.start()
    P.profile_enable(True)
    P.profile_read()
    launches0 = P.launch_count()
    pdist.barrier(device)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.steps):
        step(i)
    e1.record()
    torch.cuda.synchronize()
    pdist.barrier(device)
    elapsed_ms = e0.elapsed_time(e1)
    launches = P.launch_count() - launches0
    main_ms, main_launches = P.profile_read()
    P.profile_enable(False)
    clocks = sampler.stop()
    lnL_last = out_d.cpu().numpy()
    if not np.all(np.isfinite(lnL_last)):
        raise SystemExit("bench.py: non-finite lnL in the timed region")

    max_ms, total_units = pdist.aggregate(elapsed_ms, B * args.steps, device)
    value = total_units / (max_ms * 1e-3)

    # ---- e2e: host buffers through pespace_loglike_host (copies inside the call)
    e2e_steps = max(1, min(args.steps, 10))
    P.loglike_host(wls[0].params, data_h, psd_h, wl.grid, wl.model)        # warm-up
    pdist.barrier(device)
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        lnL_host = P.loglike_host(wls[i % n_batches].params, data_h, psd_h, wl.grid, wl.model)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_max_ms, e2e_units = pdist.aggregate(e2e_ms, B * e2e_steps, device)
    h2d = wl.params.nbytes + data_h.nbytes + psd_h.nbytes
    d2h = lnL_host.nbytes

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (per launch, timed live with CUDA events in the library)
    peak_tflops = SM_COUNT * FP64_LANES_PER_SM * 2 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    dfma_tflops, _ = P.fp64_peak(8192)
    n_det = len(wl.model.detectors)
    kern_ms = main_ms / max(1, main_launches)                 # one launch = one detector, B x N bin-evals
    ops = EXEC_FP64_PER_BIN_EVAL.get(args.config, {"dfma": 0, "dmul": 0, "dadd": 0})
    flop_per_unit = (2.0 * ops["dfma"] + ops["dmul"] + ops["dadd"]) / n_det   # per (sample, bin, detector)
    inst_per_unit = (ops["dfma"] + ops["dmul"] + ops["dadd"]) / n_det
    achieved = flop_per_unit * B * N / (kern_ms * 1e-3) / 1e12
    survey_unit = SURVEY_FLOP_PER_BIN_EVAL[args.config] / n_det
    roofline = {
        "bound": "alu", "kernel": "loglike_kernel", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops, "traffic": None,
        "peak_source": "148 SM x 64 FP64 lanes x 2 x clocks.max.sm (DESIGN.md); DFMA micro-benchmark alongside",
        "peak_dfma_measured": dfma_tflops,
        "fp64_pipe_frac": inst_per_unit * B * N / (kern_ms * 1e-3) / (peak_tflops * 1e12 / 2.0),
        "flop_per_launch": flop_per_unit * B * N, "kernel_ms": kern_ms, "kernel_launches": main_launches,
        "kernel_share_of_step": main_ms / elapsed_ms,
        "flop_basis": "executed FP64 (2*DFMA+DMUL+DADD per bin-eval from ncu, profiles/fp64_ops_per_bin_eval.json)",
        "survey_algorithmic": {"flop_per_bin_eval": SURVEY_FLOP_PER_BIN_EVAL[args.config],
                               "achieved": survey_unit * B * N / (kern_ms * 1e-3) / 1e12,
                               "frac": survey_unit * B * N / (kern_ms * 1e-3) / 1e12 / peak_tflops},
    }
    traffic_path = os.path.join(ROOT, "profiles", "dram_traffic_per_launch.json")
    if os.path.exists(traffic_path):
        roofline["traffic"] = json.load(open(traffic_path)).get(str(args.config))

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        rate, sec, cores, n_ref = oracle_timed(W.config(args.config), args.ref_samples, 1, 1)
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{n_ref} of {B} samples (evenly spaced) x all {N} bins, one pass, "
                                  f"{sec:.1f} s, OpenMP over samples"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "bin_evals_per_sec": value * N,
        "config": workload_config(wl, args, l2="256 MiB buffer rewritten before every step, inside the timed region"),
        "clocks": clocks,
        "e2e": {"value": e2e_units / (e2e_max_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                "api": "pespace_loglike_host (pageable host buffers; cudaMalloc/free inside the call)"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "lnL_check": {"min": float(lnL_last.min()), "max": float(lnL_last.max())},
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4])
    ap.add_argument("--ref-samples", type=int, default=None,
                    help="samples per oracle pass (default: sized for ~15 s of CPU work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
