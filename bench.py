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

# ---- roofline constants
# FP64 ALU peak: 148 SMs x 64 FP64 lanes x 2 flop x clocks.max.sm (1965 MHz) = 37.22 TFLOP/s.  The
# library's own DFMA micro-benchmark (pespace_fp64_peak) is run in the same process and reported next
# to it: mode 0 (two register operands) reaches ~98 % of that figure, mode 1 (three distinct register
# operands, the common case in this kernel) ~66 % (profiles/r01_fp64_operand_bandwidth.md).
SM_COUNT, FP64_LANES_PER_SM = 148, 64
# FP64 operations of loglike_kernel per (sample, bin, detector), thread level, counted by ncu
# (smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum / (B*N), profiles/r01_kernels_ncu.md).
# They equal the operation list of the reduced formulas in DESIGN.md ("Algorithmic work") to <1 %; the
# kernel has no redundant evaluation, so executed = algorithmic.  flop = 2*DFMA + DMUL + DADD.
FP64_OPS_PER_UNIT = {
    # (kernel, detector kind, mode-class mask): per (sample, bin, detector); profiles/r01_kernels_ncu.md
    ("loglike", 0, 2): {"dfma": 140.00, "dmul": 53.02, "dadd": 40.53},      # kind 0, (2,2) only  -- config 2
    ("loglike", 0, 15): {"dfma": 554.00, "dmul": 188.11, "dadd": 101.08},   # kind 0, five modes  -- configs 3, 4
    ("loglike", 1, 15): {"dfma": 526.00, "dmul": 224.11, "dadd": 109.08},   # kind 1, five modes  -- config 4
    ("fisher", 0, 15): {"dfma": 3150.00, "dmul": 1246.25, "dadd": 640.61},  # config 5
    ("fisher", 1, 15): {"dfma": 3030.00, "dmul": 1330.25, "dadd": 632.61},
    ("loglike_tab", 0, 2): {"dfma": 136.00, "dmul": 52.03, "dadd": 46.03},   # --waveform tab, config 2 (one mode)
}
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel (same ncu captures; config 4:
# mean of the three launches of a step)
DRAM_TRAFFIC_PER_LAUNCH = {2: 35.91e6 + 5.18e6, 3: 36.18e6 + 5.39e6, 4: (40.4e6 + 36.6e6 + 42.1e6 + 37.2e6 + 41.3e6 + 37.9e6) / 3,
                           5: 36.9e6 + 57.6e6}
# SURVEY.md 8(d) survey-time estimate (library-cost transcendentals: sincos 40, cbrt 30, log 35, ...);
# kept for reference only -- the reduced algorithm needs less than half of it.
SURVEY_FLOP_PER_BIN_EVAL = {2: 970.0, 3: 4500.0, 4: 11200.0, 5: 100000.0}
OPS_SOURCE = "profiles/r01_kernels_ncu.md"
METRIC, UNIT = "lnL_evals_per_sec", "lnL/s"
FISHER_METRIC, FISHER_UNIT = "fisher_evals_per_sec", "F/s"     # --config 5 only (S10: F and grad per sample)


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


FISHER_REF_BINS = 8192   # the oracle's Fisher pass costs ~45 core-seconds per sample at N = 262144: time a bin subset


def oracle_timed(config: int, n_samples, steps: int, target_s: float = 12.0, tab_nodes: int = 0):
    """Time the oracle, as it stands, on a bounded sample of the workload: `n_samples` samples (None: sized from a
    one-sample-per-core calibration pass for ~target_s of wall time) x all N bins per step; for the Fisher path
    (config 5) x the first FISHER_REF_BINS bins, the rate scaled by FISHER_REF_BINS / N (the cost per bin is uniform).
    -> (rate in full-N evaluations/s, seconds per step, cores, description of the sample)."""
    import oracle
    fisher = config == 5
    full = W.config(config)
    wl = W.config(config, N=FISHER_REF_BINS) if fisher else full
    scale = wl.grid.N / full.grid.N
    psd = wl.psd()
    cores = oracle.get_threads()
    if tab_nodes:
        f_all = wl.grid.freqs()
        fnodes = W.log_nodes(f_all[0], f_all[-1], tab_nodes)
        tab = lambda p: W.chirp_table(p, wl.model.mode_mask, fnodes)
        data = wl.data(lambda p, fr, m: oracle.response_tab(p, tab(p), fr, m))
        call = lambda p: oracle.loglike_tab(p, tab(p), data, psd, wl.grid, wl.model)
    else:
        data = wl.data(lambda p, fr, m: oracle.response(p, fr, m))
    if tab_nodes:
        pass
    elif fisher:
        call = lambda p: oracle.fisher(p, data, psd, wl.grid, wl.model)
    else:
        call = lambda p: oracle.loglike(p, data, psd, wl.grid, wl.model)
    t0 = time.perf_counter()
    call(wl.params[:cores])                                                  # warm-up + calibration
    t_cal = time.perf_counter() - t0
    if n_samples is None:
        n_samples = int(min(wl.B, max(cores, cores * round(target_s / max(t_cal, 1e-3)))))
    idx = np.linspace(0, wl.B - 1, n_samples).astype(int)
    t0 = time.perf_counter()
    for _ in range(steps):
        call(wl.params[idx])
    dt = time.perf_counter() - t0
    # one-thread figure (the paper's own CPU protocol is one core): two samples on one thread
    oracle.set_threads(1)
    t1 = time.perf_counter()
    call(wl.params[idx[:2]])
    one_thread = 2 / (time.perf_counter() - t1) * scale
    oracle.set_threads(0)
    oracle_timed.one_thread = one_thread
    bins = f"all {wl.grid.N} bins" if not fisher else f"the first {wl.grid.N} of {full.grid.N} bins (rate scaled by {scale:.5f})"
    desc = (f"{n_samples} of {full.B} samples (evenly spaced) x {bins} per pass, {steps} pass(es), "
            f"{dt / steps:.1f} s per pass, OpenMP over samples")
    return n_samples * steps / dt * scale, dt / steps, cores, desc


def run_reference(args):
    rank, _, world = pdist.env_world()
    if rank != 0:
        return
    wl = W.config(args.config)
    fisher_mode = args.config == 5
    METRIC, UNIT = (FISHER_METRIC, FISHER_UNIT) if fisher_mode else (globals()["METRIC"], globals()["UNIT"])
    rate, sec_per_step, cores, sample = oracle_timed(args.config, args.ref_samples, args.steps,
                                                     target_s=max(2.0, 60.0 / max(1, args.steps)),
                                                     tab_nodes=args.tab_nodes if args.waveform == "tab" else 0)
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec_per_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "bin_evals_per_sec": rate * wl.grid.N,
        "config": workload_config(wl, args, l2="n/a (CPU)"),
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "value_one_thread": oracle_timed.one_thread},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(wl, args, l2):
    tab = f" + tabulated mode waveforms (K={args.tab_nodes} log-spaced nodes)" if args.waveform == "tab" else ""
    if getattr(args, "grad_only", False) and args.config == 5:
        tab += " (gradient only)"
    return {"workload": f"config{args.config}{tab}: B={wl.B} x N={wl.grid.N}, {len(wl.model.detectors)} detector(s) "
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

    # ---- inputs: synthetic, seeded; the injection comes from this library's own response call
    fisher_mode = args.config == 5
    tab_mode = args.waveform == "tab"
    mixed_mode = args.precision == "mixed"
    if mixed_mode and (fisher_mode or tab_mode):
        raise SystemExit("bench.py: --precision mixed applies to the analytic likelihood configs 2-4")
    if tab_mode and fisher_mode:
        raise SystemExit("bench.py: --waveform tab applies to the likelihood configs 2-4")
    n_batches = 2 if tab_mode else 4
    wls = [W.config(args.config, param_seed=pdist.rank_seed(1000 + i, rank)) for i in range(n_batches)]
    wl = wls[0]
    B, N = wl.B, wl.grid.N
    freqs_d = torch.from_numpy(wl.grid.freqs()).to(device)

    def gpu_response(p, fr, m):
        return P.response(torch.from_numpy(np.ascontiguousarray(p)).to(device), freqs_d, m).cpu().numpy()

    if tab_mode:
        # synthetic tables (workloads.chirp_table: inspiral-shaped power laws) on K log-spaced nodes covering the grid
        f_all = wl.grid.freqs()
        fnodes = W.log_nodes(f_all[0], f_all[-1], args.tab_nodes)
        tabs_h = [tuple(torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
                        for x in W.chirp_table(w.params, wl.model.mode_mask, fnodes)) for w in wls]
        tabs_d = [P.WaveTable(*(x.to(device) for x in t)) for t in tabs_h]
        inj_tab = P.WaveTable(*(torch.from_numpy(np.ascontiguousarray(x)).to(device)
                                for x in W.chirp_table(wl.theta_inj[None], wl.model.mode_mask, fnodes)))

        def gpu_response(p, fr, m):                                   # noqa: F811  (injection from the same tables)
            return P.response_tab(torch.from_numpy(np.ascontiguousarray(p)).to(device), inj_tab, freqs_d, m).cpu().numpy()

    # host copies live in pinned memory: the e2e leg copies them to the device every step
    data_h = torch.from_numpy(np.ascontiguousarray(wl.data(gpu_response))).pin_memory()
    psd_h = torch.from_numpy(np.ascontiguousarray(wl.psd())).pin_memory()
    params_h = [torch.from_numpy(np.ascontiguousarray(w.params)).pin_memory() for w in wls]
    params_d = [p.to(device) for p in params_h]
    if fisher_mode:
        fis = P.Fisher(data_h.to(device), psd_h.to(device), wl.grid, wl.model, B)
        F_d = torch.empty((B, P.NPAR, P.NPAR), dtype=torch.float64, device=device)
        g_d = torch.empty((B, P.NPAR), dtype=torch.float64, device=device)
    elif tab_mode:
        lik = P.LikelihoodTab(data_h.to(device), psd_h.to(device), wl.grid, wl.model, B)
        out_d = torch.empty(B, dtype=torch.float64, device=device)
    else:
        lik = P.Likelihood(data_h.to(device), psd_h.to(device), wl.grid, wl.model, B)
        out_d = torch.empty(B, dtype=torch.float64, device=device)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)   # > 126 MB L2

    def step(i):
        flush.zero_()
        if fisher_mode:
            fis(params_d[i % n_batches], F_d, g_d, grad_only=args.grad_only)
        elif tab_mode:
            lik(params_d[i % n_batches], tabs_d[i % n_batches], out_d)
        else:
            lik(params_d[i % n_batches], out_d, mixed=mixed_mode)

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
    last = ((g_d if args.grad_only else F_d) if fisher_mode else out_d).cpu().numpy()
    if not np.all(np.isfinite(last)):
        raise SystemExit("bench.py: non-finite result in the timed region")

    max_ms, total_units = pdist.aggregate(elapsed_ms, B * args.steps, device)
    value = total_units / (max_ms * 1e-3)

    # ---- e2e: HOST buffers through the C ABI (pespace_session_*): every step copies that step's inputs
    # (theta, data set, PSD) from pinned host memory to the device and reads the result back, all inside
    # the timed region.  e2e_resident_data: the sampler-facing use, data set copied once, theta per step.
    e2e_steps = max(1, min(args.steps, 10))
    ses = P.Session(wl.grid, wl.model, B, want_fisher=fisher_mode)
    if tab_mode:
        res_h = torch.empty(B, dtype=torch.float64).pin_memory()

        def e2e_step(i, copy_data):
            if copy_data:
                ses.set_data(data_h, psd_h)
            ses.loglike_tab(params_h[i % n_batches], tabs_h[i % n_batches], res_h)
    grad_h = torch.empty((B, P.NPAR), dtype=torch.float64).pin_memory()
    if not tab_mode:
        res_h = torch.empty((B, P.NPAR, P.NPAR) if fisher_mode else (B,), dtype=torch.float64).pin_memory()

        def e2e_step(i, copy_data):
            if copy_data:
                ses.set_data(data_h, psd_h)
            if fisher_mode:
                ses.fisher(params_h[i % n_batches], True, res_h, grad_h, grad_only=args.grad_only)
            else:
                ses.loglike(params_h[i % n_batches], res_h, mixed=mixed_mode)

    e2e = {}
    for key, copy_data in (("full", True), ("resident", False)):
        e2e_step(0, True)                                                   # warm-up
        pdist.barrier(device)
        t0 = time.perf_counter()
        for i in range(e2e_steps):
            e2e_step(i, copy_data)
        e2e_ms = (time.perf_counter() - t0) * 1e3                           # the calls are synchronous
        e2e_max_ms, e2e_units = pdist.aggregate(e2e_ms, B * e2e_steps, device)
        e2e[key] = e2e_units / (e2e_max_ms * 1e-3)
    ses.close()
    nbytes = lambda t: t.numel() * t.element_size()
    h2d = nbytes(params_h[0]) + nbytes(data_h) + nbytes(psd_h) + (sum(nbytes(x) for x in tabs_h[0]) if tab_mode else 0)
    d2h = nbytes(res_h) + (nbytes(grad_h) if fisher_mode else 0)

    # ---- optional: pespace_response on a slice of the batch (48 B written per (sample, bin, detector))
    response_info = None
    if args.response and not tab_mode:
        Br = min(B, args.response_batch)
        out_r = torch.empty((Br, len(wl.model.detectors), 3, N, 2), dtype=torch.float64, device=device)
        pr = params_d[0][:Br].contiguous()
        for _ in range(2):
            P.response(pr, freqs_d, wl.model, out_r)
        torch.cuda.synchronize()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        for _ in range(5):
            P.response(pr, freqs_d, wl.model, out_r)
        r1.record()
        torch.cuda.synchronize()
        r_ms = r0.elapsed_time(r1) / 5
        response_info = {"batch": Br, "ms_per_call": r_ms, "bin_evals_per_sec": Br * N / (r_ms * 1e-3),
                         "bytes_written_per_call": out_r.numel() * 8,
                         "write_gbs": out_r.numel() * 8 / (r_ms * 1e-3) / 1e9}
        del out_r

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (per launch, timed live with CUDA events in the library)
    kernel = "fisher" if fisher_mode else ("loglike_tab" if tab_mode else ("loglike_mixed" if mixed_mode else "loglike"))
    metric, unit = (FISHER_METRIC, FISHER_UNIT) if fisher_mode else (METRIC, UNIT)
    peak_tflops = SM_COUNT * FP64_LANES_PER_SM * 2 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    dfma_tflops, _ = P.fp64_peak(8192, mode=0)
    dfma3_tflops, _ = P.fp64_peak(8192, mode=1)
    n_det = len(wl.model.detectors)
    kern_ms = main_ms / max(1, main_launches)                 # one launch = one detector, B x N (sample, bin) units
    cmask = (2 if wl.model.mode_mask & 9 else 0) | (1 if wl.model.mode_mask & 2 else 0) | \
            (4 if wl.model.mode_mask & 4 else 0) | (8 if wl.model.mode_mask & 16 else 0)
    per_det = [FP64_OPS_PER_UNIT.get((kernel, d.kind, cmask)) for d in wl.model.detectors]
    known = [o for o in per_det if o]
    ops = {k: sum(o[k] for o in known) / len(known) for k in ("dfma", "dmul", "dadd")} if len(known) == n_det else None
    if fisher_mode and args.grad_only:
        ops = None                    # no ncu op counts for the gradient-only variant
    roofline = {"bound": "alu", "kernel": f"{kernel}_kernel", "achieved": None, "peak": peak_tflops,
                "unit": "TFLOP/s", "frac": None, "traffic": DRAM_TRAFFIC_PER_LAUNCH.get(args.config)}
    if ops:
        flop_per_unit = 2.0 * ops["dfma"] + ops["dmul"] + ops["dadd"]
        inst_per_unit = ops["dfma"] + ops["dmul"] + ops["dadd"]
        achieved = flop_per_unit * B * N / (kern_ms * 1e-3) / 1e12
        # issue cost on the FP64 pipe (profiles/r01_fp64_operand_bandwidth.md): one 64-bit register operand
        # per cycle and SM sub-partition, at least 2 cycles per instruction -> a DFMA with three distinct
        # register operands takes 3 cycles.  The bound below charges every DFMA 3 cycles and DMUL/DADD 2.
        cyc = 3.0 * ops["dfma"] + 2.0 * (ops["dmul"] + ops["dadd"])
        t_operand = cyc * (B * N / 32.0) / (SM_COUNT * 4) / ((clocks.get("sm_max_mhz") or 1965.0) * 1e6)
        roofline.update({
            "achieved": achieved, "frac": achieved / peak_tflops,
            "flop_per_unit": flop_per_unit, "unit_of_work": "(sample, bin, detector)",
            "flop_per_launch": flop_per_unit * B * N,
            "fma_share_of_fp64_instructions": ops["dfma"] / inst_per_unit,
            "fp64_pipe_frac": inst_per_unit * B * N / (kern_ms * 1e-3) / (peak_tflops * 1e12 / 2.0),
            "operand_bandwidth_bound_ms": t_operand * 1e3,
            "frac_of_operand_bandwidth_bound": t_operand * 1e3 / kern_ms,
        })
    roofline.update({
        "peak_source": "148 SM x 64 FP64 lanes x 2 flop x clocks.max.sm (DESIGN.md; no FP64 entry in "
                       "MEASURED_PEAKS.json); DFMA micro-benchmarks of this library alongside",
        "peak_dfma_measured": dfma_tflops, "peak_dfma_3reg_measured": dfma3_tflops,
        "frac_of_dfma_measured": (roofline["achieved"] / dfma_tflops) if roofline["achieved"] else None,
        "kernel_ms": kern_ms, "kernel_launches": main_launches, "kernel_share_of_step": main_ms / elapsed_ms,
        "flop_basis": "FP64 operations of the reduced algorithm = executed 2*DFMA+DMUL+DADD per unit, averaged over "
                      f"the detectors, ncu ({OPS_SOURCE})",
        "hbm_gbs_achieved": (roofline["traffic"] / (kern_ms * 1e-3) / 1e9) if roofline["traffic"] else None,
        "survey_estimate_flop_per_bin_eval": SURVEY_FLOP_PER_BIN_EVAL.get(args.config),
    })

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        rate, sec, cores, desc = oracle_timed(args.config, args.ref_samples, 1,
                                              tab_nodes=args.tab_nodes if tab_mode else 0)
        cpu_baseline = {"value": rate, "unit": unit, "cores": cores, "kind": "oracle", "sample": desc,
                        "value_one_thread": oracle_timed.one_thread}

    line = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64+f32 (mixed: FP64 phases, FP32 geometry)" if mixed_mode else "f64", "data": "synthetic",
        "bin_evals_per_sec": value * N,
        "config": workload_config(wl, args, l2="256 MiB buffer rewritten before every step, inside the timed region"),
        "clocks": clocks,
        "e2e": {"value": e2e["full"], "unit": unit, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                "api": ("pespace_session_set_data + pespace_session_loglike_tab per step: theta, the step's waveform "
                        "tables, data set and PSD copied from pinned host memory, lnL read back" if tab_mode else
                        "pespace_session_set_data + pespace_session_" + ("fisher" if fisher_mode else "loglike") +
                        " per step: theta, data set and PSD copied from pinned host memory, result read back"),
                "precision_note": "pespace_session_loglike_mixed" if mixed_mode else None,
                "value_resident_data": e2e["resident"],
                "resident_data_note": "same call with the data set copied once (sampler use): theta in, result out"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "result_check": {"min": float(last.min()), "max": float(last.max())},
        "response": response_info,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4, 5])
    ap.add_argument("--precision", choices=["f64", "mixed"], default="f64",
                    help="mixed: pespace_loglike_mixed (FP64 phases, FP32 geometry; SURVEY 8(f) N2) in the device-timed leg")
    ap.add_argument("--response", action="store_true", help="also time pespace_response on a slice of the batch")
    ap.add_argument("--response-batch", type=int, default=256)
    ap.add_argument("--grad-only", action="store_true",
                    help="config 5: d lnL / d theta only (pespace_fisher with d_out_F = NULL)")
    ap.add_argument("--waveform", choices=["analytic", "tab"], default="analytic",
                    help="tab: pespace_loglike_tab on synthetic tabulated mode waveforms (SURVEY 8(f) N1)")
    ap.add_argument("--tab-nodes", type=int, default=4096, help="nodes K of the waveform tables")
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
