#!/usr/bin/env python
"""bench.py -- throughput of the batched likelihood hot path on B200 (one JSON line on stdout).

  python bench.py --gpus N --steps K --warmup W [--config 2|3|4|5] [--path ...] [--impl reference]

A "step" is one pass of the whole hot path (per-bin table -> per-sample constants ->
fused per-bin kernel -> fixed-order combine) over one batch of B synthetic samples: one pespace_loglike call.  The
workload at N=1 is BASELINE.json configs[1] ("config 2": B=4096 x N=262144, one LISA-like detector, (2,2) mode), the
one the metric is quoted on.  With N>1 GPUs (torchrun) every rank evaluates its own batch of B samples on replicated
data -- no data-path collective -- so scaling is "weak" and `value` is the whole-job rate; `--scaling strong` splits
ONE global batch over the ranks (dist.ShardedLikelihood: all-gather of lnL inside the timed region).

value          device-timed evaluations/s, inputs resident in HBM (CUDA events, max over ranks)
e2e            the same metric through the C ABI with HOST buffers (pespace_session_*): H2D of theta + data + PSD and
               D2H of the result inside the timed region
roofline       the dominant kernel against the FP64 ALU peak; operation counts from profiles/r02_ops.json (ncu),
               marked stale when the kernel sources have changed since they were counted
other_configs  (default run only) short device-timed runs of configs 3, 4, 5 (Fisher), the adjoint gradient and
               pespace_response, so that every BASELINE.json config and every north-star call is in the driver's line;
               single_theta_latency: one sample x N bins per call, plain, with pespace_prepare, and the prepared call
               replayed from a CUDA graph (wall clock, us)
cpu_baseline / --impl reference   the oracle, as it stands, on the box's host cores

--path selects the entry point that is timed: loglike (default; config 5: fisher), mixed, tab, orb, grad (adjoint
lnL + gradient), fisher-grad (forward-mode gradient, pespace_fisher with d_out_F = NULL).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2602_12011_b200 import build as pbuild        # noqa: E402
from paper_2602_12011_b200 import dist as pdist          # noqa: E402
from paper_2602_12011_b200 import workloads as W         # noqa: E402

# ---- roofline constants
# FP64 ALU peak: 148 SMs x 64 FP64 lanes x 2 flop x clocks.max.sm (1965 MHz) = 37.22 TFLOP/s; MEASURED_PEAKS.json has no
# FP64 entry, so the library's own DFMA micro-benchmark (pespace_fp64_peak) is run in the same process and reported
# beside it.  The operation counts per unit of work come from profiles/r02_ops.json (written from ncu CSVs by
# paper_2602_12011_b200/ops_from_ncu.py and stamped with the content hash of the kernel sources).
SM_COUNT, FP64_LANES_PER_SM = 148, 64
OPS_FILE = os.path.join(ROOT, "profiles", "r02_ops.json")
# SURVEY.md 8(d) survey-time estimate (library-cost transcendentals); kept for reference only
SURVEY_FLOP_PER_BIN_EVAL = {2: 970.0, 3: 4500.0, 4: 11200.0, 5: 100000.0}
UNITS = {"loglike": ("lnL_evals_per_sec", "lnL/s"), "mixed": ("lnL_evals_per_sec", "lnL/s"),
         "tab": ("lnL_evals_per_sec", "lnL/s"), "orb": ("lnL_evals_per_sec", "lnL/s"),
         "fisher": ("fisher_evals_per_sec", "F/s"), "fisher-grad": ("grad_evals_per_sec", "grad/s"),
         "grad": ("lnL_and_grad_evals_per_sec", "(lnL+grad)/s")}
KERNEL_OF = {"loglike": "loglike", "mixed": "loglike_mixed", "tab": "loglike_tab", "orb": "loglike_orb",
             "fisher": "fisher", "fisher-grad": "fisher", "grad": "loglike_grad"}


def load_ops():
    try:
        doc = json.load(open(OPS_FILE))
    except (OSError, ValueError):
        return {"kernels": {}, "csrc_hash": None}
    return doc


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


def oracle_timed(config: int, path: str, n_samples, steps: int, target_s: float = 12.0, tab_nodes: int = 0):
    """Time the oracle, as it stands, on a bounded sample of the workload: `n_samples` samples (None: sized from a
    one-sample-per-core calibration pass for ~target_s of wall time) x all N bins per step; for the derivative paths
    x the first FISHER_REF_BINS bins, the rate scaled by FISHER_REF_BINS / N (the cost per bin is uniform).
    -> (rate in full-N evaluations/s, seconds per step, cores, description of the sample)."""
    import oracle
    deriv = path in ("fisher", "fisher-grad", "grad")
    full = W.config(config)
    wl = W.config(config, N=FISHER_REF_BINS) if deriv else full
    scale = wl.grid.N / full.grid.N
    psd = wl.psd()
    cores = oracle.get_threads()
    if path == "tab":
        f_all = wl.grid.freqs()
        fnodes = W.log_nodes(f_all[0], f_all[-1], tab_nodes)
        tab = lambda p: W.chirp_table(p, wl.model.mode_mask, fnodes)
        data = wl.data(lambda p, fr, m: oracle.response_tab(p, tab(p), fr, m))
        call = lambda p: oracle.loglike_tab(p, tab(p), data, psd, wl.grid, wl.model)
    elif path == "orb":
        otab = orbit_table_for(wl)
        data = wl.data(lambda p, fr, m: oracle.response_orb(p, otab, fr, m))
        call = lambda p: oracle.loglike_orb(p, otab, data, psd, wl.grid, wl.model)
    else:
        data = wl.data(lambda p, fr, m: oracle.response(p, fr, m))
        if deriv:
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
    bins = f"all {wl.grid.N} bins" if not deriv else f"the first {wl.grid.N} of {full.grid.N} bins (rate scaled by {scale:.5f})"
    what = " (the oracle's forward-mode F + gradient pass)" if deriv else ""
    desc = (f"{n_samples} of {full.B} samples (evenly spaced) x {bins} per pass, {steps} pass(es), "
            f"{dt / steps:.1f} s per pass, OpenMP over samples{what}")
    return n_samples * steps / dt * scale, dt / steps, cores, desc


def orbit_table_for(wl, dt: float = 1800.0):
    """seeded toy ephemeris covering every t_lm of the workload with margin (input recipe only: workloads.py)"""
    T = 1.0 / wl.grid.df                 # t_44(1e-4 Hz) = t_22(5e-5 Hz) lies 12.5 T before t_c for the config masses
    t_lo, t_hi = -16.0 * T, 2.2 * T
    return W.synthetic_orbit_table(wl.model.detectors, t_lo, dt, int((t_hi - t_lo) / dt) + 2, seed=17)


def default_path(args) -> str:
    if args.path:
        return args.path
    return "fisher" if args.config == 5 else "loglike"


def workload_config(wl, args, path, l2):
    extra = {"tab": f" + tabulated mode waveforms (K={args.tab_nodes} log-spaced nodes)", "orb": " + tabulated orbits",
             "grad": " (lnL + adjoint gradient)", "fisher-grad": " (forward-mode gradient only)",
             "mixed": " (mixed precision)"}.get(path, "")
    return {"workload": f"config{args.config}{extra}: B={wl.B} x N={wl.grid.N}, {len(wl.model.detectors)} detector(s) "
                        f"[{', '.join(d.name for d in wl.model.detectors)}], mode_mask={wl.model.mode_mask}, "
                        f"TDI {wl.model.detectors[0].tdi_gen / 10:.1f}, f0={wl.grid.f0} Hz, df=1/(30 d)",
            "path": path, "B_per_gpu": wl.B, "N_bins": wl.grid.N, "n_det": len(wl.model.detectors),
            "mode_mask": wl.model.mode_mask,
            "parallelism": (f"one global batch split over {args.gpus} rank(s), all-gather of lnL" if args.scaling == "strong"
                            else f"sample-sharded x{args.gpus} (no data-path collective)"),
            "l2": l2}


def run_reference(args):
    rank, _, world = pdist.env_world()
    if rank != 0:
        return
    if world > 1:
        # torchrun sets OMP_NUM_THREADS=1 for every rank when it starts several; the other ranks have exited, so rank 0
        # gives the oracle the host cores it has under plain `python bench.py --impl reference`
        import oracle
        oracle.set_threads(len(os.sched_getaffinity(0)))
    path = default_path(args)
    wl = W.config(args.config)
    metric, unit = UNITS[path]
    rate, sec_per_step, cores, sample = oracle_timed(args.config, path, args.ref_samples, args.steps,
                                                     target_s=max(2.0, 60.0 / max(1, args.steps)),
                                                     tab_nodes=args.tab_nodes)
    line = {
        "impl": "reference", "metric": metric, "value": rate, "unit": unit, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec_per_step * 1e3,
        "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "bin_evals_per_sec": rate * wl.grid.N,
        "config": workload_config(wl, args, path, l2="n/a (CPU)"),
        "cpu_baseline": {"value": rate, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample,
                         "value_one_thread": oracle_timed.one_thread},
        "e2e": {"value": rate, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ device side
class Bench:
    """One (config, path) workload resident on the device: builds the inputs, exposes step(i)."""

    def __init__(self, P, torch, device, rank, config, path, args, B=None, world=1):
        self.P, self.torch, self.device, self.path = P, torch, device, path
        n_batches = 2 if path == "tab" else 4
        strong = args.scaling == "strong" and world > 1
        seed_rank = 0 if strong else rank                 # strong scaling: every rank holds the SAME global batch
        self.wls = [W.config(config, B=B, param_seed=pdist.rank_seed(1000 + i, seed_rank)) for i in range(n_batches)]
        wl = self.wl = self.wls[0]
        self.B, self.N, self.n_batches = wl.B, wl.grid.N, n_batches
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
        self.freqs_d = dev(wl.grid.freqs())
        self.tabs_h = self.tabs_d = self.orbit = None
        if path == "tab":
            f_all = wl.grid.freqs()
            fnodes = W.log_nodes(f_all[0], f_all[-1], args.tab_nodes)
            self.tabs_h = [tuple(torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
                                 for x in W.chirp_table(w.params, wl.model.mode_mask, fnodes)) for w in self.wls]
            self.tabs_d = [P.WaveTable(*(x.to(device) for x in t)) for t in self.tabs_h]
            inj_tab = P.WaveTable(*(dev(x) for x in W.chirp_table(wl.theta_inj[None], wl.model.mode_mask, fnodes)))
            resp = lambda p, fr, m: P.response_tab(dev(p), inj_tab, self.freqs_d, m).cpu().numpy()
        elif path == "orb":
            ot = orbit_table_for(wl)
            self.orbit = P.OrbitTable(ot[0], ot[1], dev(ot[2]), dev(ot[3]))
            resp = lambda p, fr, m: P.response_orb(dev(p), self.orbit, self.freqs_d, m).cpu().numpy()
        else:
            resp = lambda p, fr, m: P.response(dev(p), self.freqs_d, m).cpu().numpy()
        # the injection comes from this library's own response call; host copies live in pinned memory
        self.data_h = torch.from_numpy(np.ascontiguousarray(wl.data(resp))).pin_memory()
        self.psd_h = torch.from_numpy(np.ascontiguousarray(wl.psd())).pin_memory()
        self.params_h = [torch.from_numpy(np.ascontiguousarray(w.params)).pin_memory() for w in self.wls]
        self.params_d = [p.to(device) for p in self.params_h]
        data_d, psd_d = self.data_h.to(device), self.psd_h.to(device)
        B = self.B
        f64 = dict(dtype=torch.float64, device=device)
        self.out_d = torch.empty(B, **f64)
        self.F_d = self.g_d = None
        if path in ("fisher", "fisher-grad"):
            self.obj = P.Fisher(data_d, psd_d, wl.grid, wl.model, B)
            self.F_d, self.g_d = torch.empty((B, P.NPAR, P.NPAR), **f64), torch.empty((B, P.NPAR), **f64)
        elif path == "grad":
            self.obj = P.LikelihoodGrad(data_d, psd_d, wl.grid, wl.model, B)
            self.g_d = torch.empty((B, P.NPAR), **f64)
        elif path == "tab":
            self.obj = P.LikelihoodTab(data_d, psd_d, wl.grid, wl.model, B)
        elif path == "orb":
            self.obj = P.LikelihoodOrb(data_d, psd_d, wl.grid, wl.model, B)
        else:
            self.obj = P.Likelihood(data_d, psd_d, wl.grid, wl.model, B)
        self.sharded = None
        if strong and path in ("loglike", "mixed"):
            self.sharded = pdist.ShardedLikelihood(lambda p: self.obj(p, mixed=(path == "mixed")))

    def step(self, i):
        p = self.params_d[i % self.n_batches]
        if self.path == "fisher":
            self.obj(p, self.F_d, self.g_d)
        elif self.path == "fisher-grad":
            self.obj(p, None, self.g_d, grad_only=True)
        elif self.path == "grad":
            self.obj(p, self.out_d, self.g_d)
        elif self.path == "tab":
            self.obj(p, self.tabs_d[i % self.n_batches], self.out_d)
        elif self.path == "orb":
            self.obj(p, self.orbit, self.out_d)
        elif self.sharded is not None:
            self.out_d = self.sharded(p)
        else:
            self.obj(p, self.out_d, mixed=(self.path == "mixed"))

    def result(self):
        t = {"fisher": self.F_d, "fisher-grad": self.g_d, "grad": self.g_d}.get(self.path, self.out_d)
        return t.cpu().numpy()


def timed_run(b: Bench, steps: int, warmup: int, flush, device):
    """-> dict(elapsed_ms, launches, kernel_ms_total, kernel_launches); exactly `steps` steps, device events, barrier +
    synchronize on both sides; the L2 flush (a 256 MiB buffer rewritten) sits inside the timed region"""
    P, torch = b.P, b.torch
    for i in range(warmup):
        flush.zero_()
        b.step(i)
    torch.cuda.synchronize()
    P.profile_enable(True)
    P.profile_read()
    launches0 = P.launch_count()
    pdist.barrier(device)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(steps):
        flush.zero_()
        b.step(i)
    e1.record()
    torch.cuda.synchronize()
    pdist.barrier(device)
    main_ms, main_launches = P.profile_read()
    P.profile_enable(False)
    return {"elapsed_ms": e0.elapsed_time(e1), "launches": P.launch_count() - launches0, "kernel_ms_total": main_ms,
            "kernel_launches": main_launches}


def class_mask(mode_mask: int) -> int:
    return (2 if mode_mask & 9 else 0) | (1 if mode_mask & 2 else 0) | (4 if mode_mask & 4 else 0) | \
           (8 if mode_mask & 16 else 0)


def roofline_of(path, wl, B, N, kern_ms, ops_doc, peak_tflops, sm_max_mhz, stale):
    """roofline object of the dominant kernel of `path` from the ncu operation table (None entries when the table has
    no row for one of the kernels involved)"""
    kernel = KERNEL_OF[path]
    cm = class_mask(wl.model.mode_mask)
    n_det = len(wl.model.detectors)
    rows = []
    if kernel == "loglike" and n_det > 1:
        kernel = "loglike_fused"                       # one launch walks all detectors: n_det x B x N units per launch
        rows = [ops_doc["kernels"].get(f"loglike_fused|0|{cm}")]
        B = B * n_det
    else:
        n_modes = bin(wl.model.mode_mask).count("1")
        for d in wl.model.detectors:
            # second key: the compile-time variant of the kernel (class mask; tab: mode count; 0 = run-time loop)
            key_mask = {"loglike_tab": n_modes if n_modes in (1, 5) else 0, "loglike_mixed": cm if cm in (2, 15) else 0,
                        "loglike_orb": cm if cm in (2, 15) else 0}.get(kernel, cm)
            key_kind = 0 if kernel == "loglike_orb" else d.kind
            rows.append(ops_doc["kernels"].get(f"{kernel}|{key_kind}|{key_mask}"))
    out = {"bound": "alu", "kernel": f"{kernel}_kernel", "achieved": None, "peak": peak_tflops, "unit": "TFLOP/s",
           "frac": None, "traffic": None, "kernel_ms": kern_ms, "stale": stale,
           "ops_source": os.path.relpath(OPS_FILE, ROOT), "ops_csrc_hash": ops_doc.get("csrc_hash")}
    if path == "fisher-grad" or not all(rows):
        return out                                         # no ncu counts for this variant
    n = len(rows)
    ops = {k: sum(r[k] for r in rows) / n for k in ("dfma", "dmul", "dadd", "dram_bytes_per_launch")}
    flop_per_unit = 2.0 * ops["dfma"] + ops["dmul"] + ops["dadd"]
    inst_per_unit = ops["dfma"] + ops["dmul"] + ops["dadd"]
    achieved = flop_per_unit * B * N / (kern_ms * 1e-3) / 1e12
    # issue cost on the FP64 pipe (profiles/r01_fp64_operand_bandwidth.md): one 64-bit register operand per cycle and
    # SM sub-partition, at least 2 cycles per instruction -> a DFMA with three distinct registers takes 3 cycles
    cyc = 3.0 * ops["dfma"] + 2.0 * (ops["dmul"] + ops["dadd"])
    t_operand = cyc * (B * N / 32.0) / (SM_COUNT * 4) / (sm_max_mhz * 1e6)
    out.update({
        "achieved": achieved, "frac": achieved / peak_tflops, "traffic": ops["dram_bytes_per_launch"],
        "flop_per_unit": flop_per_unit, "unit_of_work": "(sample, bin, detector)",
        "flop_per_launch": flop_per_unit * B * N,
        "fma_share_of_fp64_instructions": ops["dfma"] / inst_per_unit,
        "fp64_pipe_frac": inst_per_unit * B * N / (kern_ms * 1e-3) / (peak_tflops * 1e12 / 2.0),
        "operand_bandwidth_bound_ms": t_operand * 1e3,
        "frac_of_operand_bandwidth_bound": t_operand * 1e3 / kern_ms,
        "hbm_gbs_achieved": ops["dram_bytes_per_launch"] / (kern_ms * 1e-3) / 1e9,
    })
    return out


def run_ours(args):
    import torch
    from paper_2602_12011_b200 import binding as P      # fails loudly if libpespace.so is missing

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle timing)")
    rank, local_rank, world = pdist.init("nccl")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    path = default_path(args)
    if path in ("fisher", "fisher-grad") and args.config != 5:
        pass                                            # any config may run the derivative paths
    metric, unit = UNITS[path]
    ops_doc = load_ops()
    stale = ops_doc.get("csrc_hash") != pbuild.csrc_hash()

    main = Bench(P, torch, device, rank, args.config, path, args, world=world)
    wl, B, N = main.wl, main.B, main.N
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)   # > 126 MB L2

    sampler = ClockSampler(local_rank)
    sampler.start()
    t = timed_run(main, args.steps, args.warmup, flush, device)
    clocks = sampler.stop()
    last = main.result()
    if not np.all(np.isfinite(last)):
        raise SystemExit("bench.py: non-finite result in the timed region")
    strong = args.scaling == "strong" and world > 1
    units_here = (B / world if strong else B) * args.steps
    max_ms, total_units = pdist.aggregate(t["elapsed_ms"], units_here, device)
    value = total_units / (max_ms * 1e-3)

    # ---- e2e: HOST buffers through the C ABI (pespace_session_*): every step copies that step's inputs (theta, data
    # set, PSD) from pinned host memory to the device and reads the result back, all inside the timed region.
    # value_resident_data: the sampler-facing use, data set copied once, theta per step.
    e2e_steps = max(1, min(args.steps, 10))
    e2e, h2d, d2h, e2e_api = {"full": None, "resident": None}, 0, 0, None
    nbytes = lambda x: x.numel() * x.element_size()
    if path != "orb":
        ses = P.Session(wl.grid, wl.model, B, want_fisher=path in ("fisher", "fisher-grad"))
        grad_h = torch.empty((B, P.NPAR), dtype=torch.float64).pin_memory()
        res_h = torch.empty((B, P.NPAR, P.NPAR) if path == "fisher" else (B,), dtype=torch.float64).pin_memory()
        nb = main.n_batches

        def e2e_step(i, copy_data):
            if copy_data:
                ses.set_data(main.data_h, main.psd_h)
            p = main.params_h[i % nb]
            if path == "tab":
                ses.loglike_tab(p, main.tabs_h[i % nb], res_h)
            elif path == "fisher":
                ses.fisher(p, True, res_h, grad_h)
            elif path == "fisher-grad":
                ses.fisher(p, True, None, grad_h, grad_only=True)
            elif path == "grad":
                ses.loglike_grad(p, res_h, grad_h)
            else:
                ses.loglike(p, res_h, mixed=(path == "mixed"))

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
        h2d = nbytes(main.params_h[0]) + nbytes(main.data_h) + nbytes(main.psd_h) + \
            (sum(nbytes(x) for x in main.tabs_h[0]) if path == "tab" else 0)
        d2h = (nbytes(res_h) if path != "fisher-grad" else 0) + (nbytes(grad_h) if path in ("fisher", "fisher-grad", "grad") else 0)
        call = {"tab": "loglike_tab", "fisher": "fisher", "fisher-grad": "fisher", "grad": "loglike_grad",
                "mixed": "loglike_mixed"}.get(path, "loglike")
        e2e_api = (f"pespace_session_set_data + pespace_session_{call} per step: theta, data set and PSD"
                   f"{' and the waveform tables' if path == 'tab' else ''} copied from pinned host memory, result read back")

    # ---- the other configs and calls, device-timed only (3 steps each after 3 warm-ups)
    others = None
    if args.others and world == 1:
        others = []
        peak0 = SM_COUNT * FP64_LANES_PER_SM * 2 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
        for cfg, pth in ((3, "loglike"), (4, "loglike"), (5, "fisher"), (5, "grad"), (2, "grad")):
            if cfg == args.config and pth == path:
                continue
            oargs = argparse.Namespace(**vars(args))
            oargs.config = cfg
            ob = Bench(P, torch, device, rank, cfg, pth, oargs)
            ot = timed_run(ob, 3, 3, flush, device)
            if not np.all(np.isfinite(ob.result())):
                raise SystemExit(f"bench.py: non-finite result in config {cfg} / {pth}")
            km = ot["kernel_ms_total"] / max(1, ot["kernel_launches"])
            rf = roofline_of(pth, ob.wl, ob.B, ob.N, km, ops_doc, peak0, clocks.get("sm_max_mhz") or 1965.0, stale)
            m_, u_ = UNITS[pth]
            others.append({"config": cfg, "path": pth, "metric": m_, "unit": u_,
                           "value": ob.B * 3 / (ot["elapsed_ms"] * 1e-3), "ms_per_step": ot["elapsed_ms"] / 3,
                           "B": ob.B, "N": ob.N, "n_det": len(ob.wl.model.detectors), "mode_mask": ob.wl.model.mode_mask,
                           "kernel_ms": km, "kernel_launches_per_step": ot["kernel_launches"] / 3,
                           "gpu_launches": int(ot["launches"]), "frac": rf["frac"], "achieved_tflops": rf["achieved"],
                           "flop_per_unit": rf.get("flop_per_unit")})
            del ob
            torch.cuda.empty_cache()

    # ---- pespace_response on a slice of the batch (48 B written per (sample, bin, detector))
    response_info = None
    if (args.response or args.others) and world == 1:
        response_info = []
        for cfg in (2, 3, 4):                         # config 4: three detectors in ONE launch (response_fused_kernel)
            wr = W.config(cfg, B=args.response_batch)
            pr = torch.from_numpy(np.ascontiguousarray(wr.params)).to(device)
            out_r = torch.empty((wr.B, len(wr.model.detectors), 3, N, 2), dtype=torch.float64, device=device)
            for _ in range(2):
                P.response(pr, main.freqs_d, wr.model, out_r)
            torch.cuda.synchronize()
            r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            r0.record()
            for _ in range(5):
                P.response(pr, main.freqs_d, wr.model, out_r)
            r1.record()
            torch.cuda.synchronize()
            r_ms = r0.elapsed_time(r1) / 5
            response_info.append({"call": "pespace_response", "mode_mask": wr.model.mode_mask, "batch": wr.B, "N": N,
                                  "n_det": len(wr.model.detectors),
                                  "ms_per_call": r_ms, "bin_evals_per_sec": wr.B * N / (r_ms * 1e-3),
                                  "bytes_written_per_call": out_r.numel() * 8,
                                  "write_gbs": out_r.numel() * 8 / (r_ms * 1e-3) / 1e9})
            del out_r

    # ---- single-theta latency (one sample x N bins; a sampler that walks one chain): the plain call rebuilds the
    # per-bin table on every call, the prepared call (pespace_prepare once) does not
    latency_info = None
    if args.others and world == 1:
        latency_info = []
        # (config, N): the full one-month grids, and the paper's own protocol -- one theta per call against the number
        # of frequency samples (Fig. 4; its PE runs use ~32.7 k bins) -- for one and five modes
        for cfg, nq in ((2, None), (4, None), (2, 4096), (2, 32768), (3, 4096), (3, 32768), (3, None)):
            wq = W.config(cfg, B=1, N=nq)
            psd_q = wq.psd()
            data_q = W.coloured_noise(psd_q, wq.grid.df, np.random.default_rng(5))
            lq = P.Likelihood(torch.from_numpy(np.ascontiguousarray(data_q)).to(device),
                              torch.from_numpy(psd_q).to(device), wq.grid, wq.model, 1)
            pq = torch.from_numpy(np.ascontiguousarray(wq.params)).to(device)
            oq = torch.empty(1, dtype=torch.float64, device=device)
            row = {"config": cfg, "B": 1, "N": wq.grid.N, "n_det": len(wq.model.detectors),
                   "mode_mask": wq.model.mode_mask}
            for key in ("pespace_loglike_us", "pespace_loglike_prepared_us"):
                if key.endswith("prepared_us"):
                    lq.prepare()
                for _ in range(20):
                    lq(pq, oq)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for _ in range(200):
                    lq(pq, oq)
                torch.cuda.synchronize()
                row[key] = (time.perf_counter() - t0) / 200 * 1e6
            # the prepared call replayed from a CUDA graph (three kernel nodes; no host-side launch work)
            try:
                gq = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gq):
                    lq(pq, oq)
                for _ in range(20):
                    gq.replay()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for _ in range(200):
                    gq.replay()
                torch.cuda.synchronize()
                row["pespace_loglike_prepared_graph_replay_us"] = (time.perf_counter() - t0) / 200 * 1e6
                del gq
            except RuntimeError as exc:                      # reported, never fatal for the bench line
                row["pespace_loglike_prepared_graph_replay_us"] = None
                row["graph_error"] = str(exc)[:200]
            # lnL + reverse-mode gradient for one theta (a gradient-based sampler's step), prepared call
            try:
                gq_ = P.LikelihoodGrad(lq.data, lq.psd, wq.grid, wq.model, 1).prepare()
                lo_, go_ = torch.empty(1, dtype=torch.float64, device=device), torch.empty((1, 11), dtype=torch.float64, device=device)
                for _ in range(20):
                    gq_(pq, lo_, go_)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                for _ in range(200):
                    gq_(pq, lo_, go_)
                torch.cuda.synchronize()
                row["pespace_loglike_grad_prepared_us"] = (time.perf_counter() - t0) / 200 * 1e6
                del gq_
            except RuntimeError as exc:
                row["pespace_loglike_grad_prepared_us"] = None
                row["grad_error"] = str(exc)[:200]
            latency_info.append(row)
            del lq

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (per launch, timed live with CUDA events in the library)
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak_tflops = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    dfma_tflops, _ = P.fp64_peak(8192, mode=0)
    dfma3_tflops, _ = P.fp64_peak(8192, mode=1)
    kern_ms = t["kernel_ms_total"] / max(1, t["kernel_launches"])   # one launch = one detector (fused likelihood: all)
    B_launch = B / world if strong else B
    roofline = roofline_of(path, wl, B_launch, N, kern_ms, ops_doc, peak_tflops, sm_max, stale)
    roofline.update({
        "peak_source": "148 SM x 64 FP64 lanes x 2 flop x clocks.max.sm (DESIGN.md; no FP64 entry in "
                       "MEASURED_PEAKS.json); DFMA micro-benchmarks of this library alongside",
        "peak_dfma_measured": dfma_tflops, "peak_dfma_3reg_measured": dfma3_tflops,
        "frac_of_dfma_measured": (roofline["achieved"] / dfma_tflops) if roofline["achieved"] else None,
        "kernel_launches": t["kernel_launches"], "kernel_share_of_step": t["kernel_ms_total"] / t["elapsed_ms"],
        "csrc_hash": pbuild.csrc_hash(),
        "flop_basis": "FP64 operations of the reduced algorithm = executed 2*DFMA+DMUL+DADD per unit, averaged over "
                      "the detectors, from the ncu captures listed in profiles/r02_ncu.md",
        "survey_estimate_flop_per_bin_eval": SURVEY_FLOP_PER_BIN_EVAL.get(args.config),
    })

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        rate, sec, cores, desc = oracle_timed(args.config, path, args.ref_samples, 1, tab_nodes=args.tab_nodes)
        cpu_baseline = {"value": rate, "unit": unit, "cores": cores, "kind": "oracle", "sample": desc,
                        "value_one_thread": oracle_timed.one_thread}

    line = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak",
        "vs_baseline": None,
        "dtype": "f64+f32 (mixed: FP64 phases, FP32 geometry)" if path == "mixed" else "f64", "data": "synthetic",
        "bin_evals_per_sec": value * N,
        "config": workload_config(wl, args, path, l2="256 MiB buffer rewritten before every step, inside the timed region"),
        "clocks": clocks,
        "e2e": {"value": e2e["full"], "unit": unit, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps, "api": e2e_api, "value_resident_data": e2e["resident"],
                "resident_data_note": "same call with the data set copied once (sampler use): theta in, result out"},
        "gpu_launches": int(t["launches"]),
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "result_check": {"min": float(last.min()), "max": float(last.max())},
        "other_configs": others,
        "response": response_info,
        "single_theta_latency": latency_info,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3, 4, 5])
    ap.add_argument("--path", choices=sorted(UNITS), default=None,
                    help="entry point to time (default: loglike; config 5: fisher)")
    ap.add_argument("--precision", choices=["f64", "mixed"], default="f64", help="mixed = --path mixed")
    ap.add_argument("--waveform", choices=["analytic", "tab"], default="analytic", help="tab = --path tab")
    ap.add_argument("--grad-only", action="store_true",
                    help="lnL + d lnL / d theta by reverse mode, pespace_loglike_grad (= --path grad); the forward-mode "
                         "gradient of round 1 (pespace_fisher with d_out_F = NULL) is --path fisher-grad")
    ap.add_argument("--scaling", choices=["weak", "strong"], default="weak",
                    help="N > 1: weak = one batch of B per rank; strong = one global batch of B split over the ranks")
    ap.add_argument("--response", action="store_true", help="also time pespace_response on a slice of the batch")
    ap.add_argument("--response-batch", type=int, default=256)
    ap.add_argument("--tab-nodes", type=int, default=4096, help="nodes K of the waveform tables")
    ap.add_argument("--ref-samples", type=int, default=None,
                    help="samples per oracle pass (default: sized for ~15 s of CPU work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", dest="others", action="store_false",
                    help="skip the short runs of the other configs / calls (other_configs, response)")
    args = ap.parse_args()
    if args.path is None:
        if args.precision == "mixed":
            args.path = "mixed"
        elif args.waveform == "tab":
            args.path = "tab"
        elif args.grad_only:
            args.path = "grad"
    # the extra short runs belong to the default invocation (the driver's command line) only
    if args.config != 2 or args.path not in (None, "loglike") or args.scaling != "weak":
        args.others = False
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
