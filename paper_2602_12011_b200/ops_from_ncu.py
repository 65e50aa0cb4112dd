"""Turn ncu metric CSVs into the operation table bench.py reads (profiles/rNN_ops.json).

  python -m paper_2602_12011_b200.ops_from_ncu --out profiles/r02_ops.json  CSV:B:N [CSV:B:N ...]

Each CSV is the `--csv --log-file` output of an `ncu --metrics ...` run of bench.py (the exact command is kept in the
`.md` beside the CSV under profiles/); B and N are the samples and bins of the profiled launches, so that one launch
processes B x N units of work (one unit = one (sample, bin, detector); for the fused multi-detector kernel, which walks
the detectors inside one launch, pass B x n_det as B).  For every profiled kernel the script stores,
per unit, the thread-level FP64 operation counts (DFMA, DMUL, DADD), the FP64-pipe warp instructions, all warp
instructions, and per launch the DRAM bytes and the duration -- keyed by "<kernel>|<kind>|<class mask>" -- together
with `csrc_hash`, the content hash of the sources they were counted on (build.csrc_hash()).  bench.py recomputes that
hash at run time and marks its roofline `stale` when the kernels have changed since.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import re
import sys

from . import build as _build

METRICS = {
    "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum": "dfma",
    "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum": "dmul",
    "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum": "dadd",
    "sm__inst_executed_pipe_fp64.sum": "fp64_warp_inst",
    "smsp__inst_executed.sum": "warp_inst",
    "dram__bytes_read.sum": "dram_read",
    "dram__bytes_write.sum": "dram_write",
    "gpu__time_duration.sum": "time_ns",
    "launch__registers_per_thread": "registers",
    "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active": "fp64_pipe_pct",
}
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "nsecond": 1.0, "usecond": 1e3, "msecond": 1e6,
              "second": 1e9}
KERNELS = ("loglike_fused_kernel", "loglike_grad_kernel", "loglike_tab_kernel", "loglike_mixed_kernel",
           "loglike_orb_kernel", "loglike_kernel", "fisher_kernel", "response_fused_kernel", "response_kernel")


def kernel_key(name: str):
    """'void pespace::loglike_kernel<0, 2>(...)' -> ('loglike', 0, 2); kernels without a class mask -> (.., kind, 0)"""
    for k in KERNELS:
        if k in name:
            m = re.search(re.escape(k) + r"<\s*(\d+)u?\s*(?:,\s*(\d+)u?)?\s*>", name)
            kind = int(m.group(1)) if m else 0
            mask = int(m.group(2)) if m and m.group(2) else 0
            if k in ("loglike_fused_kernel", "loglike_orb_kernel", "response_fused_kernel"):   # one argument: the mask
                kind, mask = 0, kind
            return k[:-len("_kernel")], kind, mask
    return None


def read_csv(path: str):
    """-> {launch id: (kernel name, {metric: value})}"""
    rows = [r for r in csv.reader(open(path, newline="")) if len(r) > 10]
    hdr = rows[0]
    out = {}
    for r in rows[1:]:
        d = dict(zip(hdr, r))
        name = METRICS.get(d.get("Metric Name", ""))
        if not name:
            continue
        try:
            v = float(d["Metric Value"].replace(",", ""))
        except ValueError:
            continue
        v *= UNIT_SCALE.get(d.get("Metric Unit", ""), 1.0)
        out.setdefault(d["ID"], (d["Kernel Name"], {}))[1][name] = v
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    ap.add_argument("captures", nargs="+", help="CSV:B:N")
    args = ap.parse_args(argv)
    table = {}
    for cap in args.captures:
        path, B, N = cap.rsplit(":", 2)
        units = float(B) * float(N)
        for _, (kname, m) in sorted(read_csv(path).items()):
            key = kernel_key(kname)
            if key is None or "dfma" not in m:
                continue
            e = table.setdefault("%s|%d|%d" % key, {"launches": 0, "source": os.path.basename(path), "B": int(B), "N": int(N)})
            n = e["launches"]
            per_unit = {"dfma": m["dfma"] / units, "dmul": m["dmul"] / units, "dadd": m["dadd"] / units,
                        "fp64_warp_inst": 32.0 * m.get("fp64_warp_inst", 0.0) / units,
                        "warp_inst": 32.0 * m.get("warp_inst", 0.0) / units,
                        "dram_bytes_per_launch": m.get("dram_read", 0.0) + m.get("dram_write", 0.0),
                        "time_ms": m.get("time_ns", 0.0) / 1e6, "registers": m.get("registers", 0.0),
                        "fp64_pipe_pct": m.get("fp64_pipe_pct", 0.0)}
            for k, v in per_unit.items():                         # running mean over the launches of this kernel
                e[k] = (e.get(k, 0.0) * n + v) / (n + 1)
            e["launches"] = n + 1
    for e in table.values():
        e["flop_per_unit"] = 2.0 * e["dfma"] + e["dmul"] + e["dadd"]
    doc = {"csrc_hash": _build.csrc_hash(), "unit": "(sample, bin, detector)",
           "note": "thread-level FP64 operations per unit from ncu (smsp__sass_thread_inst_executed_op_d*_pred_on.sum / "
                   "(B N)); flop = 2 DFMA + DMUL + DADD; written by paper_2602_12011_b200/ops_from_ncu.py",
           "kernels": dict(sorted(table.items()))}
    with open(args.out, "w") as f:
        json.dump(doc, f, indent=1, sort_keys=True)
        f.write("\n")
    print(f"{args.out}: {len(table)} kernels, csrc_hash {doc['csrc_hash']}", file=sys.stderr)


if __name__ == "__main__":
    main()
