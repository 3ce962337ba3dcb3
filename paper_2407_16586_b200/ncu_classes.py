"""Per-class summary of an ncu metrics pass over one tdg_gradient call (measurement tooling of the library).

The pass (one B200, after the same command exited 0 without ncu):

    ncu --metrics <METRICS below, comma separated> --clock-control none --csv --log-file gpurun_out/ncu_classes_cfg3.csv \
        python -m paper_2407_16586_b200.profile_run 3 1

then, anywhere (no GPU needed):

    python -m paper_2407_16586_b200.ncu_classes gpurun_out/ncu_classes_cfg3.csv profiles/r02_ncu_classes_cfg3 "cfg3 ..." gpurun_out/profile_run_cfg3.json

writes <out>.md (table, per quartet class) and <out>.json (numbers bench.py reads: executed FP64 FLOPs and DRAM bytes per
class for this workload, stamped with the hash of the kernel sources they were captured on).

Executed FP64 FLOPs = 2*DFMA + DMUL + DADD thread-level predicated-on instruction counts (BASELINE.json north_star:
"achieved FP64 FLOP/s against the B200 FP64 peak" by ncu counters).  Times under ncu are serialised and cold-cache:
only their SHARES are meaningful; bench.py divides the FLOP counts by its own CUDA-event times.
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import re
import sys

METRICS = [
    "gpu__time_duration.sum",
    "sm__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "sm__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "sm__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active",
    "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
    "dram__bytes_read.sum",
    "dram__bytes_write.sum",
    "l1tex__t_bytes_pipe_lsu_mem_local_op_ld.sum",
    "l1tex__t_bytes_pipe_lsu_mem_local_op_st.sum",
    "launch__registers_per_thread",
]
HERE = os.path.dirname(os.path.abspath(__file__))
_KERNEL = re.compile(r"tdg_grad(b?)_kernel<(?:\(int\))?(\d), (?:\(int\))?(\d), (?:\(int\))?(\d), (?:\(int\))?(\d)[,>]")
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "ns": 1.0, "us": 1e3, "usecond": 1e3, "ms": 1e6, "msecond": 1e6,
         "s": 1e9, "second": 1e9, "nsecond": 1.0}


def source_hash() -> str:
    """SHA-256 over the kernel sources and the build script: identifies the build a capture belongs to."""
    h = hashlib.sha256()
    csrc = os.path.join(HERE, "csrc")
    files = sorted(f for f in os.listdir(csrc) if f.endswith((".cu", ".cuh", ".h", ".inc")))
    for f in [os.path.join(csrc, f) for f in files] + [os.path.join(HERE, "build.py")]:
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def parse(path):
    """-> list of launches: dict(kernel, cls or None, metrics{name: value in base units})."""
    launches = {}
    with open(path, newline="") as fh:
        lines = [l for l in fh if l.startswith('"')]
    for row in csv.DictReader(lines):
        i = int(row["ID"])
        L = launches.setdefault(i, dict(kernel=row["Kernel Name"], m={}))
        v = float(row["Metric Value"].replace(",", "")) if row["Metric Value"] not in ("", "n/a") else float("nan")
        L["m"][row["Metric Name"]] = v * _UNIT.get(row["Metric Unit"], 1.0)
    out = []
    for i in sorted(launches):
        L = launches[i]
        mt = _KERNEL.search(L["kernel"])
        L["cls"] = tuple(int(x) for x in mt.groups()[1:]) if mt else None
        L["kind"] = ("block/quartet" if mt.group(1) else "thread/quartet") if mt else None
        out.append(L)
    return out


def summarise(launches):
    s = "spdf"
    per = {}
    for L in launches:
        if L["cls"] is None:
            continue
        name = "(%s%s|%s%s)" % tuple(s[x] for x in L["cls"])
        m = L["m"]
        t = m.get("gpu__time_duration.sum", 0.0)
        c = per.setdefault(name, dict(kind=L["kind"], launches=0, ns=0.0, dfma=0.0, dmul=0.0, dadd=0.0, dram_read=0.0, dram_write=0.0,
                                      local_bytes=0.0, regs=0, _fp64=0.0, _warps=0.0, _issue=0.0, _l1=0.0))
        c["launches"] += 1
        c["ns"] += t
        c["dfma"] += m.get("sm__sass_thread_inst_executed_op_dfma_pred_on.sum", 0.0)
        c["dmul"] += m.get("sm__sass_thread_inst_executed_op_dmul_pred_on.sum", 0.0)
        c["dadd"] += m.get("sm__sass_thread_inst_executed_op_dadd_pred_on.sum", 0.0)
        c["dram_read"] += m.get("dram__bytes_read.sum", 0.0)
        c["dram_write"] += m.get("dram__bytes_write.sum", 0.0)
        c["local_bytes"] += m.get("l1tex__t_bytes_pipe_lsu_mem_local_op_ld.sum", 0.0) + m.get("l1tex__t_bytes_pipe_lsu_mem_local_op_st.sum", 0.0)
        c["regs"] = max(c["regs"], int(m.get("launch__registers_per_thread", 0)))
        c["_fp64"] += t * m.get("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", 0.0)
        c["_warps"] += t * m.get("sm__warps_active.avg.pct_of_peak_sustained_active", 0.0)
        c["_issue"] += t * m.get("smsp__issue_active.avg.pct_of_peak_sustained_active", 0.0)
        c["_l1"] += t * m.get("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", 0.0)
    for c in per.values():
        c["flops"] = 2.0 * c["dfma"] + c["dmul"] + c["dadd"]
        c["tflops_under_ncu"] = c["flops"] / c["ns"] * 1e-3 if c["ns"] else 0.0
        for k, src in (("fp64_pipe_pct", "_fp64"), ("warps_active_pct", "_warps"), ("issue_active_pct", "_issue"), ("l1_wavefronts_pct", "_l1")):
            c[k] = c.pop(src) / c["ns"] if c["ns"] else 0.0
    return per


def main():
    src, out = sys.argv[1], sys.argv[2]
    workload = sys.argv[3] if len(sys.argv) > 3 else ""
    launches = parse(src)
    per = summarise(launches)
    total_ns = sum(L["m"].get("gpu__time_duration.sum", 0.0) for L in launches)
    rec = dict(source_hash=source_hash(), workload=workload, csv=os.path.basename(src), launches=len(launches), total_ms_under_ncu=total_ns * 1e-6,
               classes=per)
    if len(sys.argv) > 4:   # per-class counts of the profiled call (written by profile_run.py)
        run = json.load(open(sys.argv[4]))
        rec["source_hash"] = run.get("source_hash", rec["source_hash"])   # hash of the sources the profiled process ran
        rec["quartets_by_class"] = run["quartets_by_class"]
        rec["prim_quartets_by_class"] = run["prim_quartets_by_class"]
    with open(out + ".json", "w") as fh:
        json.dump(rec, fh, indent=1, sort_keys=True)
    rows = sorted(per.items(), key=lambda kv: -kv[1]["ns"])
    with open(out + ".md", "w") as fh:
        fh.write("# ncu metrics pass, per quartet class — %s\n\n" % workload)
        fh.write("Command (B200, after the same command exited 0 without ncu):\n\n    ncu --metrics %s --clock-control none --csv --log-file gpurun_out/%s "
                 "python -m paper_2407_16586_b200.profile_run ...\n    python -m paper_2407_16586_b200.ncu_classes gpurun_out/%s %s\n\n"
                 % (",".join(METRICS), os.path.basename(src), os.path.basename(src), out))
        fh.write("Kernel sources hash `%s`; %d launches, %.1f ms under ncu (serialised, cold cache: read the SHARES).  FLOP = 2 DFMA + DMUL + DADD "
                 "(thread-level, predicated on).\n\n" % (rec["source_hash"], len(launches), total_ns * 1e-6))
        fh.write("| class | kernel | launches | share of time | executed GFLOP | TFLOP/s under ncu | FP64 pipe % | warps active % | issue active % | "
                 "L1 wavefronts % | DFMA:DMUL:DADD | regs | DRAM GB (r+w) | local-memory MB |\n|---|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
        for name, c in rows:
            tot = max(c["dfma"] + c["dmul"] + c["dadd"], 1.0)
            fh.write("| %s | %s | %d | %.1f %% | %.1f | %.2f | %.1f | %.1f | %.1f | %.1f | %.2f:%.2f:%.2f | %d | %.2f | %.1f |\n"
                     % (name, c["kind"], c["launches"], 100.0 * c["ns"] / total_ns, c["flops"] * 1e-9, c["tflops_under_ncu"], c["fp64_pipe_pct"],
                        c["warps_active_pct"], c["issue_active_pct"], c["l1_wavefronts_pct"], c["dfma"] / tot, c["dmul"] / tot, c["dadd"] / tot,
                        c["regs"], (c["dram_read"] + c["dram_write"]) * 1e-9, c["local_bytes"] * 1e-6))
    print("wrote %s.md / .json (%d classes)" % (out, len(per)))


if __name__ == "__main__":
    main()
