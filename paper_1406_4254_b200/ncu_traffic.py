"""Turn an `ncu --page raw --csv` export of a bench.py run into the per-kernel DRAM-traffic / executed-fp64 file that
bench.py reports as `traffic` (profiles/traffic_<workload>.json).

    ncu -i prof.ncu-rep --page raw --csv > raw.csv
    python -m paper_1406_4254_b200.ncu_traffic raw.csv <workload> "<the ncu command that made prof.ncu-rep>" > profiles/traffic_<workload>.json
    python -m paper_1406_4254_b200.ncu_traffic --summary raw.csv <workload>     # key metrics of the first launch of every kernel (text)

The file records a hash of the kernel sources it was captured from (kernel_source_hash below); bench.py reports the
numbers only while that hash is the one of the sources it runs, so a capture can never outlive the kernels it measured.
Figures are per STEP: sums over the kernels' launches divided by the number of steps in the capture (= launches of the
SCF evaluation kernel, or of the MEX evaluation kernel when the workload has no SCF leg).
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))

# bench.py kernel key -> regex on the ncu kernel name
GROUPS = {
    "scf_accumulate(+finalize)": r"scf_accumulate_kernel|scf_finalize_kernel",
    "scf_eval": r"scf_eval_kernel",
    "mex_sort": r"mex_sort_",
    "mex_gather_totals": r"mex_gather_totals_kernel",
    "mex_tilescan": r"mex_tilescan_kernel",
    "mex_evaluate(+unpack)": r"mex_evaluate_kernel|mex_unpack_kernel",
}
METRICS = {
    "dram_read_bytes": "dram__bytes_read.sum",
    "dram_write_bytes": "dram__bytes_write.sum",
    "dfma": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "dmul": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "dadd": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "duration_ns": "gpu__time_duration.sum",
    "fp64_pipe_pct": "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
}
UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9, "usecond": 1e3,
        "nsecond": 1.0, "msecond": 1e6, "second": 1e9}


def kernel_source_hash() -> str:
    """sha256 over the CUDA sources and the public header (what the kernels are built from)."""
    h = hashlib.sha256()
    files = sorted(os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc")) if f.endswith((".cu", ".cuh")))
    files.append(os.path.join(os.path.dirname(HERE), "include", "etics.h"))
    for f in files:
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def _num(v: str) -> float:
    return float(v.replace(",", "")) if v not in ("", "n/a") else 0.0


def extract(raw_csv: str) -> dict:
    with open(raw_csv) as f:
        rows = [r for r in csv.reader(l for l in f if not l.startswith("=="))]
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    out = {k: {m: 0.0 for m in METRICS} | {"launches": 0} for k in GROUPS}
    for r in rows[2:]:
        name = r[col["Kernel Name"]]
        for key, pat in GROUPS.items():
            if re.search(pat, name):
                g = out[key]
                g["launches"] += 1
                for m, ncu_name in METRICS.items():
                    if ncu_name in col:
                        v = _num(r[col[ncu_name]]) * UNIT.get(units[col[ncu_name]], 1.0)
                        g[m] = max(g[m], v) if m == "fp64_pipe_pct" else g[m] + v
                break
    steps = out["scf_eval"]["launches"] or sum(1 for r in rows[2:] if "mex_evaluate_kernel" in r[col["Kernel Name"]]) or 1
    res = {}
    for key, g in out.items():
        if not g["launches"]:
            continue
        res[key] = {"launches_per_step": g["launches"] / steps,
                    "dram_bytes": (g["dram_read_bytes"] + g["dram_write_bytes"]) / steps,
                    "dram_read_bytes": g["dram_read_bytes"] / steps, "dram_write_bytes": g["dram_write_bytes"] / steps,
                    "dfma": g["dfma"] / steps, "dmul": g["dmul"] / steps, "dadd": g["dadd"] / steps,
                    "duration_us_under_ncu": g["duration_ns"] / steps / 1e3, "fp64_pipe_pct_max": g["fp64_pipe_pct"]}
    return {"steps_in_capture": steps, "kernels": res}


def load(workload: str) -> tuple[dict, str | None]:
    """(per-kernel figures, reason they are unavailable or None) for bench.py."""
    path = os.path.join(os.path.dirname(HERE), "profiles", f"traffic_{workload}.json")
    if not os.path.exists(path):
        return {}, f"no capture committed for workload {workload}"
    with open(path) as f:
        d = json.load(f)
    if d.get("kernel_source_hash") != kernel_source_hash():
        return {}, f"capture {os.path.basename(path)} was taken from other kernel sources ({d.get('kernel_source_hash')} != {kernel_source_hash()})"
    return d.get("kernels", {}), None


SUMMARY_METRICS = [
    "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "launch__registers_per_thread",
    "launch__grid_size", "launch__block_size", "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
    "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum", "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
]
STALL = re.compile(r"smsp__average_warps?_issue_stalled_(\w+)_per_issue_active\.ratio")


def summary(raw_csv: str, workload: str) -> str:
    """Key metrics of the FIRST launch of every kernel in the capture, as text (profiles/*_ncu_full_metrics.txt)."""
    with open(raw_csv) as f:
        rows = [r for r in csv.reader(l for l in f if not l.startswith("=="))]
    hdr, units = rows[0], rows[1]
    col = {h: i for i, h in enumerate(hdr)}
    seen, out = set(), [f"===== workload {workload} (kernel_source_hash {kernel_source_hash()}) ====="]
    for r in rows[2:]:
        name = r[col["Kernel Name"]]
        if name in seen:
            continue
        seen.add(name)
        out.append("-----")
        out.append(f"  {'Kernel Name':<80} {name}")
        for m in SUMMARY_METRICS:
            if m in col and r[col[m]] not in ("", "n/a"):
                out.append(f"  {m:<80} {r[col[m]]} {units[col[m]]}")
        stalls = sorted(((_num(r[i]), STALL.match(h).group(1)) for h, i in col.items() if STALL.match(h) and r[i] not in ("", "n/a")),
                        reverse=True)[:6]
        if stalls:
            out.append("  stalls per issue: " + ", ".join(f"{n} {v:.2f}" for v, n in stalls))
    return "\n".join(out) + "\n"


if __name__ == "__main__":
    if sys.argv[1] == "--summary":
        sys.stdout.write(summary(sys.argv[2], sys.argv[3]))
        sys.exit(0)
    raw, workload, command = sys.argv[1], sys.argv[2], sys.argv[3]
    d = extract(raw)
    d = {"workload": workload, "kernel_source_hash": kernel_source_hash(), "command": command,
         "note": "per step; dram_bytes = dram__bytes_read.sum + dram__bytes_write.sum; dfma/dmul/dadd = executed thread instructions"} | d
    json.dump(d, sys.stdout, indent=1)
    print()
