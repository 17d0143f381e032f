"""The measurement tooling bench.py relies on (paper_1406_4254_b200/ncu_traffic.py): per-step sums from an `ncu --page raw --csv`
export, the key-metric summary, and the refusal of a capture taken from other kernel sources.  Synthetic CSV, no GPU."""
import json
import os

from paper_1406_4254_b200 import ncu_traffic as T

HDR = ["ID", "Kernel Name", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
       "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum", "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
       "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active",
       "launch__registers_per_thread", "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
       "smsp__average_warp_issue_stalled_wait_per_issue_active.ratio"]
UNITS = ["", "", "us", "Mbyte", "Kbyte", "inst", "inst", "inst", "%", "register/thread", "inst", "inst"]
ROWS = [
    ["0", "void etics::scf_accumulate_kernel<6, 1>(const double *)", "100.5", "32", "8", "1,000", "200", "30", "46.5", "128", "0.7", "1.9"],
    ["1", "etics::scf_finalize_kernel(const double *)", "5", "1", "4", "0", "10", "20", "1.0", "32", "0.1", "0.2"],
    ["2", "void etics::scf_eval_kernel<6, 11, 0>(const double *)", "150", "24", "1000", "3000", "500", "60", "73.0", "128", "0.0", "1.2"],
    ["3", "void etics::scf_accumulate_kernel<6, 1>(const double *)", "99.5", "32", "8", "1,000", "200", "30", "47.5", "128", "0.7", "1.9"],
    ["4", "etics::scf_finalize_kernel(const double *)", "5", "1", "4", "0", "10", "20", "1.0", "32", "0.1", "0.2"],
    ["5", "void etics::scf_eval_kernel<6, 11, 0>(const double *)", "150", "24", "1000", "3000", "500", "60", "72.0", "128", "0.0", "1.2"],
]


def write_csv(path):
    q = lambda xs: ",".join('"%s"' % x for x in xs)
    with open(path, "w") as f:
        f.write("==PROF== some banner line\n")
        for r in [HDR, UNITS] + ROWS:
            f.write(q(r) + "\n")


def test_extract_per_step_sums(tmp_path):
    p = tmp_path / "raw.csv"
    write_csv(p)
    d = T.extract(str(p))
    assert d["steps_in_capture"] == 2                      # = launches of the SCF evaluation kernel
    acc = d["kernels"]["scf_accumulate(+finalize)"]
    assert acc["launches_per_step"] == 2.0                 # accumulate + finalize
    assert acc["dram_read_bytes"] == 33e6 and acc["dram_write_bytes"] == 12e3 and acc["dram_bytes"] == 33e6 + 12e3
    assert acc["dfma"] == 1000 and acc["dmul"] == 210 and acc["dadd"] == 50
    assert abs(acc["duration_us_under_ncu"] - 105.0) < 1e-9
    assert acc["fp64_pipe_pct_max"] == 47.5                # the maximum over the group's launches, not a sum
    ev = d["kernels"]["scf_eval"]
    assert ev["dram_bytes"] == 24e6 + 1e6 and ev["dfma"] == 3000
    assert "mex_sort" not in d["kernels"]                 # kernels that did not run are absent


def test_summary_lists_first_launch_of_every_kernel(tmp_path):
    p = tmp_path / "raw.csv"
    write_csv(p)
    s = T.summary(str(p), "c1")
    assert s.count("Kernel Name") == 3 and T.kernel_source_hash() in s.splitlines()[0]
    assert "gpu__time_duration.sum" in s and "100.5 us" in s and "99.5 us" not in s
    assert "stalls per issue: wait 1.90, barrier 0.70" in s


def test_stale_capture_is_refused(tmp_path, monkeypatch):
    prof = tmp_path / "profiles"
    prof.mkdir()
    monkeypatch.setattr(T, "HERE", str(tmp_path / "pkg"))   # load() looks for ../profiles next to the package
    os.makedirs(tmp_path / "pkg")
    monkeypatch.setattr(T, "kernel_source_hash", lambda: "aaaaaaaaaaaaaaaa")
    kernels, why = T.load("c9")
    assert kernels == {} and "no capture" in why
    (prof / "traffic_c9.json").write_text(json.dumps({"kernel_source_hash": "bbbbbbbbbbbbbbbb", "kernels": {"scf_eval": {"dram_bytes": 1.0}}}))
    kernels, why = T.load("c9")
    assert kernels == {} and "other kernel sources" in why
    (prof / "traffic_c9.json").write_text(json.dumps({"kernel_source_hash": "aaaaaaaaaaaaaaaa", "kernels": {"scf_eval": {"dram_bytes": 1.0}}}))
    kernels, why = T.load("c9")
    assert why is None and kernels["scf_eval"]["dram_bytes"] == 1.0


def test_committed_captures_match_the_committed_kernel_sources():
    """profiles/traffic_*.json should have been captured from the sources in the tree (bench.py reports null with the reason
    otherwise).  A stale capture is reported as a skip, not a failure: it says "re-capture", not "the code is wrong"."""
    import pytest
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    stale = []
    for w in ("c1", "c2c3", "c4", "c5"):
        with open(os.path.join(root, "profiles", f"traffic_{w}.json")) as f:
            if json.load(f)["kernel_source_hash"] != T.kernel_source_hash():
                stale.append(w)
    if stale:
        pytest.skip(f"captures {stale} were taken from other kernel sources: re-capture (profiles/r2_summary.md has the commands)")
