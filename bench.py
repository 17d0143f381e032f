#!/usr/bin/env python
"""bench.py — one JSON line for the ETICS hot path on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path over one particle set: SCF full force calculation (etics_scf_coeffs +
etics_scf_force, BASELINE.json configs[1]) followed by MEX full force calculation (etics_mex_force from unsorted
input, configs[2]) on the same N = 10^6 Hernquist sphere.  `value` = particles pushed through such a step per
second with inputs resident in HBM; `e2e` = the same through the host-buffer C-ABI calls (H2D + D2H inside).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c2c3|c4|c5]

N > 1 (torchrun): replicas only — each rank runs the same step on its own particle set, no collective on the
data path; time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "particles/s through one full force calculation by each method (SCF nmax=10,lmax=6 + MEX lmax=6), N=1e6, fp64"
UNIT = "particles/s"

WORKLOADS = {
    # name: (description, model, N, axes, (nmax, lmax) or None, mex lmax or None)
    "c2c3": ("BASELINE.json configs[1]+configs[2]: N=1e6 Hernquist sphere (a=1, r<=300), SCF (nmax,lmax)=(10,6) "
             "full force calc + MEX lmax=6 full force calc", "hernquist", 1_000_000, (1.0, 1.0, 1.0), (10, 6), 6),
    "c4": ("BASELINE.json configs[3]: N=1e7 triaxial Hernquist (1,0.8,0.6), SCF (20,10) full force calc",
           "hernquist", 10_000_000, (1.0, 0.8, 0.6), (20, 10), None),
    "c5": ("BASELINE.json configs[4]: N=1e8 Plummer sphere (r<=100), SCF (10,6) + MEX lmax=8 full force calcs",
           "plummer", 100_000_000, (1.0, 1.0, 1.0), (10, 6), 8),
}

# Paper's own figures for this workload (Tesla K20, context only): SCF 0.16 s + MEX 0.15 s at N=1e6.
PAPER_STEP_SECONDS = {"c2c3": 0.16 + 0.15}

FP64_LANES_PER_SM = 64   # 148 SMs x 64 fp64 FMA lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s


def num_lm(lmax):
    return (lmax + 1) * (lmax + 2) // 2


# ---- algorithmic work per particle (restated in DESIGN.md "Rooflines") -----------------------
def flops_scf_coeffs(nmax, lmax):
    L = num_lm(lmax); T = (nmax + 1) * L
    return 4 * T + 6 * (nmax + 1) * (lmax + 1) + 8 * L + 60


def flops_scf_eval(nmax, lmax):
    L = num_lm(lmax); T = (nmax + 1) * L
    return 8 * T + 24 * L + 12 * (nmax + 1) * (lmax + 1) + 100


def flops_mex_aggregate(lmax):
    return 16 * num_lm(lmax) + 30


def flops_mex_evaluate(lmax):
    return 54 * num_lm(lmax) + 70


BYTES_KEYGEN = 32 + 12 + 32     # read pos + mass, write key + index and the packed (x,y,z,m) record
BYTES_RADIX_PASS = 24           # read key+index, write key+index
BYTES_GATHER = 4 + 32 + 56 + 4  # read index, one 32-byte sector of (x,y,z,m), write the geometry record + index
BYTES_SCATTER = 32              # acc + pot at the original index


def ncu_traffic(workload):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of each kernel, from the committed
    `ncu --set full` capture of this workload (profiles/traffic_<workload>.json names the capture); {} if none."""
    path = os.path.join(ROOT, "profiles", f"traffic_{workload}.json")
    if not os.path.exists(path):
        return {}
    with open(path) as f:
        return json.load(f).get("dram_bytes_per_launch", {})


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    BITS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int, period=0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self._stop, self._thr, self._h = period, threading.Event(), None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:   # NVML unavailable: report nulls rather than fail the bench
            self._h = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for bit, name in self.BITS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self._h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def max_over_ranks(x: float, device) -> float:
    """Max of a per-rank scalar over all ranks (identity at world size 1): the timing rule for N > 1."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_seed(rank: int) -> int:
    """Replicas only: rank r draws its own particle set from seed r."""
    return int(rank)


def whole_job_value(world: int, n_per_rank: int, ms_per_step: float) -> float:
    """Particles per second over all replicas: every rank pushed n_per_rank particles through each step."""
    return world * n_per_rank / (ms_per_step * 1e-3)


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ================================================================================================================
# reference arm: the CPU oracle as it stands, on the box's host cores (the only other place that may run oracle/)
# ================================================================================================================
def oracle_step_seconds(pos, mass, scf, mex_lmax, reps=1):
    import oracle
    cores = oracle.num_threads(0)
    parts = {"scf_coeffs_s": 0.0, "scf_force_s": 0.0, "mex_force_s": 0.0}
    t_all = time.perf_counter()
    for _ in range(reps):
        if scf is not None:
            t = time.perf_counter()
            A, B = oracle.scf_coeffs(pos, mass, scf[0], scf[1])
            parts["scf_coeffs_s"] += time.perf_counter() - t
            t = time.perf_counter()
            oracle.scf_force(pos, scf[0], scf[1], A, B)
            parts["scf_force_s"] += time.perf_counter() - t
        if mex_lmax is not None:
            t = time.perf_counter()
            oracle.mex_force(pos, mass, mex_lmax)
            parts["mex_force_s"] += time.perf_counter() - t
    total = time.perf_counter() - t_all
    return total / reps, cores, {k: v / reps for k, v in parts.items()}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1406_4254_b200 import workloads as W
    desc, model, n_full, axes, scf, mex_lmax = WORKLOADS[args.workload]
    # bounded sample: calibrate the oracle's rate on 20k particles, then size each step so that the whole
    # --steps/--warmup run takes about args.ref_budget seconds (particle k depends only on (seed, k), so the
    # first n particles of the workload are a prefix of the full set)
    n0 = min(n_full, 20_000)
    pos, mass = W.particles(model, n0, seed=0, axes=axes)
    t0, _, _ = oracle_step_seconds(pos, mass, scf, mex_lmax)
    rate = n0 / t0
    n = int(min(n_full, max(2_000, rate * args.ref_budget / (args.steps + args.warmup))))
    pos, mass = W.particles(model, n, seed=0, axes=axes)
    times = []
    cores = 1
    for i in range(args.warmup + args.steps):
        t, cores, parts = oracle_step_seconds(pos, mass, scf, mex_lmax)
        if i >= args.warmup:
            times.append(t)
    sec = float(np.mean(times))
    value = n / sec
    sample = f"each step = the oracle (OpenMP SCF on {cores} threads, single-thread streaming MEX) on {n} particles of the workload"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": desc, "sample_particles": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ================================================================================================================
# our arm
# ================================================================================================================
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_1406_4254_b200 import binding as E
    from paper_1406_4254_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    E.lib()
    E.etics_init()

    desc, model, N, axes, scf, mex_lmax = WORKLOADS[args.workload]
    pos_np, mass_np = W.particles(model, N, seed=replica_seed(rank), axes=axes)   # one replica per rank, own particle set
    pos = torch.from_numpy(pos_np).cuda()
    mass = torch.from_numpy(mass_np).cuda()
    acc = torch.empty((3, N), dtype=torch.float64, device="cuda")
    pot = torch.empty(N, dtype=torch.float64, device="cuda")
    acc2, pot2 = torch.empty_like(acc), torch.empty_like(pot)
    if scf is not None:
        nmax, lmax = scf
        T = (nmax + 1) * num_lm(lmax)
        A = torch.empty(T, dtype=torch.float64, device="cuda")
        B = torch.empty_like(A)
        ws_scf = torch.empty(E.etics_workspace_bytes(E.ETICS_WS_SCF_COEFFS, N, nmax, lmax), dtype=torch.uint8, device="cuda")
    if mex_lmax is not None:
        ws_mex = torch.empty(E.etics_workspace_bytes(E.ETICS_WS_MEX_FORCE, N, 0, mex_lmax), dtype=torch.uint8, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def scf_coeffs():
        E.etics_scf_coeffs(pos, mass, nmax, lmax, A, B, ws_scf)

    def scf_force():
        E.etics_scf_force(pos, nmax, lmax, A, B, acc, pot)

    def mex_force():
        E.etics_mex_force(pos, mass, mex_lmax, acc2, pot2, ws_mex)

    def step():
        if scf is not None:
            scf_coeffs()
            scf_force()
        if mex_lmax is not None:
            mex_force()

    launches_per_step = (3 if scf is not None else 0) + (14 if mex_lmax is not None else 0)

    def timed(fn, iters, warmup):
        """Per-iteration CUDA-event times (ms) with an L2 flush before every iteration (outside the events)."""
        for _ in range(warmup):
            flush.zero_()
            fn()
        torch.cuda.synchronize()
        evs = []
        for _ in range(iters):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            evs.append((a, b))
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- the timed region: exactly K steps ---------------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    barrier()
    with ClockSampler(physical_gpu_index(local_rank)) as clk:
        wall0 = time.perf_counter()
        ms = timed(step, args.steps, 0)
        barrier()
        wall = time.perf_counter() - wall0
    ms_per_step = max_over_ranks(float(np.sum(ms)), "cuda") / args.steps
    value = whole_job_value(world, N, ms_per_step)

    # ---- end to end through the host-buffer C-ABI calls ----------------------------------------------------------
    e2e_steps = max(3, min(args.steps, 20))
    pos_h, mass_h = torch.from_numpy(pos_np).pin_memory(), torch.from_numpy(mass_np).pin_memory()
    acc_h, pot_h = torch.empty((3, N), dtype=torch.float64).pin_memory(), torch.empty(N, dtype=torch.float64).pin_memory()
    h2d = d2h = 0
    if scf is not None:
        A_h, B_h = torch.empty(T, dtype=torch.float64).pin_memory(), torch.empty(T, dtype=torch.float64).pin_memory()
        scr_scf = torch.empty(E.etics_host_scratch_bytes(0, N, nmax, lmax), dtype=torch.uint8, device="cuda")
        h2d += 32 * N
        d2h += 32 * N + 16 * T
    if mex_lmax is not None:
        scr_mex = torch.empty(E.etics_host_scratch_bytes(1, N, 0, mex_lmax), dtype=torch.uint8, device="cuda")
        h2d += 32 * N
        d2h += 32 * N

    def e2e_step():
        if scf is not None:
            E.etics_scf_full_host(pos_h, mass_h, nmax, lmax, acc_h, pot_h, scr_scf, A_h, B_h)
        if mex_lmax is not None:
            E.etics_mex_full_host(pos_h, mass_h, mex_lmax, acc_h, pot_h, scr_mex)

    e2e_ms = timed(e2e_step, e2e_steps, 2)
    e2e_value = whole_job_value(world, N, max_over_ranks(float(np.sum(e2e_ms)), "cuda") / e2e_steps)
    if scf is not None:
        del scr_scf
    if mex_lmax is not None:
        del scr_mex

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- per-kernel times (rank 0), live, CUDA events, L2 flushed before each -------------------------------------
    peaks = measured_peaks()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    fp64_peak_tf = sms * FP64_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    k_iters = max(5, min(args.steps, 30))
    kernels = {}

    def add(name, ms_list, bound, work, launches=1):
        t = float(np.mean(ms_list))
        if bound == "alu":
            ach, peak, unit = work / (t * 1e-3) / 1e12, fp64_peak_tf, "TFLOP/s"
        else:
            ach, peak, unit = work / (t * 1e-3) / 1e9, peaks["hbm_gbs"], "GB/s"
        kernels[name] = {"ms": t, "ms_min": float(np.min(ms_list)), "launches": launches, "bound": bound,
                         "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak}

    phases = {}
    if scf is not None:
        c = timed(scf_coeffs, k_iters, 2)
        f = timed(scf_force, k_iters, 2)
        phases["scf_coeffs_ms"], phases["scf_force_ms"] = float(np.mean(c)), float(np.mean(f))
        add("scf_accumulate(+finalize)", c, "alu", N * flops_scf_coeffs(nmax, lmax), 2)
        add("scf_eval", f, "alu", N * flops_scf_eval(nmax, lmax))
    if mex_lmax is not None:
        m = timed(mex_force, k_iters, 2)
        phases["mex_force_ms"] = float(np.mean(m))
        st = {k: [] for k in E.MEX_STAGES}
        for i in range(k_iters + 2):
            flush.zero_()
            r = E.etics_mex_force_timed(pos, mass, mex_lmax, acc2, pot2, ws_mex)
            if i >= 2:
                for k, v in r.items():
                    st[k].append(v)
        add("mex_keygen(+clear)", st["keygen"], "hbm", N * BYTES_KEYGEN)
        add("mex_radix_pass x8", st["radix_passes"], "hbm", N * BYTES_RADIX_PASS * 8, 8)
        add("mex_gather", st["gather"], "hbm", N * BYTES_GATHER)
        add("mex_aggregate", st["aggregate"], "alu", N * flops_mex_aggregate(mex_lmax))
        add("mex_tilescan", st["tilescan"], "hbm", 0)
        add("mex_evaluate(+unpack)", st["evaluate"], "alu", N * flops_mex_evaluate(mex_lmax), 2)
    traffic = ncu_traffic(args.workload)
    for k in kernels:
        kernels[k]["traffic"] = traffic.get(k)
    dom = max((k for k in kernels if kernels[k]["achieved"] > 0), key=lambda k: kernels[k]["ms"])
    d = kernels[dom]
    roofline = {"kernel": dom, "bound": d["bound"], "achieved": d["achieved"], "peak": d["peak"], "unit": d["unit"],
                "frac": d["frac"], "traffic": d["traffic"], "share_of_step": d["ms"] / sum(v["ms"] for v in kernels.values()),
                "peak_source": ("148 SMs x 64 fp64 lanes x 2 x sm_max_mhz (DESIGN.md)" if d["bound"] == "alu" else peaks["source"])}

    # measured fp64 FMA rate of this GPU (register-resident DFMA chains), for context beside the derived peak
    sink = torch.zeros(8, dtype=torch.float64, device="cuda")
    fl = [0.0]

    def probe():
        fl[0] = E.etics_probe_dfma(20000, sink)

    pm = timed(probe, 5, 2)
    dfma_tf = fl[0] / (min(pm) * 1e-3) / 1e12

    # ---- CPU baseline: the oracle as it stands, on this box's host cores, bounded sample -------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_cpu = min(N, 1_000_000)
        sec, cores, parts = oracle_step_seconds(pos_np[:, :n_cpu].copy(), mass_np[:n_cpu].copy(), scf, mex_lmax, reps=2)
        cpu = {"value": n_cpu / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"2 repetitions of the same step on the first {n_cpu} particles (SCF legs OpenMP over {cores} threads, "
                         f"MEX streaming sweeps single-threaded)", "seconds_per_step": sec, **parts}

    clocks = clk.summary()
    paper = PAPER_STEP_SECONDS.get(args.workload)
    line = {
        "metric": METRIC if args.workload == "c2c3" else f"particles/s through one full force calculation ({args.workload})",
        "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (value / world) / (N / paper) if paper else None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "N_per_gpu": N, "scf": scf, "mex_lmax": mex_lmax, "seed": "rank",
                   "l2": "flushed before every timed step (256 MiB memset, outside the events)",
                   "parallelism": "replicas only (no data-path collective)" if world > 1 else "single GPU"},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks, "wall_s_timed_region": wall,
        "roofline": roofline, "kernels": kernels, "phases_ms": phases,
        "fp64_fma_probe_tflops": dfma_tf,
        "cpu_baseline": cpu,
        "paper_context": {"k20_step_seconds": paper, "note": "Tesla K20, PAPER.md:275,281; context, not the target"} if paper else None,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="c2c3")
    ap.add_argument("--ref-budget", type=float, default=90.0, help="seconds of oracle time for the whole --impl reference run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
