#!/usr/bin/env python
"""bench.py — one JSON line for the ETICS hot path on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path over one particle set: SCF full force calculation (etics_scf_coeffs +
etics_scf_force, BASELINE.json configs[1]) followed by MEX full force calculation (etics_mex_force from unsorted
input, configs[2]) on the same N = 10^6 Hernquist sphere.  `value` = particles pushed through such a step per
second with inputs resident in HBM; `e2e` = the same through the host-buffer C-ABI calls (H2D + D2H inside).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c1|c2c3|c4|c5]

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
    "c1": ("BASELINE.json configs[0]: N=1e4 Hernquist sphere (a=1, r<=300), SCF (nmax,lmax)=(10,6): one coefficient pass + "
           "one evaluation", "hernquist", 10_000, (1.0, 1.0, 1.0), (10, 6), None),
    "c2c3": ("BASELINE.json configs[1]+configs[2]: N=1e6 Hernquist sphere (a=1, r<=300), SCF (nmax,lmax)=(10,6) "
             "full force calc + MEX lmax=6 full force calc", "hernquist", 1_000_000, (1.0, 1.0, 1.0), (10, 6), 6),
    "c4": ("BASELINE.json configs[3]: N=1e7 triaxial Hernquist (1,0.8,0.6), SCF (20,10) full force calc",
           "hernquist", 10_000_000, (1.0, 0.8, 0.6), (20, 10), None),
    "c5": ("BASELINE.json configs[4]: N=1e8 Plummer sphere (r<=100), SCF (10,6) + MEX lmax=8 full force calcs",
           "plummer", 100_000_000, (1.0, 1.0, 1.0), (10, 6), 8),
}

# Paper's own figures for this workload (Tesla K20, context only): SCF 0.16 s + MEX 0.15 s at N=1e6.
PAPER_STEP_SECONDS = {"c2c3": 0.16 + 0.15}

FP64_LANES_PER_SM = 64   # 148 SMs x 64 fp64 FMA lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s (derived)


def num_lm(lmax):
    return (lmax + 1) * (lmax + 2) // 2


# ---- algorithmic work per particle: SURVEY.md §8(d)'s counts (fractions are quoted against THESE) --------------------
def flops_scf_coeffs(nmax, lmax):
    L = num_lm(lmax); T = (nmax + 1) * L
    return 4 * T + 6 * (nmax + 1) * (lmax + 1) + 8 * L + 60


def flops_scf_eval(nmax, lmax):
    L = num_lm(lmax); T = (nmax + 1) * L
    return 8 * T + 24 * L + 12 * (nmax + 1) * (lmax + 1) + 100


def flops_mex_moments(lmax):      # M4 + M5a
    return 16 * num_lm(lmax) + 30


def flops_mex_evaluate(lmax):     # M5c + M6 + M7
    return 54 * num_lm(lmax) + 70


# SURVEY §8(d) "MEX sort": key-gen 24 + 12, histogram 8, P digit passes x 24 with P = 6 (sign and constant exponent bits
# skipped).  The shipped sort moves fewer bytes (one 8-byte word per particle and pass); that figure is printed beside it.
BYTES_SORT_SURVEY = 24 + 12 + 8 + 6 * 24
BYTES_GATHER_SURVEY = 4 + 32 + 32            # index, packed record read, sorted record written (ours writes 56 + 4)
BYTES_EVAL_SURVEY = 32 + 32 + 32             # two reads of the sorted records, one scattered 32-byte write
BYTES_TILESCAN_PER_ROW_TILE = 16             # every tile total read and written once


def bytes_sort_actual(N, launches, pack):
    single_wave = launches == 2
    passes, fix = (3, 12) if single_wave else (4, 12)
    return (24 + 8 + (40 if pack else 0)) + 16 + passes * 24 + fix


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
def oracle_step_seconds(pos, mass, scf, mex_lmax, reps=1, threads=0):
    import oracle
    cores = oracle.num_threads(threads)
    parts = {"scf_coeffs_s": 0.0, "scf_force_s": 0.0, "mex_force_s": 0.0}
    t_all = time.perf_counter()
    for _ in range(reps):
        if scf is not None:
            t = time.perf_counter()
            A, B = oracle.scf_coeffs(pos, mass, scf[0], scf[1], threads)
            parts["scf_coeffs_s"] += time.perf_counter() - t
            t = time.perf_counter()
            oracle.scf_force(pos, scf[0], scf[1], A, B, threads)
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
    from paper_1406_4254_b200 import ncu_traffic
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
    nmax = lmax = T = None
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

    mex_launches = E.etics_kernel_launches(E.ETICS_WS_MEX_FORCE, N) if mex_lmax is not None else 0
    launches_per_step = (3 if scf is not None else 0) + mex_launches

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

    # ---- end to end through the host-buffer C-ABI call: ONE upload, both methods, copies overlapped on a second stream ----
    e2e_steps = max(3, min(args.steps, 20))
    pos_h, mass_h = torch.from_numpy(pos_np).pin_memory(), torch.from_numpy(mass_np).pin_memory()
    acc_h, pot_h = torch.empty((3, N), dtype=torch.float64).pin_memory(), torch.empty(N, dtype=torch.float64).pin_memory()
    h2d = 32 * N
    if scf is not None and mex_lmax is not None:
        acc2_h, pot2_h = torch.empty((3, N), dtype=torch.float64).pin_memory(), torch.empty(N, dtype=torch.float64).pin_memory()
        A_h, B_h = torch.empty(T, dtype=torch.float64).pin_memory(), torch.empty(T, dtype=torch.float64).pin_memory()
        scr = torch.empty(E.etics_step_host_scratch_bytes(N, nmax, lmax, mex_lmax), dtype=torch.uint8, device="cuda")
        cs = torch.cuda.Stream()
        d2h = 64 * N + 16 * T
        e2e_api = "etics_step_host (one upload, copies on a second stream)"

        def e2e_step():
            E.etics_step_host(pos_h, mass_h, nmax, lmax, mex_lmax, acc_h, pot_h, acc2_h, pot2_h, scr, A_h, B_h, copy_stream=cs)
    else:
        A_h, B_h = torch.empty(T, dtype=torch.float64).pin_memory(), torch.empty(T, dtype=torch.float64).pin_memory()
        scr = torch.empty(E.etics_host_scratch_bytes(0, N, nmax, lmax), dtype=torch.uint8, device="cuda")
        d2h = 32 * N + 16 * T
        e2e_api = "etics_scf_full_host"

        def e2e_step():
            E.etics_scf_full_host(pos_h, mass_h, nmax, lmax, acc_h, pot_h, scr, A_h, B_h)

    e2e_ms = timed(e2e_step, e2e_steps, 2)
    e2e_value = whole_job_value(world, N, max_over_ranks(float(np.sum(e2e_ms)), "cuda") / e2e_steps)
    del scr

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline denominators: the fp64 FMA rate this GPU sustains (register-resident DFMA chains), measured here ----
    peaks = measured_peaks()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    fp64_derived_tf = sms * FP64_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    sink = torch.zeros(8, dtype=torch.float64, device="cuda")
    fl = [0.0]

    def probe():
        fl[0] = E.etics_probe_dfma(20000, sink)

    pm = timed(probe, 5, 2)
    fp64_peak_tf = fl[0] / (min(pm) * 1e-3) / 1e12

    # ---- per-kernel times (rank 0), live, CUDA events, L2 flushed before each -------------------------------------
    k_iters = max(5, min(args.steps, 30))
    kernels = {}
    ncu, ncu_reason = ncu_traffic.load(args.workload)

    def add(name, ms_list, bound, flops=None, nbytes=None, launches=1, note=None):
        t = float(np.mean(ms_list))
        k = {"ms": t, "ms_min": float(np.min(ms_list)), "launches": launches, "bound": bound}
        if flops is not None:
            k["tflops"] = flops / (t * 1e-3) / 1e12
            k["frac_fp64"] = k["tflops"] / fp64_peak_tf
        if nbytes is not None:
            k["gbs"] = nbytes / (t * 1e-3) / 1e9
            k["frac_hbm"] = k["gbs"] / peaks["hbm_gbs"]
        if bound == "alu":
            k.update(achieved=k["tflops"], peak=fp64_peak_tf, unit="TFLOP/s", frac=k["frac_fp64"])
        else:
            k.update(achieved=k["gbs"], peak=peaks["hbm_gbs"], unit="GB/s", frac=k["frac_hbm"])
        if note:
            k["note"] = note
        m = ncu.get(name)
        k["traffic"] = m["dram_bytes"] if m else None
        if m:   # executed fp64 thread instructions per launch, beside the algorithmic count
            k["executed_fp64"] = {"dfma": m["dfma"], "dmul": m["dmul"], "dadd": m["dadd"],
                                  "flops": 2 * m["dfma"] + m["dmul"] + m["dadd"], "fp64_pipe_pct_under_ncu": m["fp64_pipe_pct_max"]}
        kernels[name] = k

    phases = {}
    if scf is not None:
        c = timed(scf_coeffs, k_iters, 2)
        f = timed(scf_force, k_iters, 2)
        phases["scf_coeffs_ms"], phases["scf_force_ms"] = float(np.mean(c)), float(np.mean(f))
        add("scf_accumulate(+finalize)", c, "alu", flops=N * flops_scf_coeffs(nmax, lmax), nbytes=32 * N, launches=2)
        add("scf_eval", f, "alu", flops=N * flops_scf_eval(nmax, lmax), nbytes=56 * N)
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
        Lm = num_lm(mex_lmax)
        tiles = (N + 255) // 256
        rows = 4 * Lm - 2 * (mex_lmax + 1)   # (cos, sin) x (q, p) running sums, no sin for m = 0
        sort_ms = [a + b for a, b in zip(st["sort"], st["sort_fallback"])]
        add("mex_sort", sort_ms, "hbm", nbytes=N * BYTES_SORT_SURVEY, launches=mex_launches - 4,
            note=f"bytes = SURVEY 8(d): 36 + 8 + 6 passes x 24 = {BYTES_SORT_SURVEY} B/particle; the shipped sort moves "
                 f"{bytes_sort_actual(N, mex_launches - 4, True)} B/particle ({'one cooperative kernel, 3 x 11-bit' if mex_launches - 4 == 2 else '4 x 9-bit passes, one kernel per phase'})")
        kernels["mex_sort"]["gbs_actual_bytes"] = N * bytes_sort_actual(N, mex_launches - 4, True) / (kernels["mex_sort"]["ms"] * 1e-3) / 1e9
        add("mex_gather_totals", st["gather_totals"], "alu", flops=N * flops_mex_moments(mex_lmax), nbytes=N * BYTES_GATHER_SURVEY,
            note="gather (SURVEY: 68 B/particle; ours writes 56-byte geometry records: 96) fused with the tile totals of the moments")
        add("mex_tilescan", st["tilescan"], "hbm", nbytes=rows * tiles * BYTES_TILESCAN_PER_ROW_TILE)
        add("mex_evaluate(+unpack)", st["evaluate"], "alu", flops=N * flops_mex_evaluate(mex_lmax), nbytes=N * BYTES_EVAL_SURVEY, launches=2,
            note="flops = SURVEY 8(d) evaluate only (54L+70); the kernel also recomputes the chunk sums (16L+30) instead of reading them back")
        kernels["mex_evaluate(+unpack)"]["frac_fp64_incl_recomputed_moments"] = \
            N * (flops_mex_evaluate(mex_lmax) + flops_mex_moments(mex_lmax)) / (kernels["mex_evaluate(+unpack)"]["ms"] * 1e-3) / 1e12 / fp64_peak_tf
    dom = max(kernels, key=lambda k: kernels[k]["ms"])
    d = kernels[dom]
    roofline = {"kernel": dom, "bound": d["bound"], "achieved": d["achieved"], "peak": d["peak"], "unit": d["unit"],
                "frac": d["frac"], "traffic": d["traffic"], "traffic_unavailable": ncu_reason,
                "share_of_step": d["ms"] / sum(v["ms"] for v in kernels.values()),
                "peak_source": (f"fp64 FMA rate measured in this run by etics_probe_dfma (derived 148 SMs x 64 lanes x 2 x sm_max_mhz = "
                                f"{fp64_derived_tf:.2f} TFLOP/s)" if d["bound"] == "alu" else peaks["source"]),
                "work_model": "SURVEY.md 8(d) algorithmic count"}


    # ---- force-only / potential-only variants beside the "both" figure --------------------------------
    variants = {}
    if scf is not None:
        variants["scf_force_ms"] = {
            "both": phases["scf_force_ms"],
            "potential_only": float(np.mean(timed(lambda: E.etics_scf_force_ex(pos, nmax, lmax, A, B, E.ETICS_WHAT_POTENTIAL, None, pot), k_iters, 2))),
            "force_only": float(np.mean(timed(lambda: E.etics_scf_force_ex(pos, nmax, lmax, A, B, E.ETICS_WHAT_FORCE, acc, None), k_iters, 2)))}
        ws_f32 = torch.empty(E.etics_workspace_bytes(E.ETICS_WS_SCF_FORCE_F32, N, nmax, lmax), dtype=torch.uint8, device="cuda")
        variants["scf_force_ms"]["both_fp32_arithmetic"] = float(np.mean(timed(
            lambda: E.etics_scf_force_f32(pos, nmax, lmax, A, B, E.ETICS_WHAT_BOTH, acc, pot, ws_f32), k_iters, 2)))
        scf_force()   # leave the fp64 results in acc, pot
    if mex_lmax is not None:
        variants["mex_force_ms"] = {
            "both": phases["mex_force_ms"],
            "potential_only": float(np.mean(timed(lambda: E.etics_mex_force_ex(pos, mass, mex_lmax, E.ETICS_WHAT_POTENTIAL, None, pot2, ws_mex), k_iters, 2))),
            "force_only": float(np.mean(timed(lambda: E.etics_mex_force_ex(pos, mass, mex_lmax, E.ETICS_WHAT_FORCE, acc2, None, ws_mex), k_iters, 2)))}

        # the shard calls of a radius-partitioned multi-GPU run, here with ONE shard holding every particle:
        # the same kernels as etics_mex_force plus the moment-vector kernels; the exchange between ranks is not in this number
        R = E.etics_mex_shard_rows(mex_lmax)
        shard_parts = torch.zeros((1, R), dtype=torch.float64, device="cuda")

        def one_shard():
            E.etics_mex_shard_moments(pos, mass, mex_lmax, ws_mex, totals=shard_parts[0])
            E.etics_mex_shard_force(N, mex_lmax, E.ETICS_WHAT_BOTH, E.etics_mex_shard_bases(shard_parts, 0, mex_lmax), ws_mex, acc2, pot2)
        variants["mex_force_ms"]["one_shard_moments_bases_force"] = float(np.mean(timed(one_shard, k_iters, 2)))

    # ---- time-stepping reuse: one leapfrog step with plain launches and as a replayed CUDA graph -----------------
    stepper = {}
    if N <= 10_000_000:
        vel = torch.zeros_like(pos)
        nst = 20

        def stepper_ms(method, nm, lm, graph):
            p2 = pos.clone()
            sp = E.Stepper(method, p2, vel, mass, 1e-6, nmax=nm, lmax=lm, use_graph=graph)
            sp.step(3)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            a.record()
            sp.step(nst)
            b.record()
            host = time.perf_counter() - t0
            torch.cuda.synchronize()
            sp.close()
            return {"device_ms_per_step": a.elapsed_time(b) / nst, "host_enqueue_ms_per_step": host * 1e3 / nst}

        if scf is not None:
            stepper["scf"] = {"plain": stepper_ms(0, nmax, lmax, False), "graph": stepper_ms(0, nmax, lmax, True)}
        if mex_lmax is not None:
            stepper["mex"] = {"plain": stepper_ms(1, 0, mex_lmax, False), "graph": stepper_ms(1, 0, mex_lmax, True)}
        stepper["note"] = ("kick-drift + force + kick per step, no L2 flush between steps, dt = 1e-6 (the second and later steps sort an "
                           "almost sorted list: an LSD radix sort does the same work either way)")

    # ---- CPU baseline: the oracle as it stands, on this box's host cores, bounded sample -------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_cpu = min(N, 1_000_000)
        pc, mc = pos_np[:, :n_cpu].copy(), mass_np[:n_cpu].copy()
        sec, cores, parts = oracle_step_seconds(pc, mc, scf, mex_lmax, reps=2)
        n_one = min(N, 250_000)
        sec1, _, parts1 = oracle_step_seconds(pos_np[:, :n_one].copy(), mass_np[:n_one].copy(), scf, mex_lmax, reps=1, threads=1)
        cpu = {"value": n_cpu / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"2 repetitions of the same step on the first {n_cpu} particles (SCF legs OpenMP over {cores} threads, "
                         f"MEX streaming sweeps single-threaded)", "seconds_per_step": sec, **parts,
               "single_thread": {"value": n_one / sec1, "unit": UNIT, "cores": 1,
                                 "sample": f"1 repetition on the first {n_one} particles, every leg on one thread", **parts1}}

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
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "ms_per_step": float(np.mean(e2e_ms)), "api": e2e_api},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks, "wall_s_timed_region": wall,
        "roofline": roofline, "kernels": kernels, "phases_ms": phases,
        "fp64_fma_probe_tflops": fp64_peak_tf, "fp64_derived_tflops": fp64_derived_tf,
        "variants": variants, "stepper": stepper,
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
