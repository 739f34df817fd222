#!/usr/bin/env python
"""Benchmark of the LJ MD hot path (arXiv 0709.3225) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c2_allpairs_32k|c3_cell_256k|c4a_cell_2048k|...] [--no-others]

A "step" is one velocity-Verlet step of the named workload (half-kick, drift + wrap, [cell
build,] force + PE + virial, half-kick + KE, reductions).  The headline workload is
BASELINE.json configs[1] (N = 32000, all-pairs); the cell-list configs and the rand48 config
are measured in the same run and reported under "others" (skip with --no-others), each with its
own roofline and oracle baseline.  Every system is generated on the product side (fcc lattice +
md_init_velocities), advanced untimed by its config's own number of steps so that the timed
state is the melted fluid (occupancy spread, FP64 queue lengths and list rebuild rate are the
fluid's, not the lattice's), and runs on a PyTorch side stream with PyTorch's caching allocator
(the binding's defaults).
Multi-GPU: the path does not shard in this build ("replicas only"):
under torchrun every rank runs an independent replica and `value` is the aggregate.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_0709_3225_b200 import workloads as wl  # noqa: E402

FP32_LANES_PER_SM = 128
FLOP_PER_PAIR_TEST = 8.0        # 3 sub + 1 mul + 2 fma; the compare is not a flop
FLOP_PER_INRANGE = 19.0
FLOP_PER_INRANGE_NO_ENERGY = 13.0   # a force-only launch (interior steps of md_step(K)) skips ~6 flop of U and r f per pair
NBR_PER_ATOM = lambda rho, rc: 4.0 / 3.0 * np.pi * rc ** 3 * rho  # noqa: E731


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


TRAFFIC_FILES = ("profiles/r03_traffic.txt", "profiles/r02_traffic.txt")


def ncu_traffic(workload):
    """(DRAM bytes per launch of the workload's dominant kernel, file it came from): dram__bytes_read.sum +
    dram__bytes_write.sum of one committed `ncu --set full` capture.  It is measured under ncu, so it cannot
    be taken live in this run; the JSON line names the file ("traffic_source")."""
    for rel in TRAFFIC_FILES:
        p = os.path.join(ROOT, rel)
        if not os.path.exists(p):
            continue
        for ln in open(p):
            f = ln.split()
            if len(f) == 3 and f[0] == workload:
                return float(f[2]), rel
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.thr.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])), mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v == "Active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(vals, dist, device):
    """Element-wise MAX of a list of timings over all ranks (the only collective of the bench:
    replicas share no data).  Works on any backend (nccl on GPUs, gloo in tests)."""
    import torch
    t = torch.tensor(list(vals), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_value(n_units_per_rank, world, ms_max):
    """Aggregate throughput of `world` independent replicas: units all ranks processed / slowest rank's time."""
    return world * n_units_per_rank / (ms_max * 1e-3)


# ----------------------------------------------------------------------------- our arm
def flush_l2(torch, buf):
    buf.add_(1)           # read + write 256 MB: larger than the 126 MB L2


def time_md(b, torch, sysd, algo, steps, warmup, flush, buf, options=None):
    """Returns dict with ms_per_step (flushed per-step timing), steady ms_per_step
    (md_step(K) back to back), per-phase times and kernel-launch counts.  The system is first advanced,
    untimed, by its config's own number of steps (sysd["steps"]): the timed state is the melted fluid."""
    N = sysd["N"]
    s = b.Sim(N, sysd["L"], rc=sysd["rc"], eps=sysd["eps"], sigma=sysd["sigma"], dt=sysd["dt"],
              shifted=sysd["shifted"])
    for k_, v_ in (options or {}).items():
        s.option(k_, v_)
    s.set_state(sysd["pos"], sysd["vel"])
    s.step(sysd["steps"], algo)                       # melt (untimed)
    s.step(warmup, algo)
    # two more untimed calls of the timed shape: md_step caches its CUDA graphs per buffer parity and
    # sort phase, and capture + instantiation is a one-time cost that does not belong in a step time
    s.step(steps, algo)
    s.step(steps, algo)
    torch.cuda.synchronize()
    # (1) steady state: K steps in one call, the way a user runs MD
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.stat("kernel_launches")
    e0.record()
    s.step(steps, algo)
    e1.record()
    torch.cuda.synchronize()
    steady_ms = e0.elapsed_time(e1) / steps
    launches = int(s.stat("kernel_launches") - l0)
    # (2) per-phase kernel timing with CUDA events inside the library (same stream)
    s.option("time_kernels", 1)
    s.step(steps, algo)
    t_force = s.stat("t_force_ms") / max(1.0, s.stat("n_force"))
    phases = {k: s.stat("t_%s_ms" % k) / steps for k in ("integrate", "build", "force", "force2", "other")}
    t_force2 = phases["force2"]
    s.option("time_kernels", 0)
    # (2b) PE and the virial evaluated on EVERY step (north_star: "LJ force and energy evaluation"): md_step(K) computes
    # them on its last step only, so this is md_step(1) K times, unflushed; first the wall figure, then the kernels
    s.step(1, algo)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        s.step(1, algo)
    e1.record()
    torch.cuda.synchronize()
    every_ms = e0.elapsed_time(e1) / steps
    s.option("time_kernels", 1)
    for _ in range(steps):
        s.step(1, algo)
    t_force_energy = s.stat("t_force_ms") / max(1.0, s.stat("n_force"))
    phases_energy = {k: s.stat("t_%s_ms" % k) / steps for k in ("integrate", "build", "force", "force2", "other")}
    s.option("time_kernels", 0)
    # (3) cold-L2 per-step timing: flush between steps, each step its own md_step(1); three repetitions of the K steps
    # (SURVEY 8(d)): the first is the headline, all three are reported with best and median
    flushed_ms, flushed_reps = None, []
    if flush:
        for _rep in range(3):
            tot = 0.0
            for _ in range(steps):
                flush_l2(torch, buf)
                e0.record()
                s.step(1, algo)
                e1.record()
                torch.cuda.synchronize()
                tot += e0.elapsed_time(e1)
            flushed_reps.append(tot / steps)
        flushed_ms = flushed_reps[0]
    ke, pe, w = s.energies()
    vl100 = None
    if algo == 2:
        # rebuild rate of the melted state: over the steps after the melt
        nb0, ns0 = s.stat("vl_builds"), s.stat("vl_steps")
        s.step(200, algo)
        vl100 = 100.0 * (s.stat("vl_builds") - nb0) / max(1.0, s.stat("vl_steps") - ns0)
    ncell = int(s.stat("ncell"))
    melted = s.get_state()
    s.close()
    return dict(vl_builds_per_100=vl100, steady_ms=steady_ms, flushed_ms=flushed_ms, flushed_reps=flushed_reps,
                every_step_energy_ms=every_ms, t_force_energy_kernel_ms=t_force_energy, phases_energy_ms=phases_energy,
                launches_per_step=launches / steps,
                t_force_kernel_ms=t_force, t_force2_kernel_ms=t_force2, phases_ms=phases, energy=ke + pe, ncell=ncell,
                melted=melted)


def time_md_e2e(b, torch, sysd, state, algo, calls, k):
    """End to end through the C ABI with HOST (pinned) buffers: every call uploads the state
    (md_set_state), advances k steps (md_step), and reads the state and the energies back.  Replacing the
    state makes the forces stale, so every call evaluates F(t) before its first step: k + 1 force
    evaluations per call (with k = 1, two per step: inherent to handing velocity Verlet a new state every
    step, not a property of the ABI; k = 10 is how a driver that wants the trajectory on the host would
    call it)."""
    N = sysd["N"]
    pos = torch.from_numpy(state[0].copy()).pin_memory()
    vel = torch.from_numpy(state[1].copy()).pin_memory()
    s = b.Sim(N, sysd["L"], rc=sysd["rc"], eps=sysd["eps"], sigma=sysd["sigma"], dt=sysd["dt"],
              shifted=sysd["shifted"])
    h = s.h
    for it in range(calls + 2):
        if it == 2:
            torch.cuda.synchronize()
            t0 = time.perf_counter()
        b.md_set_state(h, pos, vel)
        b.md_step(h, k, algo)
        b.md_get_state(h, pos, vel)
        b.md_get_energies(h)
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / (calls * k)
    s.close()
    return dict(ms_per_step=dt * 1e3, h2d=2 * N * 12 / k, d2h=(2 * N * 12 + 24) / k, k=k)


def fp32_peak_tflops(peaks, n_sms):
    return n_sms * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12


def allpairs_roofline(N, rho, rc, t_filter_ms, t_eval_ms, peaks, n_sms):
    """Algorithmic flops (8 per ordered pair test + 19 per in-range pair) over the time of the
    two kernels that do that work: k_allpairs_filter (every pair test) + k_allpairs_eval (the in-range pairs,
    FP64).  executed_frac counts what the filter really issues: 3 FMA = 6 flop per test."""
    pairs = float(N) * (N - 1)
    inrange = N * NBR_PER_ATOM(rho, rc)
    flops = pairs * FLOP_PER_PAIR_TEST + inrange * FLOP_PER_INRANGE
    peak = fp32_peak_tflops(peaks, n_sms)
    t = (t_filter_ms + t_eval_ms) * 1e-3
    ach = flops / t / 1e12
    return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
            "kernel": "all-pairs force: k_allpairs_filter + k_allpairs_eval",
            "kernel_ms": t_filter_ms + t_eval_ms, "filter_kernel_ms": t_filter_ms, "eval_kernel_ms": t_eval_ms,
            "frac_filter_kernel_alone": (pairs * FLOP_PER_PAIR_TEST / (t_filter_ms * 1e-3) / 1e12) / peak,
            "executed_frac": ((pairs * 6.0 + inrange * FLOP_PER_INRANGE) / t / 1e12) / peak,
            "pair_tests_per_s": pairs / (t_filter_ms * 1e-3),
            "peak_source": "derived: SMs x 128 FP32 lanes x 2 x clocks.max.sm (DESIGN.md section 8)"}


def cell_roofline(N, rho, rc, ncell, t_kernel_ms, peaks, n_sms, t_noenergy_ms=None):
    """t_kernel_ms: the force kernel WITH PE and the virial (the launch md_step(1) makes; 19 flop per in-range pair).
    t_noenergy_ms: the force-only launch of the interior steps of md_step(K), credited 13 flop per in-range pair."""
    cand = 27.0 * N / ncell ** 3 * N                    # ordered candidate pairs per launch
    inr = N * NBR_PER_ATOM(rho, rc)
    flops = cand * FLOP_PER_PAIR_TEST + inr * FLOP_PER_INRANGE
    peak = fp32_peak_tflops(peaks, n_sms)
    ach = flops / (t_kernel_ms * 1e-3) / 1e12
    extra = {}
    if t_noenergy_ms:
        a2 = (cand * FLOP_PER_PAIR_TEST + inr * FLOP_PER_INRANGE_NO_ENERGY) / (t_noenergy_ms * 1e-3) / 1e12
        extra = {"force_only_kernel_ms": t_noenergy_ms, "force_only_frac": a2 / peak}
    return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
            "kernel": "cell-list force with PE and virial: k_fc2<ENERGY=1>", "kernel_ms": t_kernel_ms, "ncell": ncell, **extra,
            "peak_source": "derived: SMs x 128 FP32 lanes x 2 x clocks.max.sm (DESIGN.md section 8)",
            "candidate_tests_per_s": cand / (t_kernel_ms * 1e-3),
            "pair_interactions_per_s": 0.5 * N * NBR_PER_ATOM(rho, rc) / (t_kernel_ms * 1e-3)}


# Algorithmic HBM bytes per atom and step of the streaming kernels of the cell path:
# kick/drift/histogram reads pos, vel, frc (48) and writes pos, vel with the rank in vel.w (32); the scatter
# reads pos, vel (32) and writes pos, vel, cell-local positions (48).  The scan moves 8 B per cell (neglected).
CELL_STREAM_BYTES_PER_ATOM = 160.0


def stream_roofline(N, phases_ms, peaks):
    """Integration + build kernels of the cell path against the measured HBM copy rate.  For systems
    that fit L2 (N <= 256,000) the achieved figure can exceed what HBM alone would allow."""
    t = (phases_ms["integrate"] + phases_ms["build"]) * 1e-3
    if t <= 0:
        return None
    gbs = CELL_STREAM_BYTES_PER_ATOM * N / t / 1e9
    return {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"],
            "traffic": None, "kernel": "kick/drift/histogram + scan + scatter", "bytes_per_atom": CELL_STREAM_BYTES_PER_ATOM}


def verlet_roofline(N, rho, rc, skin, t_kernel_ms, peaks, n_sms):
    """List evaluation kernel: one distance test (8 flop) per list entry, ~19 flop per in-range pair."""
    entries = N * NBR_PER_ATOM(rho, rc + skin)
    flops = entries * FLOP_PER_PAIR_TEST + N * NBR_PER_ATOM(rho, rc) * FLOP_PER_INRANGE
    peak = fp32_peak_tflops(peaks, n_sms)
    ach = flops / (t_kernel_ms * 1e-3) / 1e12
    return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
            "kernel": "neighbour-list force: k_vl_force", "kernel_ms": t_kernel_ms,
            "list_entries_per_s": entries / (t_kernel_ms * 1e-3)}


def bench_rand48(b, torch, steps, peaks, with_cpu):
    """Config 5: 65536 streams x 4096 draws and one stream of 2^28 draws, uint32 and double: device buffers
    (value), host buffers through the same C-ABI call (e2e), and the oracle's sequential 64-bit LCG on one
    host core ("a self-written CPU version using 64-bit arithmetics")."""
    res = {}
    seeds_h = wl.stream_seeds(wl.MASTER_SEED, wl.C5_NSTREAMS)
    seeds0 = torch.from_numpy(seeds_h.astype(np.int64)).cuda()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for name, ns, nd in (("streams_65536x4096", wl.C5_NSTREAMS, wl.C5_NDRAWS), ("single_2p28", 1, wl.C5_SINGLE_NDRAWS)):
        for kind, tdt, esz in ((0, torch.int32, 4), (2, torch.float64, 8)):
            out = torch.empty(ns * nd, dtype=tdt, device="cuda")     # 1.07 / 2.15 GB > L2
            seeds = seeds0[:ns].clone()
            for _ in range(2):
                b.rand48_fill(seeds.data_ptr(), ns, nd, kind, out.data_ptr())
            e0.record()
            for _ in range(steps):
                b.rand48_fill(seeds.data_ptr(), ns, nd, kind, out.data_ptr())
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            gbs = ns * nd * esz / (ms * 1e-3) / 1e9
            key = "%s_%s" % (name, "u32" if kind == 0 else "f64")
            res[key] = {
                "draws_per_s": ns * nd / (ms * 1e-3), "ms": ms, "store_GBps": gbs,
                "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": gbs / peaks["hbm_gbs"], "traffic": None, "kernel": "k_rand48_fill"}}
            del out
            # e2e: host seeds in, host (pinned) output back, through the same call
            hout = torch.empty(ns * nd, dtype=tdt).pin_memory()
            hseeds = torch.from_numpy(seeds_h[:ns].astype(np.int64).copy()).pin_memory()
            b.rand48_fill(hseeds.data_ptr(), ns, nd, kind, hout.data_ptr())
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(2):
                b.rand48_fill(hseeds.data_ptr(), ns, nd, kind, hout.data_ptr())
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) / 2
            res[key]["e2e"] = {"value": ns * nd / dt, "unit": "draws/s", "h2d_bytes_per_step": ns * 8,
                               "d2h_bytes_per_step": ns * nd * esz + ns * 8, "ms": dt * 1e3}
            del hout
            if with_cpu:
                import oracle
                sample_ns = ns
                sample_nd = nd
                t0 = time.perf_counter()
                oracle.rand48_fill(seeds_h[:sample_ns], sample_nd, kind)
                dt = time.perf_counter() - t0
                res[key]["cpu_baseline"] = {"value": sample_ns * sample_nd / dt, "unit": "draws/s", "cores": 1,
                                            "kind": "oracle", "sample": "%d streams x %d draws, sequential LCG, %.2f s"
                                            % (sample_ns, sample_nd, dt)}
    return res


def product_velocities(b, pos, L):
    """velocity_source for workloads.md_system on the product side: md_init_velocities (Maxwell-Boltzmann
    from one rand48 stream, generated on the device), read back."""
    def src(N, T, seed48):
        with b.Sim(N, L) as s:
            s.set_state(pos, np.zeros_like(pos))
            s.init_velocities(T, seed48)
            return s.get_state()[1]
    return src


def make_system(b, name):
    cfg = wl.CONFIGS[name]
    pos, L = wl.fcc_positions(cfg["n"], cfg["rho"])
    return wl.md_system(name, product_velocities(b, pos, L))


def cpu_baseline_md(sysd, state, algo, budget_steps, threads):
    """The oracle as it stands, timed on this box's host cores on a bounded sample: a few velocity-Verlet
    steps from the melted state the GPU was timed on.  algo 0: the O(N^2) half loop (no OpenMP pragma: one
    thread); algo 1: the linked-cell full-shell loop (OpenMP over atoms)."""
    import oracle
    oracle.set_threads(threads)
    pos, vel = state[0].astype(np.float64), state[1].astype(np.float64)
    t0 = time.perf_counter()
    oracle.verlet_run(pos, vel, sysd["L"], budget_steps, rc=sysd["rc"], eps=sysd["eps"], sigma=sysd["sigma"],
                      dt=sysd["dt"], mode=sysd["shifted"], algo=algo)
    dt = time.perf_counter() - t0
    evals = budget_steps + 1                        # verlet_run evaluates forces once at entry
    return {"value": sysd["N"] * evals / dt, "unit": "atom-steps/s", "cores": threads, "kind": "oracle",
            "sample": "%d force evaluations (%d velocity-Verlet steps) of the same melted N=%d system, %s loop, %.1f s"
                      % (evals, budget_steps, sysd["N"], "all-pairs" if algo == 0 else "linked-cell", dt)}


def bench_extras(b, torch, sysd, steps):
    """Throughput of the SURVEY 8(f) extensions on the config-3 system: md_init_velocities and md_step with the
    Andersen thermostat on (rand48 consumed in registers), skin cells, and the Yukawa pair potential."""
    N = sysd["N"]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    out = {}
    with b.Sim(N, sysd["L"]) as s:
        s.set_state(sysd["pos"], sysd["vel"])
        s.init_velocities(1.0, 12345)
        e0.record()
        for _ in range(5):
            s.init_velocities(1.0, 12345)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 5
        out["md_init_velocities"] = {"N": N, "ms": ms, "atoms_per_s": N / (ms * 1e-3), "draws_per_s": 6 * N / (ms * 1e-3)}
        s.set_state(sysd["pos"], sysd["vel"])
        s.option("andersen_T", 1.0)
        s.option("andersen_seed", 777)
        s.option("andersen_nu", 10.0)
        s.step(sysd["steps"], 1)
        e0.record()
        s.step(steps, 1)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        out["md_step_andersen_cell"] = {"N": N, "ms_per_step": ms, "atom_steps_per_s": N / (ms * 1e-3),
                                        "note": "nu dt = 0.05; every atom skips ahead to its 7 draws of the step (rand48 consumed in registers)"}
    # (f2) skin cells: the same system with cells of side >= rc + 0.3 re-sorted on the device's decision
    with b.Sim(N, sysd["L"]) as s:
        s.option("cell_skin", 0.3)
        s.set_state(sysd["pos"], sysd["vel"])
        s.step(sysd["steps"], 1)
        nb0, ns0 = s.stat("vl_builds"), s.stat("vl_steps")
        e0.record()
        s.step(2 * steps, 1)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / (2 * steps)
        out["md_step_skin_cells"] = {"N": N, "ms_per_step": ms, "atom_steps_per_s": N / (ms * 1e-3), "skin": 0.3,
                                     "resorts_per_100_steps": 100.0 * (s.stat("vl_builds") - nb0) / max(1.0, s.stat("vl_steps") - ns0)}
    # neighbour lists with Newton's third law (option "vl_half"): every pair once, reactions through reductions
    with b.Sim(N, sysd["L"]) as s:
        s.option("vl_half", 1)
        s.set_state(sysd["pos"], sysd["vel"])
        s.step(sysd["steps"], 2)
        e0.record()
        s.step(2 * steps, 2)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / (2 * steps)
        out["md_step_verlet_half_lists"] = {"N": N, "ms_per_step": ms, "atom_steps_per_s": N / (ms * 1e-3)}
    # (f4) second pair potential: screened Coulomb (Yukawa), every in-range pair in FP64, on the three paths
    for label, algo in (("cell", 1), ("verlet", 2)):
        with b.Sim(N, sysd["L"]) as s:
            s.potential(b.MD_POT_YUKAWA, 6.0, 1.2)
            s.set_state(sysd["pos"], sysd["vel"])
            s.step(100, algo)
            e0.record()
            s.step(steps, algo)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            out["md_step_yukawa_" + label] = {"N": N, "ms_per_step": ms, "atom_steps_per_s": N / (ms * 1e-3),
                                              "potential": "U = 6 exp(-1.2 r) / r, rc = 2.5, energy-shifted"}
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_0709_3225_b200 import binding as b
    side = torch.cuda.Stream()                       # the library runs on PyTorch's current stream
    with torch.cuda.stream(side):
        line = measure(args, b, torch, dist, rank, local_rank, world)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


def measure(args, b, torch, dist, rank, local_rank, world):
    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(local_rank)
    n_sms = props.multi_processor_count
    ncores = os.cpu_count() or 1
    name = args.workload
    cfg = wl.CONFIGS[name]
    sysd = make_system(b, name)
    algo = cfg["algo"]
    if args.algo == "verlet":
        algo = b.MD_VERLET
    buf = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")
    steps, warmup = args.steps, max(3, args.warmup)
    opts = {kv.split("=", 1)[0]: float(kv.split("=", 1)[1]) for kv in args.opt}

    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    with ClockSampler(local_rank) as clk:
        r = time_md(b, torch, sysd, algo, steps, warmup, True, buf, options=opts)
    ms = r["flushed_ms"]
    e2e = time_md_e2e(b, torch, sysd, r["melted"], algo, min(steps, 50), 1)
    e2e10 = time_md_e2e(b, torch, sysd, r["melted"], algo, max(2, min(steps, 50) // 5), 10)
    if world > 1:
        ms, r["steady_ms"], e2e["ms_per_step"], e2e10["ms_per_step"] = max_over_ranks(
            [ms, r["steady_ms"], e2e["ms_per_step"], e2e10["ms_per_step"]], dist, "cuda")
    N = sysd["N"]
    value = whole_job_value(N, world, ms)
    if algo == 0:
        roof = allpairs_roofline(N, cfg["rho"], wl.RC, r["t_force_kernel_ms"], r["t_force2_kernel_ms"], peaks, n_sms)
    elif algo == 2:
        roof = verlet_roofline(N, cfg["rho"], wl.RC, 0.3, r["t_force_kernel_ms"], peaks, n_sms)
    else:
        roof = cell_roofline(N, cfg["rho"], wl.RC, r["ncell"], r["t_force_energy_kernel_ms"], peaks, n_sms,
                             t_noenergy_ms=r["t_force_kernel_ms"])
    roof["traffic"], roof["traffic_source"] = ncu_traffic(name if algo != 2 else name + "_verlet")
    stream_roof = stream_roofline(N, r["phases_ms"], peaks) if algo == 1 else None
    roof["kernel_share_of_step"] = roof["kernel_ms"] / max(1e-12, sum((r["phases_energy_ms"] if algo == 1 else r["phases_ms"]).values()))
    # the derived "alu" peak checked live: the library's register-only FFMA-chain kernel (csrc/probe.cu)
    chain_tf, chain_ms = b.md_probe_fp32_peak()
    roof["peak_check"] = {"ffma_chain_tflops": chain_tf, "frac_of_derived_peak": chain_tf / fp32_peak_tflops(peaks, n_sms),
                          "kernel": "k_probe_ffma, best of 3 launches, CUDA events", "kernel_ms": chain_ms}

    def e2e_obj(e):
        return {"value": world * N / (e["ms_per_step"] * 1e-3), "unit": "atom-steps/s",
                "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"], "ms_per_step": e["ms_per_step"],
                "steps_per_call": e["k"], "force_evaluations_per_step": (e["k"] + 1.0) / e["k"]}

    line = {
        "metric": "LJ MD atom-steps/s", "value": value, "unit": "atom-steps/s", "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (state, distance tests, far pair terms), f64 (close or all in-range pair terms, energy sums)",
        "data": "synthetic",
        "config": {"workload": name, "N": N, "rho": cfg["rho"], "T": cfg["T"], "rc": wl.RC, "dt": wl.DT,
                   "algo": ("allpairs", "cell", "verlet")[algo], "shifted": wl.SHIFTED,
                   "state": "fcc lattice + md_init_velocities, advanced %d steps (the config's length) before timing" % cfg["steps"],
                   "l2": "flushed between steps (256 MB read-modify-write); steady_state is the unflushed md_step(K) loop",
                   "stream": "PyTorch side stream, PyTorch caching allocator", "options": opts,
                   "parallelism": "replicas x%d" % world if world > 1 else "single GPU"},
        "steady_state": {"ms_per_step": r["steady_ms"], "value": world * N / (r["steady_ms"] * 1e-3),
                         "note": "md_step(K) back to back, L2 not flushed; PE and the virial are evaluated on the last step of a call only"},
        "energy_every_step": {"ms_per_step": r["every_step_energy_ms"], "value": world * N / (r["every_step_energy_ms"] * 1e-3),
                              "note": "md_step(1) K times, L2 not flushed: KE, PE and the virial evaluated and reduced on every step",
                              "phases_ms": r["phases_energy_ms"]},
        "repeats": {"ms_per_step": r["flushed_reps"], "best": min(r["flushed_reps"]), "median": float(np.median(r["flushed_reps"])),
                    "note": "three repetitions of the K flushed steps on this rank; `value` is the first"},
        "phases_ms": r["phases_ms"],
        "roofline": roof,
        "roofline_streaming_kernels": stream_roof,
        "e2e": e2e_obj(e2e),
        "e2e_10_steps_per_call": e2e_obj(e2e10),
        "gpu_launches": int(round(r["launches_per_step"] * steps)),
        "clocks": clk.summary(),
        "peaks": peaks,
    }
    if algo == 2:
        line["list_builds_per_100_steps"] = r["vl_builds_per_100"]
    if rank == 0 and world == 1:
        if algo == 0:
            nb = 2 if N >= 20000 else 20
            line["cpu_baseline"] = cpu_baseline_md(sysd, r["melted"], 0, nb, 1)
            if N >= 4000:       # the same system through the oracle's OpenMP loop (linked cells) on all cores
                line["cpu_baseline_all_cores"] = cpu_baseline_md(sysd, r["melted"], 1, 10, ncores)
        else:
            line["cpu_baseline"] = cpu_baseline_md(sysd, r["melted"], 1, 3 if N <= 300000 else 1, ncores)
    if rank == 0 and world == 1 and not args.no_others:
        others = {}
        for oname in ("c1_allpairs_500", "c3_cell_256k", "c4a_cell_2048k", "c4b_cell_2048k_rho03"):
            if oname == name:
                continue
            ocfg = wl.CONFIGS[oname]
            osys = make_system(b, oname)
            oN = osys["N"]
            osteps = 200 if ocfg["n"] <= 5 else (20 if ocfg["n"] >= 80 else 50)
            rr = time_md(b, torch, osys, ocfg["algo"], osteps, 5, False, buf)
            ent = {"N": oN, "atom_steps_per_s": oN / (rr["steady_ms"] * 1e-3),
                   "ms_per_step": rr["steady_ms"], "phases_ms": rr["phases_ms"],
                   "energy_every_step": {"ms_per_step": rr["every_step_energy_ms"],
                                         "atom_steps_per_s": oN / (rr["every_step_energy_ms"] * 1e-3),
                                         "phases_ms": rr["phases_energy_ms"]},
                   "force_kernel_ms": rr["t_force_kernel_ms"], "launches_per_step": rr["launches_per_step"]}
            if ocfg["algo"] == 1:
                ent["roofline"] = cell_roofline(oN, ocfg["rho"], wl.RC, rr["ncell"], rr["t_force_energy_kernel_ms"], peaks, n_sms,
                                                t_noenergy_ms=rr["t_force_kernel_ms"])
                # the cell-list half of the metric, compact, inside a key the driver's record keeps
                line["roofline"].setdefault("cell_list", {})[oname] = {
                    "N": oN, "atom_steps_per_s": ent["atom_steps_per_s"],
                    "atom_steps_per_s_energy_every_step": ent["energy_every_step"]["atom_steps_per_s"],
                    "force_kernel_ms": ent["roofline"]["kernel_ms"], "frac": ent["roofline"]["frac"],
                    "target_atom_steps_per_s": 1e10 if oN >= 256000 else None}
                ent["roofline"]["traffic"], ent["roofline"]["traffic_source"] = ncu_traffic(oname)
                ent["roofline_streaming_kernels"] = stream_roofline(oN, rr["phases_ms"], peaks)
                ent["cpu_baseline"] = cpu_baseline_md(osys, rr["melted"], 1, 3 if oN <= 300000 else 1, ncores)
            else:
                ent["roofline"] = allpairs_roofline(oN, ocfg["rho"], wl.RC, rr["t_force_kernel_ms"],
                                                    rr["t_force2_kernel_ms"], peaks, n_sms)
                ent["cpu_baseline"] = cpu_baseline_md(osys, rr["melted"], 0, 20, 1)
            others[oname] = ent
            if ocfg["algo"] == 1:
                # the same system through the neighbour-list path (algo = MD_VERLET):
                # an extension beyond the named configs, reported beside them
                rv = time_md(b, torch, osys, b.MD_VERLET, max(osteps, 100), 5, False, buf)
                vr = verlet_roofline(oN, ocfg["rho"], wl.RC, 0.3, rv["t_force_kernel_ms"], peaks, n_sms)
                vr["traffic"], vr["traffic_source"] = ncu_traffic(oname + "_verlet")
                others[oname + "_verlet"] = {"N": oN, "atom_steps_per_s": oN / (rv["steady_ms"] * 1e-3),
                                             "ms_per_step": rv["steady_ms"], "phases_ms": rv["phases_ms"],
                                             "force_kernel_ms": rv["t_force_kernel_ms"],
                                             "launches_per_step": rv["launches_per_step"],
                                             "list_builds_per_100_steps": rv.get("vl_builds_per_100"),
                                             "roofline": vr}
            if oname == "c3_cell_256k":
                others["extensions_c3"] = bench_extras(b, torch, osys, osteps)
        others["c5_rand48"] = bench_rand48(b, torch, 5, peaks, True)
        line["others"] = others
    return line


# ----------------------------------------------------------------------- reference arm
def run_reference(args):
    """The oracle as it stands on the host cores, same config/metric (bounded sample per step)."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    import oracle
    name = args.workload
    cfg = wl.CONFIGS[name]

    sysd = wl.md_system(name, lambda N_, T_, seed48: oracle.mb_velocities(N_, T_, seed48)[0])
    algo, N = cfg["algo"], sysd["N"]
    threads = (os.cpu_count() or 1) if algo == 1 else 1
    oracle.set_threads(threads)
    pos, vel = sysd["pos"].astype(np.float64), sysd["vel"].astype(np.float64)
    steps, warmup = max(1, min(args.steps, 3)), min(args.warmup, 1)
    pos, vel, _, _ = oracle.verlet_run(pos, vel, sysd["L"], warmup, algo=algo) if warmup else (pos, vel, None, None)
    t0 = time.perf_counter()
    oracle.verlet_run(pos, vel, sysd["L"], steps, algo=algo)
    dt = time.perf_counter() - t0
    evals = steps + 1
    value = N * evals / dt
    line = {"impl": "reference", "metric": "LJ MD atom-steps/s", "value": value, "unit": "atom-steps/s",
            "n_gpus": world, "steps": steps, "warmup": warmup, "ms_per_step": dt / evals * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "N": N, "rho": cfg["rho"], "T": cfg["T"], "rc": wl.RC, "dt": wl.DT,
                       "algo": "allpairs" if algo == 0 else "cell", "shifted": wl.SHIFTED},
            "cpu_baseline": {"value": value, "unit": "atom-steps/s", "kind": "oracle", "cores": threads,
                             "sample": "%d force evaluations of the same N=%d system (steps clamped to 3 so the run "
                                       "ends within minutes)" % (evals, N)},
            "e2e": {"value": value, "unit": "atom-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2_allpairs_32k", choices=sorted(wl.CONFIGS))
    ap.add_argument("--algo", default=None, choices=["verlet"],
                    help="run the workload's system through the neighbour-list path instead of its named path")
    ap.add_argument("--no-others", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="md_set_option for the headline workload, e.g. --opt cell_kernel=3 (repeatable)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
