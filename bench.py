#!/usr/bin/env python
"""bench.py -- atom-timesteps/s of the MD hot path (force + neighbor + integrate) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg C] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is ONE PASS OF THE WHOLE HOT PATH over one batch of synthetic input: the workload's full
``md_run`` (its ``nsteps`` velocity-Verlet time steps: cell binning + counting sort + reorder, Verlet
list build, displacement-triggered rebuilds, pair forces, integration) from the seeded initial state.
The default workload is BASELINE.json config 5 (LJ liquid, 4,000,000 atoms, mixed precision, 200 time
steps), the one HBM-scale configuration;
``--cfg`` selects another.  ``per_config`` in the JSON line carries the other four configs.

value     whole-job atom-timesteps/s, inputs already resident in HBM (device buffers handed to
          md_set_positions / md_set_velocities), CUDA events on the library's stream, max over ranks
e2e       the same through the C ABI with HOST (pinned) buffers: H2D of x and v, md_run, D2H of the
          final positions and the kinetic energy, every step, inside the timed region
roofline  dominant kernel = the pair-force tile kernel; SURVEY.md 8(d)'s algorithmic bytes per launch / its
          mean launch duration (CUDA events on the library's stream inside md_run, sampled steps of the
          timed region); traffic = measured DRAM bytes per launch from the committed ncu summary profiles/r02_ncu_full_force_cfgN.md
cpu_baseline   the oracle (oracle/md_oracle.c, as it stands) on the host cores, bounded sample

N > 1: independent replicas, one per GPU, no data-path collective ("scaling": "weak").
``--impl reference`` times the oracle alone (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1009_4330_b200 import dist as mdist          # noqa: E402
from paper_1009_4330_b200 import workloads as wl        # noqa: E402
from paper_1009_4330_b200 import ncu_summary            # noqa: E402  (text parsing only)

METRIC = "atom-timesteps/s (force+neighbor+integrate)"
UNIT = "atom-timesteps/s"
L2_BYTES = 126 * 1024 * 1024

# CPU-baseline samples: (unit cells per edge, time steps) -- a bounded sample of the same workload
# (same lattice, potential, seeds, rebuild rule; atom-steps/s is intensive), ~10-30 s on 8 cores.
CPU_SAMPLE = {1: (10, 100), 2: (20, 300), 3: (20, 20), 4: (30, 40), 5: (50, 20)}


def measured_peaks() -> tuple[float, str]:
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append((time.perf_counter(), line.strip()))
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        inside = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in inside:
            c = [q.strip() for q in r.split(",")]
            try:
                sm.append(float(c[0])); smax.append(float(c[1])); power.append(float(c[2]))
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(c) > 4 + k and c[4 + k].lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "power_w_max": float(max(power)), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------
# algorithmic bytes of the dominant kernel: the pair-force tile kernel
# ---------------------------------------------------------------------------------------------------------
def survey_force_bytes(natoms: int, mean_neighbors: float, style: int) -> float:
    """ALGORITHMIC bytes of one force evaluation as SURVEY.md §8(d) charges them: per atom the
    neighbor-index stream at 4 B per full-list entry, numneigh (4 B), the atom's own fp64 position (24 B) and
    the fp64 force store (24 B); gathered neighbor positions are charged to cache, not HBM (the optimistic
    ceiling of §8(d), which the measured DRAM traffic confirms).  EAM runs two list passes: indices +
    numneigh + own position twice, plus the rho / F' stores (16 B) and the F' read (8 B)."""
    per_atom = 4.0 * mean_neighbors + 4 + 24 + 24
    if style == wl.PAIR_EAM:
        per_atom = 2 * (4.0 * mean_neighbors + 4 + 24) + 16 + 8 + 24
    return per_atom * natoms


# SURVEY.md 8(d) "optimistic ceilings": algorithmic HBM bytes of ONE atom-timestep of the whole path (index stream at
# 4 B per list entry + per-atom state + fused integration; gathers charged to cache; list build excluded)
PATH_BYTES = {1: 540.0, 2: 540.0, 3: 2330.0, 4: 880.0, 5: 540.0}
PROFILE_MD = "profiles/r02_ncu_full_force_cfg%d.md"     # written by `python -m paper_1009_4330_b200.ncu_summary full ...`


def roofline_block(cfg: int, w, st: dict, value: float, hbm_gbs: float, peak_src: str) -> dict:
    """The `roofline` object of one configuration: dominant kernel = the pair-force kernel (both passes for EAM)."""
    nf = max(1, st["nforce_sampled"])
    ms_force = st["ms_force_sampled"] / nf
    sbytes = survey_force_bytes(w.natoms, st["mean_neighbors"], w.style)
    lbytes = layout_force_bytes(w.natoms, st["mean_row"], w.style)
    achieved = sbytes / (ms_force * 1e-3) / 1e9 if ms_force > 0 else 0.0
    persistent = w.precision == wl.PREC_MIXED
    r = {
        "bound": "hbm", "achieved": achieved, "peak": hbm_gbs, "unit": "GB/s", "frac": achieved / hbm_gbs,
        "frac_of_nominal_8TBps": achieved / 8000.0, "traffic": None, "peak_source": peak_src,
        "kernel": "%s<%s,K=%d>" % ("k_tile_force_p" if persistent else "k_tile_force", "LJ" if w.style == wl.PAIR_LJ else "EAM density+force",
                                   st["lanes_per_atom"]),
        "algorithmic_bytes_per_launch": sbytes,
        "algorithmic_bytes_definition": "SURVEY.md 8(d): (4 B x exact list entries + 52 B) per atom (EAM: two passes), DESIGN.md 6",
        "own_layout_bytes_per_launch": lbytes,
        "ms_per_launch": ms_force, "launches_sampled": st["nforce_sampled"],
        "path_bytes_per_atom_step": PATH_BYTES[cfg],
        "path_frac": value / (hbm_gbs * 1e9 / PATH_BYTES[cfg]),
        "note": "frac is SURVEY 8(d)'s ALGORITHMIC-bytes ceiling over the measured HBM copy rate, not the share of the binding "
                "resource: the kernel moves fewer bytes than that (2-byte slot codes, one row per pair of atoms: "
                "own_layout_bytes_per_launch) and ncu shows it bound by the FP32 (FMA) pipe and latency, DRAM at ~30 % "
                "(profiles/, DESIGN.md 6)",
    }
    if w.style == wl.PAIR_EAM and ms_force > 0:
        p1 = st["ms_force_pass1_sampled"] / nf
        r["ms_pass1_density"] = p1
        r["ms_pass2_force"] = ms_force - p1
    t = ncu_summary.traffic(os.path.join(ROOT, PROFILE_MD % cfg), sections=2 if w.style == wl.PAIR_EAM else 1)
    if t is not None:
        r["traffic"] = t
        r["traffic_source"] = (PROFILE_MD % cfg) + " (ncu --set full: dram__bytes_read.sum + dram__bytes_write.sum; both passes summed for EAM)"
    return r


def layout_force_bytes(natoms: int, mean_neighbors: float, style: int) -> float:
    """The same with THIS library's list layout (16-bit tile-local slot codes: 2 B per entry) -- what the
    kernel itself must move; reported beside the SURVEY figure, never as ``achieved``."""
    per_atom = 2.0 * (0.5 * mean_neighbors) + 2 + 24 + 24        # mean_neighbors here = entries per stored PAIR row (md_stats.mean_row)
    if style == wl.PAIR_EAM:
        per_atom = 2 * (2.0 * (0.5 * mean_neighbors) + 2 + 24) + 16 + 8 + 24
    return per_atom * natoms


# ---------------------------------------------------------------------------------------------------------
# the reference arm / cpu_baseline: the oracle on the host cores
# ---------------------------------------------------------------------------------------------------------
def oracle_sample(cfg: int, reps: int = 1, warm: int = 0, shrink: int = 1) -> dict:
    """Times oracle.run_nve (cell grid + Verlet list + rebuild rule, fp64, OpenMP over atoms) on a bounded
    sample of config ``cfg``.  Returns atom-timesteps/s and what the sample was."""
    import oracle
    n, steps = CPU_SAMPLE[cfg]
    steps = max(2, steps // max(1, shrink))
    w = wl.make(cfg, n_override=n)
    m = np.full(w.natoms, w.mass[0])
    cores = oracle.max_threads()
    times = []
    for it in range(warm + reps):
        t0 = time.perf_counter()
        oracle.run_nve(w.x, w.v, w.box, m, w.style, w.params, w.rc, w.skin, w.dt, steps, ftm2v=w.ftm2v, mvv2e=w.mvv2e)
        t1 = time.perf_counter()
        if it >= warm:
            times.append(t1 - t0)
    full = wl._TABLE[cfg][2]
    sample = ("config %d lattice cut to %d^3 fcc cells (%d atoms; full size %d^3), first %d time steps, same potential, "
              "seed, skin and rebuild rule; oracle.run_nve fp64" % (cfg, n, w.natoms, full, steps))
    return {"value": w.natoms * steps * len(times) / sum(times), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": sample, "seconds": sum(times), "natoms": w.natoms, "steps": steps, "times": times}


def run_reference(args, rk) -> None:
    if not rk.is_root:
        return
    w_meta = wl._TABLE[args.cfg]
    # keep the whole --steps K --warmup W run within a few minutes: fewer time steps per sample when K is large
    r = oracle_sample(args.cfg, reps=max(1, args.steps), warm=min(args.warmup, 1),
                      shrink=math.ceil((args.steps + min(args.warmup, 1)) / 6))
    ms = 1e3 * r["seconds"] / max(1, args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg%d: %s" % (args.cfg, w_meta[0]), "sample": r["sample"]},
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------
def _flush_l2(torch, scratch):
    scratch.add_(1)      # writes 2 x L2 bytes on the same stream, outside the event-timed region


def time_workload(torch, md, w, stream, steps: int, warmup: int, kernel: int, list_kind: int, host_io: bool, options: dict | None = None):
    """Runs ``warmup`` + ``steps`` passes of the whole hot path for workload ``w``.  Returns per-pass
    device times (ms, CUDA events on ``stream``), the stats of the last pass and launches per pass."""
    N = w.natoms
    with torch.cuda.stream(stream):
        s = md.from_workload(w, kernel=kernel, list_kind=list_kind, stream=int(stream.cuda_stream), options=options)
        if host_io:
            x_in = torch.from_numpy(w.x).pin_memory(); v_in = torch.from_numpy(w.v).pin_memory()
            x_out = torch.empty((N, 3), dtype=torch.float64).pin_memory()
        else:
            x_in = torch.from_numpy(w.x).cuda(non_blocking=False); v_in = torch.from_numpy(w.v).cuda(non_blocking=False)
            x_out = None
        state_bytes = N * (24 * 6 + 16) + 2 * 80 * N
        scratch = torch.zeros(2 * L2_BYTES // 4, dtype=torch.int32, device="cuda") if state_bytes < 2 * L2_BYTES else None
        times, wall = [], []
        launches = 0
        st = None
        for it in range(warmup + steps):
            if scratch is not None:
                _flush_l2(torch, scratch)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            stream.synchronize()
            t0 = time.perf_counter()
            e0.record(stream)
            s.md_set_positions(x_in)
            s.md_set_velocities(v_in)
            s.md_run(w.nsteps, w.dt)
            if host_io:
                s.md_get_positions(x_out)
                ke = s.md_kinetic_energy()
            e1.record(stream)
            stream.synchronize()
            t1 = time.perf_counter()
            if it >= warmup:
                times.append(e0.elapsed_time(e1)); wall.append(1e3 * (t1 - t0))
                st = s.md_get_stats()
                # the library's own launches inside the timed region: md_run's, the two scatter kernels of
                # md_set_positions / md_set_velocities and, with host buffers, the gather + kinetic-energy kernels
                launches += st["launches_last_run"] + 2 + (2 if host_io else 0)
        if st is None:
            st = s.md_get_stats()
        s.close()
    return {"ms": times, "wall_ms": wall, "stats": st, "launches": launches, "flushed_l2": scratch is not None}


def run_ours(args, rk) -> None:
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    from paper_1009_4330_b200 import md            # fails loudly if libmd_b200.so is missing
    dev = rk.local_rank if rk.world > 1 else 0
    torch.cuda.set_device(dev)
    stream = torch.cuda.Stream()
    hbm_gbs, peak_src = measured_peaks()
    kernel = {"auto": md.MD_KERNEL_AUTO, "tpa": md.MD_KERNEL_TPA, "subwarp8": md.MD_KERNEL_SUBWARP, "warp": md.MD_KERNEL_WARP,
              "cell": md.MD_KERNEL_CELL, "subwarp4": md.MD_KERNEL_SUBWARP4, "subwarp2": md.MD_KERNEL_SUBWARP2}[args.kernel]
    list_kind = md.MD_LIST_HALF if args.half else md.MD_LIST_FULL

    w = wl.make(args.cfg, seed_offset=mdist.replica_seed_offset(rk))
    sampler = ClockSampler(dev)
    mdist.barrier(rk); torch.cuda.synchronize()
    if rk.is_root:
        sampler.start()
    t_region0 = time.perf_counter()
    options = {kv.split("=")[0]: int(kv.split("=")[1], 0) for kv in args.opt}
    dev_run = time_workload(torch, md, w, stream, args.steps, args.warmup, kernel, list_kind, host_io=False, options=options)
    torch.cuda.synchronize(); mdist.barrier(rk)
    t_region1 = time.perf_counter()
    clocks = sampler.stop(t_region0, t_region1) if rk.is_root else None

    units = float(w.natoms) * w.nsteps * args.steps
    value, tmax = mdist.aggregate_throughput(rk, units, sum(dev_run["ms"]) * 1e-3)

    mdist.barrier(rk)
    e2e_run = time_workload(torch, md, w, stream, args.steps, min(args.warmup, 3), kernel, list_kind, host_io=True, options=options)
    e2e_value, _ = mdist.aggregate_throughput(rk, units, sum(e2e_run["wall_ms"]) * 1e-3)
    launches = mdist.all_sum(rk, dev_run["launches"])

    st = dev_run["stats"]
    # roofline of the dominant kernel: sampled force launches inside the timed md_run
    nf = max(1, st["nforce_sampled"])
    ms_force = st["ms_force_sampled"] / nf
    nruns = max(1, args.steps)
    ms_per_step = 1e3 * tmax / nruns
    roofline = roofline_block(args.cfg, w, st, value, hbm_gbs, peak_src)
    roofline["share_of_step"] = {"force": ms_force * w.nsteps / (1e3 * tmax / nruns) if tmax > 0 else None,
                                 "build": st["ms_build_in_run"] / (1e3 * tmax / nruns) if tmax > 0 else None}
    # the resource ncu shows busiest: the FP32 pipe.  A list entry costs 14 packed f32x2 operations for the two atoms of its
    # row (3 sub, 3 for r^2, 5 for the LJ factor, 3 accumulate); a packed operation occupies the pipe for 2 cycles per warp
    # (measured: DESIGN.md 6), so one launch needs entries/32 x 28 pipe cycles on 148 x 4 sub-cores at full lanes
    passes = 2 if w.style == wl.PAIR_EAM else 1
    entries = passes * 0.5 * w.natoms * st["mean_row"]
    sm_clock = 1.965e9
    fp32_floor_ms = entries / 32.0 * 28.0 / (148 * 4) / sm_clock * 1e3
    roofline["fp32_pipe"] = {
        "list_entries_per_launch": entries, "packed_ops_per_entry": 14, "pipe_cycles_per_packed_warp_op": 2,
        "floor_ms_full_lanes": fp32_floor_ms, "frac_of_floor": fp32_floor_ms / ms_force if ms_force > 0 else None,
        "note": "LJ count; the floor assumes every lane of every warp busy (the rows of a warp differ in length: ~25 % of the "
                "lanes idle) and no prologue/epilogue; EAM bodies cost more per entry"}
    # the other heavy kernel: the list build, ALU-bound.  Tests = N x 27 x atoms per cell; peak = fp32
    # lanes x clock / 5 lane-instructions per test (3 packed sub/fma pairs = 3, compare, emit), 148 SMs x 128 lanes
    ncell = float(st["ncells"][0] * st["ncells"][1] * st["ncells"][2])
    tests = 27.0 * w.natoms * w.natoms / ncell
    ms_build = st["ms_build_in_run"] / max(1, st["nbuilds_in_run"])
    peak_tests = 148 * 128 * 1.965e9 / 5.0
    roofline_build = {
        "kernel": "k_build_list (+ bin, sort, reorder, tables: the whole build)", "bound": "alu",
        "achieved": tests / (ms_build * 1e-3) / 1e12 if ms_build > 0 else 0.0, "peak": peak_tests / 1e12, "unit": "T distance tests/s",
        "frac": tests / (ms_build * 1e-3) / peak_tests if ms_build > 0 else 0.0, "ms_per_build": ms_build,
        "builds_per_step": st["nbuilds_in_run"], "tests_per_build": tests,
        "note": "peak counts 5 fp32 lane-instructions per candidate test at 148 SMs x 128 lanes x 1.965 GHz; a cell holds "
                "~20 atoms for 32 lanes and each accepted entry costs a store and a pointer update (DESIGN.md 6)"}
    if not rk.is_root:
        return
    per_config = {}
    if args.all_configs and rk.world == 1:
        sampler2 = ClockSampler(dev)
        sampler2.start()
        t_pc0 = time.perf_counter()
        for c in (1, 2, 3, 4, 5):
            if c == args.cfg:
                continue
            wc = wl.make(c)
            r = time_workload(torch, md, wc, stream, 5, 3, md.MD_KERNEL_AUTO if args.kernel == "auto" else kernel,
                              list_kind if wc.style == wl.PAIR_LJ else md.MD_LIST_FULL, host_io=False)
            sc = r["stats"]
            vc = wc.natoms * wc.nsteps * len(r["ms"]) / (sum(r["ms"]) * 1e-3)
            per_config["cfg%d" % c] = {
                "workload": wc.name, "value": vc, "unit": UNIT, "passes_timed": len(r["ms"]),
                "ms_per_pass": sum(r["ms"]) / len(r["ms"]), "time_steps": wc.nsteps, "builds": sc["nbuilds_in_run"],
                "ms_per_build": sc["ms_build_in_run"] / max(1, sc["nbuilds_in_run"]),
                "variant": md.KERNEL_NAMES[sc["kernel_variant"]], "brick": sc["brick"], "tiles": sc["ntiles"],
                "mean_neighbors": sc["mean_neighbors"], "mean_row": sc["mean_row"],
                "roofline": roofline_block(c, wc, sc, vc, hbm_gbs, peak_src),
                "l2_flushed_between_passes": r["flushed_l2"]}
        # the synthetic two-species Buckingham + cutoff-Coulomb workload (110,592 ions, rc 8 A)
        w6 = wl.make(6)
        r = time_workload(torch, md, w6, stream, 5, 3, md.MD_KERNEL_AUTO if args.kernel == "auto" else kernel, md.MD_LIST_FULL, host_io=False)
        sc = r["stats"]
        msf = sc["ms_force_sampled"] / max(1, sc["nforce_sampled"])
        per_config["cfg6_buck_coul"] = {
            "workload": w6.name, "value": w6.natoms * w6.nsteps * len(r["ms"]) / (sum(r["ms"]) * 1e-3), "unit": UNIT, "passes_timed": len(r["ms"]),
            "ms_per_pass": sum(r["ms"]) / len(r["ms"]), "time_steps": w6.nsteps, "builds": sc["nbuilds_in_run"],
            "variant": md.KERNEL_NAMES[sc["kernel_variant"]], "brick": sc["brick"], "tiles": sc["ntiles"], "mean_neighbors": sc["mean_neighbors"],
            "force_ms_per_launch": msf,
            "force_GBps_survey_bytes": (4.0 * sc["mean_neighbors"] + 52) * w6.natoms / (msf * 1e-3) / 1e9 if msf > 0 else None,
            "note": "next-row workload (SURVEY 8(f)-2): parity in tests/test_gpu_parity.py::test_buck_coul_*; rc 8 A instead of the paper's 15 A (DESIGN.md, known limits)"}
        # SURVEY.md 8(f)-2, second half: cfg 4 with its potential given as 2001-point tables
        w7 = wl.make(7)
        r = time_workload(torch, md, w7, stream, 5, 3, md.MD_KERNEL_AUTO if args.kernel == "auto" else kernel, md.MD_LIST_FULL, host_io=False)
        sc = r["stats"]
        msf = sc["ms_force_sampled"] / max(1, sc["nforce_sampled"])
        per_config["cfg7_eam_tabulated"] = {
            "workload": w7.name, "value": w7.natoms * w7.nsteps * len(r["ms"]) / (sum(r["ms"]) * 1e-3), "unit": UNIT, "passes_timed": len(r["ms"]),
            "ms_per_pass": sum(r["ms"]) / len(r["ms"]), "time_steps": w7.nsteps, "builds": sc["nbuilds_in_run"],
            "variant": md.KERNEL_NAMES[sc["kernel_variant"]], "brick": sc["brick"], "tiles": sc["ntiles"], "mean_neighbors": sc["mean_neighbors"],
            "force_ms_per_launch": msf, "ms_pass1_density": sc["ms_force_pass1_sampled"] / max(1, sc["nforce_sampled"]),
            "note": "next-row workload (SURVEY 8(f)-2): parity in tests/test_gpu_parity.py::test_tabulated_eam_*; table lookups through the read-only path"}
        per_config["clocks"] = sampler2.stop(t_pc0, time.perf_counter())
        # the paper's comparison (Eq. 1): neighbor-list kernel against the direct cell-list kernel, and
        # the half list (Newton's third law, atomics), on the bench workload itself
        for name, kv, lk in (("cell_list", md.MD_KERNEL_CELL, md.MD_LIST_FULL), ("half_list_tpa", md.MD_KERNEL_TPA, md.MD_LIST_HALF)):
            if w.style != wl.PAIR_LJ:
                continue
            r = time_workload(torch, md, w, stream, 1, 1, kv, lk, host_io=False)
            sc = r["stats"]
            msf = sc["ms_force_sampled"] / max(1, sc["nforce_sampled"])
            per_config["cfg%d_%s" % (args.cfg, name)] = {
                "workload": w.name, "value": w.natoms * w.nsteps * len(r["ms"]) / (sum(r["ms"]) * 1e-3), "unit": UNIT,
                "ms_per_pass": sum(r["ms"]) / len(r["ms"]), "time_steps": w.nsteps, "builds": sc["nbuilds_in_run"],
                "variant": md.KERNEL_NAMES[sc["kernel_variant"]], "force_ms_per_launch": msf, "passes_timed": 1}
    cpu = oracle_sample(args.cfg) if (rk.world == 1 and not args.no_cpu_baseline) else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": rk.world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if w.precision == wl.PREC_MIXED else "f64",
        "dtype_detail": ("pair terms in f32 on tile-centred coordinates; per-atom force, energy and virial accumulators, positions, "
                         "velocities, integration and the list's distance decisions in f64 (BASELINE.json: fp32 compute / fp64 accumulate)")
                        if w.precision == wl.PREC_MIXED else "everything in f64", "data": "synthetic",
        "config": {"workload": "cfg%d: %s" % (args.cfg, w.name), "natoms": w.natoms, "time_steps_per_step": w.nsteps,
                   "rc": w.rc, "skin": w.skin, "dt": w.dt, "list": "half" if args.half else "full",
                   "variant": md.KERNEL_NAMES[st["kernel_variant"]], "mean_neighbors": st["mean_neighbors"],
                   "builds_per_step": st["nbuilds_in_run"], "tiles": st["ntiles"], "brick": st["brick"],
                   "parallelism": "replicas x%d (no collective)" % rk.world,
                   "launch": ("one fused kernel per time step (two for EAM) with programmatic dependent launch; rebuild flag read "
                              "once per batch of steps; rebuilds enqueued without waiting, replayed as a CUDA graph"
                              + ("; options " + ",".join(args.opt) if args.opt else "")),
                   "l2": "L2 flushed between passes (2x126 MB write)" if dev_run["flushed_l2"] else
                         "inputs larger than L2 (state + list >> 126 MB)"},
        "clocks": clocks, "roofline": roofline, "roofline_build": roofline_build,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * 24 * w.natoms, "d2h_bytes_per_step": 24 * w.natoms + 8,
                "ms_per_step": sum(e2e_run["wall_ms"]) / nruns},
        "gpu_launches": int(launches),
    }
    if cpu is not None:
        line["cpu_baseline"] = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
    if per_config:
        line["per_config"] = per_config
    print(json.dumps(line), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "tpa", "subwarp2", "subwarp4", "subwarp8", "warp", "cell"])
    ap.add_argument("--half", action="store_true", help="half list (Newton's third law, atomics); TPA only")
    ap.add_argument("--all-configs", dest="all_configs", action="store_true", default=True)
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="md_set_option tuning knob for the bench workload (include/md_b200.h), e.g. --opt tile_shape=0x334; repeatable")
    args = ap.parse_args()
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        if rank == 0:
            run_reference(args, mdist.Rank(0, 0, 1, None))
        return
    rk = mdist.init()
    try:
        run_ours(args, rk)
    finally:
        mdist.finalize(rk)


if __name__ == "__main__":
    main()
