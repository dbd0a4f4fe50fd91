"""Cutoff sweep of the force-kernel variants on B200 (the shape of PAPER.md Fig. 3 / Fig. 4).

    python -m paper_1009_4330_b200.sweep [--cells 20,40,100] [--rc 2.0,2.5,...,6.0] [--precision mixed,fp64] [--melt 60] > profiles/rNN_cutoff_sweep.md

For the LJ fluid of BASELINE.json (density 0.8442, T* = 1.44, skin 0.3 sigma; mixed precision and fp64) at
32,000, 256,000 and 4,000,000 atoms, and cutoffs from 2.0 to 6.0 sigma, it times one force evaluation (device time
of ``md_compute_forces``, CUDA events inside the library, best of ``--reps``) with every variant:
thread per row (K = 1), 2, 4 and 8 lanes per row, warp per row (the paper's BpA), direct cell list, and the
half list with atomic scatter, plus the list build, after ``--melt`` time steps so that the structure is
a liquid's.  Pure measurement on the library's public API; prints a markdown table.
"""
from __future__ import annotations

import argparse
import dataclasses
import sys

import numpy as np


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--cells", default="20,40,100", help="fcc unit cells per box edge (20 -> 32,000 atoms, 40 -> 256,000, 100 -> 4,000,000)")
    ap.add_argument("--precision", default="mixed,fp64")
    ap.add_argument("--rc", default="2.0,2.5,3.0,3.5,4.0,4.5,5.0,5.5,6.0")
    ap.add_argument("--melt", type=int, default=60)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--nsweep", default="", help="also: whole-path throughput against system size (the shape of Fig. 7, L182-192): "
                    "comma-separated fcc cells per edge, e.g. 6,8,10,14,20,28,40,56,80,100")
    ap.add_argument("--nsteps", type=int, default=200)
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device; the CUDA path has no CPU fallback")
    from . import md, workloads as wl

    variants = [("tpa", md.MD_KERNEL_TPA, md.MD_LIST_FULL), ("subwarp2", md.MD_KERNEL_SUBWARP2, md.MD_LIST_FULL),
                ("subwarp4", md.MD_KERNEL_SUBWARP4, md.MD_LIST_FULL),
                ("subwarp8", md.MD_KERNEL_SUBWARP, md.MD_LIST_FULL),
                ("warp", md.MD_KERNEL_WARP, md.MD_LIST_FULL), ("cell", md.MD_KERNEL_CELL, md.MD_LIST_FULL),
                ("half", md.MD_KERNEL_TPA, md.MD_LIST_HALF)]
    print("# Cutoff sweep of the force-kernel variants (LJ fluid, density 0.8442, skin 0.3)\n")
    print("Command: `python -m paper_1009_4330_b200.sweep%s --cells %s --rc %s --precision %s --melt %d --reps %d` on %s.\n"
          % ((" --nsweep " + args.nsweep) if args.nsweep else "", args.cells, args.rc, args.precision, args.melt, args.reps,
             torch.cuda.get_device_name(0)))
    print("Times are ms per force evaluation (device time, best of %d); `build` is ms per list build with the thread-per-atom "
          "layout; `G entries/s` = N x exact list entries / best full-list time; the planner chooses the tile shape of every cell "
          "(no autotuning: MD_KERNEL_* given explicitly).\n" % args.reps)
    if args.nsweep:
        print("## Whole path (md_run: builds + forces + integration) against system size, rc = 2.5, %d steps, MD_KERNEL_AUTO\n" % args.nsteps)
        print("| atoms | tile shape | tiles | variant | builds | ms per step | atom-steps/s |")
        print("|---|---|---|---|---|---|---|")
        for n in [int(c) for c in args.nsweep.split(",")]:
            w = wl.make(2, n_override=n)
            s = md.from_workload(w, kernel=md.MD_KERNEL_AUTO)
            s.md_run(args.nsteps, w.dt)                      # melts the lattice; selects variant and tile shape
            s.md_run(args.nsteps, w.dt)
            st = s.md_get_stats()
            print("| %d | %s | %d | %s | %d | %.4f | %.3e |" % (w.natoms, "x".join(str(b) for b in st["brick"]), st["ntiles"],
                  md.KERNEL_NAMES[st["kernel_variant"]], st["nbuilds_in_run"], st["ms_run"] / args.nsteps,
                  w.natoms * args.nsteps / (st["ms_run"] * 1e-3)), flush=True)
            s.close()
        print()
    for n in [int(c) for c in args.cells.split(",") if c]:
        base = wl.make(2, n_override=n)
        # melt once with the default cutoff so that every cutoff sees the same liquid snapshot
        s = md.from_workload(base, kernel=md.MD_KERNEL_TPA)
        s.md_run(args.melt, base.dt)
        x = np.zeros((base.natoms, 3))
        s.md_get_positions(x)
        s.close()
        for prec_name in args.precision.split(","):
            rc_table(md, base, x, n, prec_name, variants, args)


def rc_table(md, base, x, n, prec_name, variants, args) -> None:
    """One table: force time of every variant against the cutoff, for one system size and precision."""
    prec = {"mixed": md.MD_MIXED, "fp64": md.MD_FP64}[prec_name]
    print("## %d atoms (%d^3 fcc cells, box %.3f sigma), %s\n" % (base.natoms, n, base.box[0], prec_name))
    print("| rc | list entries/atom | " + " | ".join(v[0] for v in variants) + " | build | fastest | G entries/s |")
    print("|---|---|" + "---|" * (len(variants) + 3))
    for rc in [float(r) for r in args.rc.split(",")]:
        if base.box[0] < 3.0 * (rc + base.skin):
            print("| %.1f | box < 3 (rc+skin) |" % rc + " |" * (len(variants) + 3))
            continue
        w = dataclasses.replace(base, rc=rc)
        times, nl, tbuild = {}, None, None
        for name, kernel, lk in variants:
            try:
                s = md.from_workload(w, precision=prec, kernel=kernel, list_kind=lk, x=x)
                s.md_build_neighbors()
                s.md_compute_forces()                     # warm-up
                best = 1e300
                for _ in range(args.reps):
                    s.md_compute_forces()
                    best = min(best, s.md_get_stats()["ms_force"])
                st = s.md_get_stats()
                times[name] = best
                if name == "tpa":
                    nl, tbuild = st["mean_neighbors"], st["ms_build"]
                s.close()
            except md.MDError as e:                      # e.g. the tile does not fit shared memory at this cutoff
                times[name] = None
                print("<!-- rc %.1f %s: %s -->" % (rc, name, e), file=sys.stderr)
        full = {k: v for k, v in times.items() if v is not None and k in ("tpa", "subwarp2", "subwarp4", "subwarp8", "warp")}
        fastest = min(full, key=full.get) if full else "-"
        rate = base.natoms * nl / (full[fastest] * 1e-3) / 1e9 if full and nl else float("nan")
        print("| %.1f | %s | " % (rc, "%.1f" % nl if nl else "-") +
              " | ".join("%.4f" % times[v[0]] if times[v[0]] is not None else "n/a" for v in variants) +
              " | %s | %s | %.0f |" % ("%.3f" % tbuild if tbuild else "-", fastest, rate), flush=True)
    print()


if __name__ == "__main__":
    main()
