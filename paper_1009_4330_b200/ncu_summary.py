"""Turns Nsight Compute output into the text summaries kept under ``profiles/`` (no GPU needed: it only reads
reports; ``ncu`` must be on PATH for ``full``).

    # one kernel of an ``ncu --set full`` report -> Markdown table (+ the machine-readable ``dram_bytes_per_launch`` line
    # that bench.py reads back as ``roofline.traffic``)
    python -m paper_1009_4330_b200.ncu_summary full gpurun_out/X.ncu-rep --capture-cmd "<the command that wrote X>" > profiles/Y.md

    # the launch list of ``ncu --metrics gpu__time_duration.sum --csv --log-file L.csv <bench command>`` -> per-kernel shares
    python -m paper_1009_4330_b200.ncu_summary launches gpurun_out/L.csv --capture-cmd "<command>" > profiles/Z.md

    # the DRAM bytes per launch recorded in a summary written by ``full``
    python -m paper_1009_4330_b200.ncu_summary traffic profiles/Y.md
"""
from __future__ import annotations

import argparse
import collections
import csv
import io
import re
import subprocess
import sys

# metric -> what it says (the ones DESIGN.md and the bench line argue from)
METRICS = [
    ("gpu__time_duration.sum", "kernel duration"),
    ("launch__grid_size", "grid"), ("launch__block_size", "block"), ("launch__registers_per_thread", "registers per thread (at launch)"),
    ("launch__shared_mem_per_block_dynamic", "dynamic shared memory per block"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "achieved occupancy"),
    ("dram__bytes_read.sum", "DRAM bytes read"), ("dram__bytes_write.sum", "DRAM bytes written"),
    ("dram__throughput.avg.pct_of_peak_sustained_elapsed", "DRAM throughput, % of peak"),
    ("lts__t_sector_hit_rate.pct", "L2 hit rate"),
    ("smsp__inst_executed.sum", "warp instructions executed"),
    ("smsp__thread_inst_executed_per_inst_executed.ratio", "active threads per warp instruction"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots busy"),
    ("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "FMA pipe busy"),
    ("sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed", "FMA-heavy pipe busy (packed f32x2 run here)"),
    ("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "ALU pipe busy"),
    ("sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "XU (MUFU) pipe busy"),
    ("sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active", "FP64 pipe busy"),
    ("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed", "L1/shared data pipe (LSU wavefronts), % of peak"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "shared-memory wavefronts"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "of which bank-conflict replays"),
    ("l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum", "global load sectors"),
    ("l1tex__t_sectors_pipe_lsu_mem_global_op_st.sum", "global store sectors"),
    ("smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio", "stall: long scoreboard (global/L2) per issue"),
    ("smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio", "stall: short scoreboard (shared, MUFU) per issue"),
    ("smsp__average_warps_issue_stalled_wait_per_issue_active.ratio", "stall: fixed-latency wait per issue"),
    ("smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio", "stall: math pipe throttle per issue"),
    ("smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio", "stall: not selected per issue"),
    ("smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio", "stall: barrier per issue"),
]
UNIT_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def _raw_rows(rep: str):
    out = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(io.StringIO(out)))
    return rows[0], rows[1], rows[2:]


def full(args) -> None:
    hdr, units, body = _raw_rows(args.report)
    col = {h: i for i, h in enumerate(hdr)}
    name_col = col.get("Kernel Name")
    print("# ncu --set full: %s\n" % args.report.split("/")[-1])
    print("Capture (on the B200 box):\n\n    %s\n" % args.capture_cmd)
    print("Read back (here, no GPU): `python -m paper_1009_4330_b200.ncu_summary full %s` = `ncu -i %s --page raw --csv` filtered to the "
          "metrics below.\n" % (args.report, args.report))
    for row in body:
        kname = row[name_col] if name_col is not None else "?"
        if args.kernel and not re.search(args.kernel, kname):
            continue
        print("## %s\n" % kname)
        print("| metric | value | unit | meaning |\n|---|---|---|---|")
        dram = 0.0
        for m, what in METRICS:
            if m not in col:
                continue
            v, u = row[col[m]], units[col[m]]
            print("| `%s` | %s | %s | %s |" % (m, v, u, what))
            if m in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                dram += float(v.replace(",", "")) * UNIT_BYTES.get(u, 1.0)
        print("\ndram_bytes_per_launch: %.0f\n" % dram)
    if args.note:
        print(args.note)


def launches(args) -> None:
    rows = list(csv.reader(open(args.csv)))
    start = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    h = {k: i for i, k in enumerate(rows[start])}
    agg = collections.OrderedDict()
    for r in rows[start + 1:]:
        if len(r) < len(h) or r[h["Metric Name"]] != "gpu__time_duration.sum":
            continue
        v = float(r[h["Metric Value"]].replace(",", "")) * {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(r[h["Metric Unit"]], 1.0)
        name = re.sub(r"\(.*$", "", r[h["Kernel Name"]])
        a = agg.setdefault(name, [0, 0.0])
        a[0] += 1
        a[1] += v
    tot = sum(a[1] for a in agg.values())
    print("# ncu launch list: %s\n" % args.csv.split("/")[-1])
    print("Capture (on the B200 box; per-launch times under ncu are cold-cache and serialised -- the SHARES are what is compared "
          "with bench.py's live CUDA-event figures):\n\n    %s\n" % args.capture_cmd)
    print("| kernel | launches | total us | us per launch | share |\n|---|---|---|---|---|")
    for n, (c, t) in sorted(agg.items(), key=lambda kv: -kv[1][1]):
        print("| `%s` | %d | %.1f | %.1f | %.1f %% |" % (n, c, t, t / c, 100 * t / tot))
    print("\ntotal: %d launches, %.1f us" % (sum(a[0] for a in agg.values()), tot))
    if args.note:
        print("\n" + args.note)


def traffic(path: str, sections: int = 1):
    """DRAM bytes per launch recorded by ``full`` in a summary file: the sum over the first ``sections`` kernel
    sections (2 for EAM: density pass + force pass), or None if the file or a section is missing."""
    found = []
    try:
        with open(path) as fh:
            for line in fh:
                m = re.match(r"dram_bytes_per_launch:\s*([0-9.eE+]+)", line)
                if m:
                    found.append(float(m.group(1)))
    except OSError:
        return None
    return sum(found[:sections]) if len(found) >= sections else None


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    sub = ap.add_subparsers(dest="cmd", required=True)
    f = sub.add_parser("full"); f.add_argument("report"); f.add_argument("--kernel", default=""); f.add_argument("--capture-cmd", default="(not recorded)")
    f.add_argument("--note", default="")
    l = sub.add_parser("launches"); l.add_argument("csv"); l.add_argument("--capture-cmd", default="(not recorded)"); l.add_argument("--note", default="")
    t = sub.add_parser("traffic"); t.add_argument("summary")
    args = ap.parse_args()
    if args.cmd == "full":
        full(args)
    elif args.cmd == "launches":
        launches(args)
    else:
        print(traffic(args.summary))


if __name__ == "__main__":
    sys.exit(main())
