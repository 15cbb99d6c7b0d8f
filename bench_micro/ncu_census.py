#!/usr/bin/env python
"""Instruction census of one profiled kernel launch from an `ncu --set full --import-source on` report.

    python bench_micro/ncu_census.py <file.ncu-rep> [--units N] [--label TEXT]

Reads the report's SOURCE page (per-SASS-instruction "Instructions Executed", warp level) and its RAW page (cycles,
pipe utilisation) with the `ncu` command-line tool - no GPU needed - and prints, as markdown:

  * executed warp instructions by opcode class, in total and per unit-MCS when --units gives the number of
    (thread, MCS) work items of the launch (e.g. 1024 rings x 32 threads x 2000 MCS);
  * the alu-pipe SLOT count of DESIGN.md 6.1 = LOP3 + SHF + PRMT + SEL + IMAD.WIDE (an IMAD.WIDE takes one alu-pipe
    slot besides its 4 clk on the fmaheavy pipe: profiles/r01_pipe_rates.md), and the cycles it implies at 2 clk per slot
    and SMSP, next to the cycles the launch took: the second, independent line of evidence for the alu roofline;
  * ncu's own pipe / issue counters of the same launch.

It is evidence tooling for profiles/, not part of the product path.
"""
from __future__ import annotations

import argparse
import csv
import io
import subprocess
import sys
from collections import Counter

ALU_SLOT = ("LOP3", "SHF", "PRMT", "SEL", "LEA", "ISETP", "IMNMX", "VOTE", "POPC_NOT", "FLO_NOT")   # alu pipe, 0.5 warp-instr/clk
# (POPC / FLO run on their own slow pipe; IADD3 / IMAD.lo issue on the fma pipes at full rate: measured, r01_pipe_rates.md)


def ncu_csv(rep: str, page: str) -> list[list[str]]:
    out = subprocess.run(["ncu", "-i", rep, "--page", page, "--csv"], check=True, capture_output=True, text=True).stdout
    return list(csv.reader(io.StringIO(out)))


def opcode(sass: str) -> str:
    s = sass.strip()
    if s.startswith("@"):
        s = s.split(None, 1)[1] if " " in s else s
    return s.split()[0].rstrip(";") if s else "?"


def classify(op: str) -> str:
    base = op.split(".")[0]
    if base == "IMAD":
        if ".WIDE" in op:
            return "IMAD.WIDE"
        if ".HI" in op:
            return "IMAD.HI"
        if ".MOV" in op:
            return "IMAD.MOV"
        return "IMAD.lo"
    return base


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--units", type=float, default=None, help="(thread, MCS) work items of the launch x 1/32 = warp-MCS")
    ap.add_argument("--label", default="")
    args = ap.parse_args()

    rows = ncu_csv(args.report, "source")
    hdr_i = next(i for i, r in enumerate(rows) if r and r[0] == "Address")
    hdr = rows[hdr_i]
    c_src, c_exec = hdr.index("Source"), hdr.index("Instructions Executed")
    kernel = rows[0][1] if rows and len(rows[0]) > 1 else "?"
    counts: Counter = Counter()
    for r in rows[hdr_i + 1:]:
        if len(r) <= c_exec or not r[c_exec]:
            continue
        try:
            n = int(float(r[c_exec]))
        except ValueError:
            continue
        counts[classify(opcode(r[c_src]))] += n
    total = sum(counts.values())

    raw = ncu_csv(args.report, "raw")
    rh, rv = raw[0], raw[-1]
    def metric(name):
        return float(rv[rh.index(name)]) if name in rh and rv[rh.index(name)] not in ("", "n/a") else None
    cyc_active = metric("smsp__cycles_active.avg")
    cyc_elapsed = metric("sm__cycles_elapsed.max")
    n_smsp = 4 * 148
    slots = sum(counts[k] for k in ("LOP3", "SHF", "PRMT", "SEL", "LEA", "IMAD.WIDE"))
    alu_only = sum(counts[k] for k in ("LOP3", "SHF", "PRMT", "SEL", "LEA"))
    alu_pipe = alu_only + sum(counts[k] for k in ("ISETP", "PLOP3", "IMNMX", "VOTE", "FLO", "BREV", "IABS", "ICMP"))

    w = args.units / 32.0 if args.units else None
    print(f"### {args.label or args.report}: kernel `{kernel}`\n")
    print(f"executed warp instructions: {total:,}" + (f" = {total / w:.1f} per warp-MCS" if w else ""))
    print()
    print("| opcode class | warp instructions | share |" + (" per warp-MCS |" if w else ""))
    print("|---|---|---|" + ("---|" if w else ""))
    for op, n in counts.most_common(18):
        print(f"| {op} | {n:,} | {100.0 * n / total:.1f} % |" + (f" {n / w:.1f} |" if w else ""))
    print()
    print(f"alu-pipe slot instructions (LOP3 + SHF + PRMT + SEL + LEA + IMAD.WIDE): {slots:,}"
          + (f" = {slots / w:.1f} per warp-MCS" if w else "") + f"; without IMAD.WIDE: {alu_only:,}")
    if cyc_elapsed:
        act = cyc_active or cyc_elapsed
        print(f"- slot instructions per SMSP x 2 clk = {2 * slots / n_smsp:,.0f} clk = {100.0 * 2 * slots / n_smsp / cyc_elapsed:.1f} % of the "
              f"{cyc_elapsed:,.0f} elapsed SM cycles (mean over {n_smsp} SMSPs): the executed slot occupancy")
        print(f"- check against ncu: LOP3 + SHF + PRMT + SEL + LEA x 2 clk = {100.0 * 2 * alu_only / n_smsp / act:.1f} % of the "
              f"{act:,.0f} ACTIVE cycles per SMSP ({100.0 * 2 * alu_pipe / n_smsp / act:.1f} % with ISETP / PLOP3 / VOTE); "
              f"ncu's `sm__pipe_alu_cycles_active` (per active cycle) is in the table below")
    print()
    print("| ncu counter | value |")
    print("|---|---|")
    for name in ("gpu__time_duration.sum", "sm__cycles_elapsed.max", "smsp__cycles_active.avg", "smsp__inst_executed.sum",
                 "smsp__issue_active.avg.pct_of_peak_sustained_active",
                 "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
                 "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
                 "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_active",
                 "sm__inst_executed_pipe_fmaheavy.avg.pct_of_peak_sustained_active",
                 "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
                 "sm__warps_active.avg.pct_of_peak_sustained_active", "launch__registers_per_thread",
                 "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
                 "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
                 "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
                 "smsp__average_warps_issue_stalled_dispatch_stall_per_issue_active.ratio",
                 "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
                 "smsp__average_warps_issue_stalled_no_instruction_per_issue_active.ratio",
                 "dram__bytes_read.sum", "dram__bytes_write.sum"):
        if name in rh:
            print(f"| `{name}` | {rv[rh.index(name)]} {raw[1][rh.index(name)]} |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
