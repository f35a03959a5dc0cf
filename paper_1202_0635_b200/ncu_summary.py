"""Summarise an Nsight Compute report of one of this library's kernels as markdown, and record the per-launch counts
that bench.py's roofline block needs in profiles/traffic.json.

    python -m paper_1202_0635_b200.ncu_summary REPORT.ncu-rep [--title T] [--phases FILE:NAME=a-b,...] [--record KEY]

Runs anywhere `ncu` is installed (no GPU needed to read a report).  What it prints:
  * the headline metrics of the launch (duration, DRAM bytes, instruction counts, pipe utilisation, occupancy, stalls);
  * the executed-opcode histogram from the source page, grouped by the pipe each opcode occupies, and the busy cycles of
    every pipe per launch under the issue model MEASURED by `bench.py --microbench` (profiles/r2_microbench.md): ALU-class
    2 cycles per warp-instruction on the ALU pipe, IMAD 2 on FMA, IMAD.WIDE 4 on FMA + 2 on ALU, IMAD.HI 4 on FMA,
    FLO/BREV/POPC 8 on XU, shared-memory / shuffle / vote 4 on the LSU, everything else one issue slot;
  * with --phases, the same split per source-line range, next to the stall samples of the range.
--record KEY stores {dram bytes, instruction counts per class} under KEY in profiles/traffic.json together with the hash of
the kernel sources, so that bench.py can tell whether the capture still describes the code it is timing.
"""
from __future__ import annotations

import argparse
import collections
import csv
import hashlib
import json
import re
import subprocess
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent
ALU = {"LOP3", "IADD3", "IADD", "ISETP", "SEL", "SHF", "LEA", "VIADD", "PRMT", "IABS", "PLOP3", "IMNMX", "VIMNMX", "BMSK", "SGXT", "P2R",
       "R2P", "MOV", "CS2R", "VABSDIFF", "I2FP", "VIADDMNMX", "FMNMX", "FSEL", "FSETP"}
XU = {"FLO", "POPC", "BREV", "MUFU", "I2F", "F2I", "F2F"}
LSU = {"LDS", "STS", "ATOMS", "SHFL", "LDG", "STG", "LD", "ST", "ATOMG", "ATOM", "RED", "REDG", "LDSM", "VOTE", "MATCH", "REDUX", "LDL", "STL"}
KEYS = ["gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum", "lts__t_bytes.sum", "smsp__inst_executed.sum",
        "smsp__inst_issued.sum", "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active",
        "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
        "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_xu_cycles_active.avg.pct_of_peak_sustained_active",
        "launch__grid_size", "launch__registers_per_thread", "launch__shared_mem_per_block_static", "launch__shared_mem_per_block_dynamic",
        "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "smsp__cycles_active.avg", "sm__cycles_elapsed.max"]


def csrc_sha256() -> str:
    h = hashlib.sha256()
    for p in sorted((ROOT / "paper_1202_0635_b200" / "csrc").glob("*")):
        h.update(p.name.encode())
        h.update(p.read_bytes())
    return h.hexdigest()


def classify(op: str):
    """-> {pipe: busy cycles per warp-instruction} under the measured issue model."""
    base = op.split(".")[0]
    if base == "IMAD" and "WIDE" in op:
        return "imad_wide", {"fma": 4, "alu": 2}
    if base == "IMAD" and ".HI" in op:
        return "imad_hi", {"fma": 4}
    if base in ("IMAD", "FFMA", "FMUL", "FADD", "HFMA2", "HADD2", "HMUL2"):
        return "fma", {"fma": 2}
    if base in ALU:
        return "alu", {"alu": 2}
    if base in XU:
        return "xu", {"xu": 8}
    if base in LSU:
        return "lsu", {"lsu": 4}
    return "other", {}


def read_raw(rep: str):
    raw = subprocess.run(["ncu", "-i", rep, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    r = list(csv.reader(raw.splitlines()))
    return {name: (val, unit) for name, unit, val in zip(r[0], r[1], r[2])}


def num(vals, k):
    v, u = vals[k]
    return float(v.replace(",", "")) * {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(u, 1)


def read_source(rep: str):
    """-> list of (file, line, opcode, warp instructions executed, {stall: samples}, samples, SASS address, thread
    instructions executed), in SASS address order."""
    src = subprocess.run(["ncu", "-i", rep, "--page", "source", "--csv", "--print-source", "cuda,sass"], capture_output=True, text=True, check=True).stdout
    out, cur, line, h = [], None, None, None
    seen = set()       # an instruction inlined from a helper is listed under every source line of its inline chain: count it once
    for r in csv.reader(src.splitlines()):
        if r and r[0] == "File Path":
            cur = r[1].split("/")[-1]
            continue
        if r and r[0] == "Line No":
            h = r
            ii, si, ti = h.index("Instructions Executed"), h.index("# Samples"), h.index("Thread Instructions Executed")
            st = {n[6:]: h.index(n) for n in h if n.startswith("stall_") and "Not Issued" not in n}
            continue
        if not r or h is None:
            continue
        if r[0].isdigit():
            line = int(r[0])
            continue
        if r[0] == "" and len(r) > ii and r[3] not in ("...", "-"):
            try:
                n = int(r[ii])
            except ValueError:
                continue
            m = re.match(r"\s*(@!?U?P\d+\s+)?([A-Z0-9_.]+)", r[3])
            if m and r[2] in seen:
                continue
            seen.add(r[2])
            if m:
                stalls = {}
                for k, ix in st.items():
                    try:
                        stalls[k] = int(r[ix] or 0)
                    except ValueError:
                        pass
                out.append((cur, line, m.group(2), n, stalls, int(r[si] or 0), int(r[2], 16), int(r[ti] or 0)))
    out.sort(key=lambda t: t[6])          # SASS address order
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--title", default=None)
    ap.add_argument("--phases", default=None, help="FILE:NAME=a-b,NAME=a-b,... (source-line ranges of FILE)")
    ap.add_argument("--record", default=None, help="key under which the per-launch counts go into profiles/traffic.json")
    ap.add_argument("--sms", type=int, default=148)
    args = ap.parse_args()

    vals = read_raw(args.report)
    print(f"## {args.title or vals.get('Kernel Name', ('?', ''))[0]}\n")
    print("| metric | value |\n|---|---|")
    for k in KEYS:
        if k in vals:
            print(f"| {k} | {vals[k][0]} {vals[k][1]} |")
    for k in sorted(vals):
        if k.startswith("smsp__average_warps_issue_stalled") and k.endswith("_per_issue_active.ratio") and "not_issued" not in k:
            try:
                if float(vals[k][0]) >= 0.3:
                    print(f"| {k} | {vals[k][0]} |")
            except ValueError:
                pass
    rows = read_source(args.report)
    ops = collections.Counter()
    cls = collections.Counter()
    busy = collections.Counter()
    for _, _, op, n, _, _, _, _ in rows:
        c, b = classify(op)
        ops["IMAD.WIDE" if c == "imad_wide" else "IMAD.HI" if c == "imad_hi" else op.split(".")[0]] += n
        cls[c] += n
        for pipe, cyc in b.items():
            busy[pipe] += cyc * n
    total = sum(cls.values())
    print("\n### executed opcodes (warp-instructions per launch, source page)\n")
    print("| opcode | M | | opcode | M |\n|---|---|---|---|---|")
    top = ops.most_common(20)
    for a, b in zip(top[:10], top[10:] + [("", 0)] * 10):
        print(f"| {a[0]} | {a[1] / 1e6:.2f} | | {b[0]} | {b[1] / 1e6:.2f} |" if b[0] else f"| {a[0]} | {a[1] / 1e6:.2f} | | | |")
    dur_us = num(vals, "gpu__time_duration.sum") * {"usecond": 1, "msecond": 1e3, "nsecond": 1e-3, "second": 1e6}.get(vals["gpu__time_duration.sum"][1], 1)
    clk = None
    if "smsp__cycles_active.avg" in vals and "sm__cycles_elapsed.max" in vals:
        clk = num(vals, "sm__cycles_elapsed.max") / dur_us      # MHz
    avail = args.sms * 4 * (clk or 1965.0) * dur_us
    print(f"\n### pipe demand per launch under the measured issue model ({args.sms} SMs x 4 sub-partitions x {clk or 1965.0:.0f} MHz x {dur_us:.1f} us = {avail / 1e6:.1f} M cycles available)\n")
    print("| pipe | busy cycles (M) | of available |\n|---|---|---|")
    for pipe in ("alu", "fma", "xu", "lsu"):
        print(f"| {pipe} | {busy[pipe] / 1e6:.1f} | {busy[pipe] / avail:.3f} |")
    print(f"| issue slots | {total / 1e6:.1f} | {total / avail:.3f} |")
    print(f"\nclasses (M warp-instructions): " + ", ".join(f"{k} {v / 1e6:.2f}" for k, v in cls.most_common()))

    if args.phases:
        fname, spec = args.phases.split(":", 1)
        ph = []
        for item in spec.split(","):
            name, rng = item.split("=")
            a, b = rng.split("-")
            ph.append((int(a), int(b), name))
        agg = collections.defaultdict(collections.Counter)
        # in SASS address order; an instruction inlined from a helper (Philox, bit scans, label loads) belongs to the phase
        # of the nearest preceding instruction that maps to a line of FILE itself
        key = "prologue"
        for f, line, op, n, stalls, smp, _, tn in rows:
            if f == fname:
                key = next((nm for a, b, nm in ph if a <= line <= b), key)
            a = agg[key]
            a["inst"] += n
            a["thread_inst"] += tn
            a["samples"] += smp
            for pipe, cyc in classify(op)[1].items():
                a[pipe] += cyc * n
            for k, v in stalls.items():
                a["stall_" + k] += v
        tot_s = sum(a["samples"] for a in agg.values()) or 1
        print("\n### by phase (source-line ranges of " + fname + ", SASS address order): instructions, active lanes, pipe cycles (M) and share of the warp-stall samples\n")
        print("| phase | inst M | lanes | alu | fma | xu | lsu | samples | top stall reasons |\n|---|---|---|---|---|---|---|---|---|")
        for k, a in agg.items():
            st = sorted(((n[6:], c) for n, c in a.items() if n.startswith("stall_")), key=lambda t: -t[1])[:4]
            print(f"| {k} | {a['inst'] / 1e6:.2f} | {a['thread_inst'] / max(1, a['inst']):.1f} | {a['alu'] / 1e6:.1f} | {a['fma'] / 1e6:.1f} | {a['xu'] / 1e6:.1f} | "
                  f"{a['lsu'] / 1e6:.1f} | {a['samples'] / tot_s:.3f} | " + ", ".join(f"{n} {c / max(1, a['samples']):.2f}" for n, c in st) + " |")

    if args.record:
        tj = ROOT / "profiles" / "traffic.json"
        d = json.loads(tj.read_text()) if tj.exists() else {}
        d[args.record] = {
            "dram_bytes": num(vals, "dram__bytes_read.sum") + num(vals, "dram__bytes_write.sum"),
            "duration_us": dur_us,
            "warp_instructions": total,
            "alu_class": cls["alu"], "imad_wide": cls["imad_wide"], "imad_hi": cls["imad_hi"], "fma_class": cls["fma"],
            "xu_class": cls["xu"], "lsu_class": cls["lsu"],
            "alu_pipe_cycles": busy["alu"], "fma_pipe_cycles": busy["fma"], "xu_pipe_cycles": busy["xu"], "lsu_pipe_cycles": busy["lsu"],
            "csrc_sha256": csrc_sha256(),
            "report": Path(args.report).name,
        }
        tj.write_text(json.dumps(d, indent=1, sort_keys=True) + "\n")


if __name__ == "__main__":
    main()
