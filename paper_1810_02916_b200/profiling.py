"""Turns ncu output into the text summaries kept under profiles/ (no arithmetic of the method).

    python -m paper_1810_02916_b200.profiling launches <ncu.csv> <out.md> --title T --command C
        per-kernel table of an `ncu --metrics gpu__time_duration.sum --csv` launch list
    python -m paper_1810_02916_b200.profiling full <raw.csv> <out.md> --title T --command C [--kernel REGEX] [--interactions I]
        the counters DESIGN.md quotes, from `ncu -i x.ncu-rep --page raw --csv`
    python -m paper_1810_02916_b200.profiling sass <out.md>
        SASS facts of the interaction kernel k_forces_warp<2, false, false> (R = 2, no masses, no dense-cell logic) in the built libnf.so (cuobjdump -sass): mnemonic
        counts that show the Blackwell instructions in use, and the body of the untracked (MODE 2) sweep loop
    python -m paper_1810_02916_b200.profiling traffic <workload> <ncu.csv> --command C
        records dram__bytes_read.sum / dram__bytes_write.sum of one interaction-kernel launch on <workload> in
        profiles/interaction_kernel_traffic.json together with the hash of the kernel sources it was captured
        from; bench.py reports it as roofline.traffic only while the sources are unchanged.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import re
import sys
from collections import OrderedDict

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "interaction_kernel_traffic.json")
KERNEL_SOURCES = ["paper_1810_02916_b200/csrc/nf_forces.cu", "paper_1810_02916_b200/csrc/nf_common.cuh"]

UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
        "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0, "nsecond": 1e-9, "usecond": 1e-6, "msecond": 1e-3, "second": 1.0}

FULL_METRICS = [
    "gpu__time_duration.sum", "sm__cycles_elapsed.avg.per_second", "launch__grid_size", "launch__block_size",
    "launch__registers_per_thread", "launch__shared_mem_per_block_dynamic", "sm__warps_active.avg.pct_of_peak_sustained_active",
    "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "smsp__thread_inst_executed_per_inst_executed.ratio", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_elapsed", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active",
    "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active", "dram__bytes_read.sum", "dram__bytes_write.sum",
    "dram__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_sector_hit_rate.pct",
    "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
    "smsp__warps_eligible.avg.per_cycle_active",
    "smsp__average_warps_issue_stalled_barrier_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_branch_resolving_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_dispatch_stall_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_mio_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_no_instruction_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_selected_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_sleeping_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_wait_per_issue_active.ratio",
    "smsp__average_warps_issue_stalled_membar_per_issue_active.ratio",
]


def kernel_source_hash() -> str:
    """sha256 over the interaction kernel's sources: what a stored ncu counter is valid for (the GPU box
    has no .git, so a commit id cannot be checked there)."""
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def read_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one interaction-kernel launch on `workload`, or None
    when no capture is recorded or it was taken from other kernel sources than the ones in this tree."""
    try:
        with open(TRAFFIC_JSON) as fh:
            rec = json.load(fh).get(workload)
    except (OSError, ValueError):
        return None
    if not rec or rec.get("kernel_source_sha256") != kernel_source_hash():
        return None
    return float(rec["dram_bytes_read"]) + float(rec["dram_bytes_write"])


def short_name(full: str) -> str:
    m = re.search(r"(k_\w+)(<[^(]*>)?", full)
    return (m.group(1) + (m.group(2) or "")) if m else full[:60]


def _rows_long(path):
    """rows of an ncu --csv log (one row per launch and metric); lines before the header are skipped"""
    with open(path, newline="") as fh:
        lines = fh.readlines()
    start = next(i for i, l in enumerate(lines) if l.startswith('"ID"'))
    return list(csv.DictReader(lines[start:]))


def _num(s: str) -> float:
    return float(s.replace(",", ""))


def cmd_launches(a):
    per = OrderedDict()
    for r in _rows_long(a.csv):
        if r["Metric Name"] != "gpu__time_duration.sum":
            continue
        k = short_name(r["Kernel Name"])
        e = per.setdefault(k, {"n": 0, "t": 0.0, "grid": r["Grid Size"], "block": r["Block Size"]})
        e["n"] += 1
        e["t"] += _num(r["Metric Value"]) * UNIT.get(r["Metric Unit"], 1e-9)
    total = sum(e["t"] for e in per.values())
    out = [f"# {a.title}", "", "Command (on the B200 box, after the same command had exited 0 without ncu):", "", f"    {a.command}", ""]
    if a.note:
        out += [a.note, ""]
    out += ["| kernel | launches | total ms | ms each | share | grid | block |", "|---|---|---|---|---|---|---|"]
    for k, e in per.items():
        out.append(f"| `{k}` | {e['n']} | {1e3 * e['t']:.3f} | {1e3 * e['t'] / e['n']:.3f} | {100 * e['t'] / total:.2f} % | {e['grid']} | {e['block']} |")
    out += ["", f"Total {1e3 * total:.1f} ms of libnf kernel time in {sum(e['n'] for e in per.values())} launches.  "
            "Times under ncu are serialised and cold-cache: what must agree with the bench line is the interaction kernel's SHARE."]
    with open(a.out, "w") as fh:
        fh.write("\n".join(out) + "\n")


def _raw_table(path, kernel_re):
    """`--page raw --csv`: one row per launch, one column per metric; the second line holds the units"""
    with open(path, newline="") as fh:
        rows = list(csv.reader(fh))
    start = next(i for i, r in enumerate(rows) if r and r[0] == "ID")
    head, units, data = rows[start], rows[start + 1], rows[start + 2:]
    ki = head.index("Kernel Name")
    sel = [r for r in data if len(r) == len(head) and re.search(kernel_re, r[ki])]
    return head, units, sel


def cmd_full(a):
    head, units, sel = _raw_table(a.csv, a.kernel)
    if not sel:
        raise SystemExit(f"no launch matching {a.kernel!r} in {a.csv}")
    r = sel[a.index]
    val = {h: (v, u) for h, u, v in zip(head, units, r)}
    out = [f"# {a.title}", "", "Command (on the B200 box, after the same command had exited 0 without ncu):", "", f"    {a.command}", "",
           f"Read with `ncu -i <rep> --page raw --csv`; kernel `{short_name(val['Kernel Name'][0])}`.", ""]
    if a.note:
        out += [a.note, ""]
    out += ["| metric | unit | value |", "|---|---|---|"]
    for m in FULL_METRICS:
        if m in val:
            out.append(f"| {m} | {val[m][1]} | {val[m][0]} |")
    if a.interactions:
        t = _num(val["gpu__time_duration.sum"][0]) * UNIT.get(val["gpu__time_duration.sum"][1], 1e-9)
        inst = _num(val["smsp__inst_executed.sum"][0])
        out += ["", f"{a.interactions:.6g} interactions in {1e3 * t:.3f} ms = {a.interactions / t:.4g} /s under ncu; "
                f"{inst / (a.interactions / 32):.3f} warp-instructions per 32 interactions."]
    with open(a.out, "w") as fh:
        fh.write("\n".join(out) + "\n")


def cmd_sass(a):
    import subprocess
    lib = os.path.join(ROOT, "paper_1810_02916_b200", "libnf.so")
    cmd = ["cuobjdump", "-sass", lib]
    txt = subprocess.run(cmd, capture_output=True, text=True, check=True).stdout
    m = re.search(r"Function : (\S*k_forces_warpILi2ELb0ELb0E\S*)(.*?)(?=\n\s*Function :|\Z)", txt, re.S)
    if not m:
        raise SystemExit("k_forces_warp<2, false, false> not found in " + lib)
    lines = []
    for l in m.group(2).splitlines():
        mm = re.match(r"\s*/\*([0-9a-f]{4,5})\*/\s+(.*?);\s*/\*", l)
        if mm:
            lines.append((int(mm.group(1), 16), mm.group(2).strip()))
    def opc(t):
        f = t.split()
        return (f[1] if f[0].startswith("@") else f[0]).split(".")[0]
    cnt = {}
    for _, t in lines:
        cnt[opc(t)] = cnt.get(opc(t), 0) + 1
    full = {}
    for _, t in lines:
        f = t.split()
        k = f[1] if f[0].startswith("@") else f[0]
        full[k] = full.get(k, 0) + 1
    addr = {a_: i for i, (a_, _) in enumerate(lines)}
    loops = []
    for i, (a_, t) in enumerate(lines):
        mm = re.search(r"\bBRA\s+0x([0-9a-f]+)", t)
        if mm and "BRA.DIV" not in t:
            tgt = int(mm.group(1), 16)
            if tgt < a_ and tgt in addr:
                body = lines[addr[tgt]:i + 1]
                n2 = sum(1 for _, b in body if re.match(r"(@\S+\s+)?(FFMA2|FADD2|FMUL2)", b))
                if n2 >= 100 and len(body) < 400:
                    loops.append((tgt, a_, body, n2))
    out = ["# SASS of the interaction kernel `k_forces_warp<2, false, false>` (built `libnf.so`, sm_100a)", "",
           "Command: `python -m paper_1810_02916_b200.profiling sass <this file>`, i.e. `cuobjdump -sass paper_1810_02916_b200/libnf.so`",
           f"on the library built from kernel sources sha256 {kernel_source_hash()[:16]}... (`python -m paper_1810_02916_b200.build`).", "",
           f"Function `{m.group(1)}`: {len(lines)} instructions.", "",
           "| mnemonic | count | what it shows |", "|---|---|---|"]
    notes = {"UBLKCP": "cp.async.bulk (TMA 1-D bulk copy global -> shared)", "SYNCS": "mbarrier operations (arrive / expect_tx / try_wait)",
             "FFMA2": "packed FP32 fused multiply-add (two sinks per instruction)", "FADD2": "packed FP32 add", "FMUL2": "packed FP32 multiply",
             "FMNMX3": "three-input min: close-pair tracking of MODE 1", "FMNMX": "two-input min: the `min` form of Eq. 2 (MODE 0)",
             "MUFU": "rsqrt (MUFU.RSQ) and the producer's reciprocal", "USETMAXREG": "setmaxnreg: registers moved from producers to consumers",
             "LDS": "shared-memory loads (LDS.128 broadcast of a source)", "FENCE": "fence.proxy.async before a bulk copy reuses a buffer",
             "NANOSLEEP": "the producer's timed sleep on its doorbell", "HMMA": "tensor-core MMA (none: not a contraction)", "UTCHMMA": "tcgen05 MMA (none)"}
    for k in ["UBLKCP", "SYNCS", "USETMAXREG", "FFMA2", "FADD2", "FMUL2", "MUFU", "FMNMX3", "FMNMX", "LDS", "FENCE", "NANOSLEEP", "HMMA", "UTCHMMA"]:
        out.append(f"| `{k}` | {cnt.get(k, 0)} | {notes[k]} |")
    out += ["", "Sweep loops (backward branches enclosing >= 100 packed FP32 instructions):", "",
            "| loop | instructions | FFMA2 | FADD2 | FMUL2 | MUFU.RSQ | FMNMX3 | FMNMX | LDS.128 | `.reuse` operands | which |", "|---|---|---|---|---|---|---|---|---|---|---|"]
    mode2 = None
    for tgt, a_, body, n2 in loops:
        c = lambda pat: sum(1 for _, b in body if re.match(r"(@\S+\s+)?" + pat, b))
        nm3, nm = c(r"FMNMX3"), c(r"FMNMX\b") + c(r"FMNMX\.")
        which = "MODE 1 (tracked)" if nm3 else ("MODE 0 (min form)" if nm else "MODE 2 (untracked r^-3)")
        if not nm3 and not nm and (mode2 is None or len(body) < len(mode2[2])):
            mode2 = (tgt, a_, body)
        out.append(f"| {tgt:#06x}-{a_:#06x} | {len(body)} | {c('FFMA2')} | {c('FADD2')} | {c('FMUL2')} | {c('MUFU.RSQ')} | {nm3} | {nm} | {c('LDS.128')} | "
                   f"{sum(b.count('.reuse') for _, b in body)} | {which} |")
    if mode2:
        tgt, a_, body = mode2
        out += ["", f"The MODE 2 loop ({tgt:#06x}-{a_:#06x}): 8 sources x 4 sinks per lane per iteration = 16 packed pairs x 11 FMA-pipe instructions + 32 MUFU.RSQ + 8 LDS.128.",
                "First 48 instructions:", "", "```"]
        out += [f"/*{x:04x}*/  {t}" for x, t in body[:48]]
        out += ["```"]
    with open(a.out, "w") as fh:
        fh.write("\n".join(out) + "\n")


def cmd_traffic(a):
    rd = wr = None
    t = None
    for r in _rows_long(a.csv):
        if not re.search("k_forces_warp", r["Kernel Name"]):
            continue
        v = _num(r["Metric Value"]) * UNIT.get(r["Metric Unit"], 1.0)
        if r["Metric Name"] == "dram__bytes_read.sum" and rd is None:
            rd = v
        elif r["Metric Name"] == "dram__bytes_write.sum" and wr is None:
            wr = v
        elif r["Metric Name"] == "gpu__time_duration.sum" and t is None:
            t = v
    if rd is None or wr is None:
        raise SystemExit("no dram__bytes_read.sum / dram__bytes_write.sum of k_forces_warp in " + a.csv)
    try:
        with open(TRAFFIC_JSON) as fh:
            d = json.load(fh)
    except (OSError, ValueError):
        d = {}
    d[a.workload] = {"dram_bytes_read": rd, "dram_bytes_write": wr, "kernel_seconds_under_ncu": t,
                     "kernel_source_sha256": kernel_source_hash(), "command": a.command,
                     "note": "one launch of k_forces_warp; bench.py reports read + write as roofline.traffic while the kernel sources hash to the value above"}
    with open(TRAFFIC_JSON, "w") as fh:
        json.dump(d, fh, indent=1, sort_keys=True)
        fh.write("\n")
    print(f"{a.workload}: read {rd / 1e9:.2f} GB + write {wr / 1e9:.2f} GB")


def main():
    ap = argparse.ArgumentParser()
    sub = ap.add_subparsers(dest="what", required=True)
    p = sub.add_parser("launches"); p.add_argument("csv"); p.add_argument("out")
    p.add_argument("--title", required=True); p.add_argument("--command", required=True); p.add_argument("--note", default="")
    p = sub.add_parser("full"); p.add_argument("csv"); p.add_argument("out")
    p.add_argument("--title", required=True); p.add_argument("--command", required=True); p.add_argument("--note", default="")
    p.add_argument("--kernel", default="k_forces_warp"); p.add_argument("--index", type=int, default=0)
    p.add_argument("--interactions", type=float, default=0.0)
    p = sub.add_parser("sass"); p.add_argument("out")
    p = sub.add_parser("traffic"); p.add_argument("workload"); p.add_argument("csv"); p.add_argument("--command", required=True)
    a = ap.parse_args()
    {"launches": cmd_launches, "full": cmd_full, "traffic": cmd_traffic, "sass": cmd_sass}[a.what](a)


if __name__ == "__main__":
    sys.exit(main())
