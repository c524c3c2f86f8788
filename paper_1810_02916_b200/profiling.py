"""Turns ncu output into the text summaries kept under profiles/ (no arithmetic of the method).

    python -m paper_1810_02916_b200.profiling launches <ncu.csv> <out.md> --title T --command C
        per-kernel table of an `ncu --metrics gpu__time_duration.sum --csv` launch list
    python -m paper_1810_02916_b200.profiling full <raw.csv> <out.md> --title T --command C [--kernel REGEX] [--interactions I]
        the counters DESIGN.md quotes, from `ncu -i x.ncu-rep --page raw --csv`
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
    p = sub.add_parser("traffic"); p.add_argument("workload"); p.add_argument("csv"); p.add_argument("--command", required=True)
    a = ap.parse_args()
    {"launches": cmd_launches, "full": cmd_full, "traffic": cmd_traffic}[a.what](a)


if __name__ == "__main__":
    sys.exit(main())
