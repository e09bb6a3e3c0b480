"""Summarises an `ncu --set full` report of one kernel launch as text for profiles/ (no GPU needed: it only reads the
.ncu-rep with `ncu -i ... --page raw --csv` / `--page source --csv`).

    python -m paper_1507_00315_b200.ncu_summary REPORT.ncu-rep --instance L20 --terms 17179869184 --label v12 \
        [--md profiles/round2_swar_ncu_L20.md] [--json profiles/ncu_metrics.json] [--commit HASH] [--command "..."]

--terms     sign vectors the profiled launch evaluated (bench.py --profile-chunks N: N x 2^(2n-1-chunk_bits))
--md        appends a markdown section: the metric table, executed thread-instructions per term, the opcode mix and
            the per-section instruction counts from the source page
--json      updates the record bench.py reads for roofline.executed_instr_per_term / issue_frac
"""
from __future__ import annotations

import argparse
import collections
import csv
import io
import json
import os
import subprocess
import sys

METRICS = [
    ("duration", "gpu__time_duration.sum"),
    ("grid", "launch__grid_size"),
    ("block", "launch__block_size"),
    ("registers/thread", "launch__registers_per_thread"),
    ("dynamic smem/block", "launch__shared_mem_per_block_dynamic"),
    ("blocks/SM (reg limit)", "launch__occupancy_limit_registers"),
    ("blocks/SM (smem limit)", "launch__occupancy_limit_shared_mem"),
    ("achieved occupancy %", "sm__warps_active.avg.pct_of_peak_sustained_active"),
    ("issue slots busy %", "smsp__issue_active.avg.pct_of_peak_sustained_active"),
    ("ALU pipe %", "sm__inst_executed_pipe_alu.avg.pct_of_peak_sustained_active"),
    ("FMA pipe (IMAD, IDP) %", "sm__inst_executed_pipe_fma.avg.pct_of_peak_sustained_active"),
    ("FMA-heavy pipe %", "sm__inst_executed_pipe_fmaheavy.avg.pct_of_peak_sustained_active"),
    ("XU pipe (POPC) %", "sm__inst_executed_pipe_xu.avg.pct_of_peak_sustained_active"),
    ("LSU pipe %", "sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active"),
    ("ADU pipe %", "sm__inst_executed_pipe_adu.avg.pct_of_peak_sustained_active"),
    ("uniform pipe %", "sm__inst_executed_pipe_uniform.avg.pct_of_peak_sustained_active"),
    ("CBU (branch) pipe %", "sm__inst_executed_pipe_cbu.avg.pct_of_peak_sustained_active"),
    ("warp instructions executed", "smsp__inst_executed.sum"),
    ("active threads per warp instruction", "smsp__thread_inst_executed_per_inst_executed.ratio"),
    ("shared store wavefronts", "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_st.sum"),
    ("shared load wavefronts", "l1tex__data_pipe_lsu_wavefronts_mem_shared_op_ld.sum"),
    ("shared bank conflicts", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum"),
    ("DRAM read", "dram__bytes_read.sum"),
    ("DRAM write", "dram__bytes_write.sum"),
]
STALLS = ["not_selected", "math_pipe_throttle", "wait", "short_scoreboard", "barrier", "dispatch_stall", "no_instruction",
          "branch_resolving", "long_scoreboard", "mio_throttle"]


def ncu_csv(rep: str, page: str):
    out = subprocess.run(["ncu", "-i", rep, "--page", page, "--csv"], capture_output=True, text=True)
    if out.returncode != 0:
        raise SystemExit("ncu -i failed: " + out.stderr[-400:])
    return list(csv.reader(io.StringIO(out.stdout)))


def raw_metrics(rep: str):
    rows = ncu_csv(rep, "raw")
    hdr, units, vals = rows[0], rows[1], rows[2]
    return {h: (vals[i], units[i]) for i, h in enumerate(hdr)}


def to_float(s: str) -> float:
    return float(s.replace(",", "")) if s not in ("", "n/a") else float("nan")


def bytes_of(value: str, unit: str) -> float:
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(unit, 1.0)
    return to_float(value) * scale


def source_breakdown(rep: str, terms: float, steps_per_block: int = 32):
    """Executed warp-instructions per 32-step block, by how often an instruction runs per block (exactly 1 = the
    unrolled walk, zero mask and slot plan; another rate above 0.3 = the drain loops, whose rounds depend on the data;
    rarely = outer flips, prefix init, tail) and by opcode."""
    rows = ncu_csv(rep, "source")
    hdr = rows[1]
    idx = {h: i for i, h in enumerate(hdr)}
    blocks = terms / 32 / steps_per_block
    sect = collections.defaultdict(lambda: [0, 0.0])
    ops = collections.Counter()
    for r in rows[2:]:
        if len(r) < len(hdr):
            continue
        ex = int(r[idx["Instructions Executed"]])
        src = r[idx["Source"]].strip().split()
        op = (src[1] if src[0].startswith("@") else src[0]).split(".")[0]
        ratio = ex / blocks
        key = "once per block (walk, zero mask, slot plan)" if abs(ratio - 1) < 1e-9 else (
            "loops inside a block (drain rounds)" if ratio > 0.3 else "rarely (outer flips, prefix init, tail)")
        sect[key][0] += 1
        sect[key][1] += ex * 32 / terms
        ops[op] += ex * 32 / terms
    return dict(sect), ops


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(prog="python -m paper_1507_00315_b200.ncu_summary")
    ap.add_argument("report")
    ap.add_argument("--instance", required=True, help="S<n> or L<n>, e.g. L20")
    ap.add_argument("--terms", type=float, required=True)
    ap.add_argument("--label", default="")
    ap.add_argument("--commit", default=None)
    ap.add_argument("--command", default=None, help="the command line that produced the report (recorded in the .md)")
    ap.add_argument("--md", default=None)
    ap.add_argument("--json", default=None)
    a = ap.parse_args(argv)

    m = raw_metrics(a.report)
    inst = to_float(m["smsp__inst_executed.sum"][0])
    per_term = inst * 32 / a.terms
    issue = to_float(m["smsp__issue_active.avg.pct_of_peak_sustained_active"][0])
    dram = bytes_of(*m["dram__bytes_read.sum"]) + bytes_of(*m["dram__bytes_write.sum"])
    lines = ["## %s %s" % (a.instance, a.label), ""]
    if a.command:
        lines += ["Command: `%s`" % a.command, ""]
    if a.commit:
        lines += ["Commit: %s.  Sign vectors in the profiled launch: %d." % (a.commit, a.terms), ""]
    lines += ["| metric | value |", "|---|---|"]
    for name, key in METRICS:
        if key in m:
            lines.append("| %s (`%s`) | %s %s |" % (name, key, m[key][0], m[key][1]))
    for s in STALLS:
        key = "smsp__average_warps_issue_stalled_%s_per_issue_active.ratio" % s
        if key in m:
            lines.append("| stall: %s (`%s`) | %s |" % (s, key, m[key][0]))
    lines += ["", "Executed thread-instructions per term: %.2f (`smsp__inst_executed.sum` x 32 / terms); issue slots busy %.1f %%; "
              "DRAM traffic %.0f bytes per launch." % (per_term, issue, dram), ""]
    sect, ops = source_breakdown(a.report, a.terms)
    lines += ["| part (source page, by executions per 32-step block) | SASS instructions | executed per term |", "|---|---|---|"]
    for k, (cnt, v) in sorted(sect.items(), key=lambda kv: -kv[1][1]):
        lines.append("| %s | %d | %.2f |" % (k, cnt, v))
    lines += ["", "Opcode mix per term: " + ", ".join("%s %.2f" % (o, c) for o, c in ops.most_common(18)) + ".", ""]
    text = "\n".join(lines)
    print(text)
    if a.md:
        with open(a.md, "a") as f:
            f.write(text + "\n")
    if a.json:
        try:
            with open(a.json) as f:
                doc = json.load(f)
        except (OSError, ValueError):
            doc = {"note": "written by python -m paper_1507_00315_b200.ncu_summary from ncu --set full captures; read by bench.py",
                   "instances": {}}
        doc["instances"][a.instance] = dict(
            kernel="swar_kernel<%d,%s>" % (0 if a.instance[0] == "S" else 1, a.instance[1:]), label=a.label, commit=a.commit,
            inst_executed_warp=inst, terms=a.terms, instr_per_term=per_term, issue_active_pct=issue,
            dram_bytes_per_launch=dram, registers=int(to_float(m["launch__registers_per_thread"][0])),
            duration_ms=to_float(m["gpu__time_duration.sum"][0]) * {"ms": 1.0, "us": 1e-3, "s": 1e3, "ns": 1e-6}.get(m["gpu__time_duration.sum"][1], 1.0),
            source=os.path.relpath(a.md, os.path.dirname(os.path.dirname(os.path.abspath(a.json)))) if a.md else None)
        with open(a.json, "w") as f:
            json.dump(doc, f, indent=1, sort_keys=True)
            f.write("\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
