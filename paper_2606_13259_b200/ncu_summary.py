"""Summarise one kernel of an `ncu --set full` report as text + JSON under profiles/.

    python -m paper_2606_13259_b200.ncu_summary REPORT.ncu-rep NAME "TITLE" "COMMAND" [--kernel REGEX]

writes profiles/NAME.md (counter table, stall reasons, the command that made the report) and
profiles/NAME.json (the numbers bench.py prints under roofline.traffic / roofline.ncu: nothing
profiler-derived is typed into bench.py by hand).  It reads the report with
`ncu -i REPORT --page raw --csv`; it runs no kernel and needs no GPU.  With `--sass` it also
writes profiles/NAME_sass.md, the opcode histogram of the kernel (executed warp instructions per
opcode from the report's source page).
"""
from __future__ import annotations

import argparse
import collections
import csv
import json
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PROFILES = os.path.join(ROOT, "profiles")

TABLE = [
    "gpu__time_duration.sum", "sm__cycles_elapsed.avg", "sm__cycles_elapsed.avg.per_second",
    "launch__grid_size", "launch__block_size", "launch__registers_per_thread", "launch__shared_mem_per_block_dynamic",
    "dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "lts__t_sector_hit_rate.pct", "lts__throughput.avg.pct_of_peak_sustained_elapsed", "lts__t_sectors_srcunit_tex_op_read.sum",
    "l1tex__throughput.avg.pct_of_peak_sustained_elapsed", "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum",
    "sm__throughput.avg.pct_of_peak_sustained_elapsed", "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_fmaheavy_cycles_active.avg.pct_of_peak_sustained_active", "sm__pipe_xu_cycles_active.avg.pct_of_peak_sustained_active",
    "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "sm__inst_executed_pipe_tmem.avg.pct_of_peak_sustained_active",
    "sm__warps_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
    "smsp__thread_inst_executed_per_inst_executed.ratio", "smsp__inst_executed_op_tma_ld.sum",
]

# the binding roofline is the largest of these utilisation counters (percent of the unit's peak)
UTILISATION = {
    "hbm": "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed",
    "l2": "lts__throughput.avg.pct_of_peak_sustained_elapsed",
    "shared_memory_lsu": "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
    "issue_slots": "smsp__issue_active.avg.pct_of_peak_sustained_active",
    "alu_pipe": "sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active",
    "fma_pipe": "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
    "tensor_pipe": "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active",
}

SCALE = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "Tbyte": 1e12}
TIME = {"ms": 1.0, "us": 1e-3, "ns": 1e-6, "s": 1e3, "second": 1e3, "msecond": 1.0, "usecond": 1e-3, "nsecond": 1e-6}


def _ncu(report, page, extra=()):
    r = subprocess.run(["ncu", "-i", report, "--page", page, "--csv", *extra], capture_output=True, text=True)
    if r.returncode != 0:
        raise SystemExit(f"ncu failed on {report}:\n{r.stderr}")
    return list(csv.reader(r.stdout.splitlines()))


def _num(s):
    try:
        return float(s.replace(",", ""))
    except ValueError:
        return None


def summarise(report, name, title, command, kernel=None, sass=False):
    rows = _ncu(report, "raw")
    hdr, units = rows[0], rows[1]
    body = [r for r in rows[2:] if len(r) == len(hdr)]
    ki = hdr.index("Kernel Name")
    if kernel:
        body = [r for r in body if re.search(kernel, r[ki])]
    if not body:
        raise SystemExit("no kernel in the report matches")
    vals = body[0]
    col = {h: i for i, h in enumerate(hdr)}

    def get(metric):
        if metric not in col:
            return None, None
        return _num(vals[col[metric]]), units[col[metric]]

    def bytes_of(metric):
        v, u = get(metric)
        return None if v is None else v * SCALE.get(u, 1.0)

    t, tu = get("gpu__time_duration.sum")
    rd, wr = bytes_of("dram__bytes_read.sum"), bytes_of("dram__bytes_write.sum")
    out = {
        "kernel": vals[ki], "report": os.path.basename(report), "command": command,
        "gpu_time_ms": None if t is None else t * TIME.get(tu, 1.0),
        "dram_bytes_read": rd, "dram_bytes_write": wr, "dram_bytes": None if rd is None or wr is None else rd + wr,
        "l2_hit_rate_pct": get("lts__t_sector_hit_rate.pct")[0],
        "warp_instructions": get("smsp__inst_executed.sum")[0],
        "sm_clock_ghz": get("sm__cycles_elapsed.avg.per_second")[0],
        "utilisation_pct": {k: get(m)[0] for k, m in UTILISATION.items() if get(m)[0] is not None},
        "note": "captured under ncu (serialised, cold caches): shares and counters, never a bench value",
    }
    stalls = {}
    for h in hdr:
        m = re.match(r"smsp__average_warps_issue_stalled_(.*)_per_issue_active\.ratio$", h)
        if m and "not_issued" not in h:
            v = _num(vals[col[h]])
            if v is not None and v >= 0.05:
                stalls[m.group(1)] = v
    out["stalls_per_issue_active"] = stalls

    os.makedirs(PROFILES, exist_ok=True)
    with open(os.path.join(PROFILES, name + ".json"), "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    with open(os.path.join(PROFILES, name + ".md"), "w") as f:
        f.write(f"# {title}\n\nCommand (under gpurun, one B200, after the same command exited 0 without ncu):\n\n```\n{command}\n```\n\n")
        f.write("Summarised with `python -m paper_2606_13259_b200.ncu_summary` (reads the report with "
                "`ncu -i <report> --page raw --csv`). Numbers under ncu are never bench values.\n\n")
        f.write(f"## {vals[ki]}\n\n| metric | unit | value |\n|---|---|---|\n")
        for m in TABLE:
            if m in col:
                f.write(f"| {m} | {units[col[m]]} | {vals[col[m]]} |\n")
        f.write("\nUtilisation counters (the binding roofline is the largest, SURVEY.md 8(d.4)):\n\n| unit | % of peak |\n|---|---|\n")
        for k, v in sorted(out["utilisation_pct"].items(), key=lambda kv: -kv[1]):
            f.write(f"| {k} | {v:.1f} |\n")
        f.write("\nWarp stall reasons (warps per issue-active cycle):\n\n| stall | ratio |\n|---|---|\n")
        for k, v in sorted(stalls.items(), key=lambda kv: -kv[1]):
            f.write(f"| {k} | {v:.3f} |\n")
    if sass:
        sass_histogram(report, name, vals[ki], command)
    return out


def sass_histogram(report, name, kernel_name, command):
    """Executed warp instructions per SASS opcode (source page of the report, `--import-source on` capture)."""
    rows = _ncu(report, "source", ("--print-source", "sass"))
    h = next(i for i, r in enumerate(rows) if "Source" in r and "Instructions Executed" in r)
    hdr = rows[h]
    si, ei = hdr.index("Source"), hdr.index("Instructions Executed")
    static, dyn = collections.Counter(), collections.Counter()
    for r in rows[h + 1:]:
        if len(r) <= max(si, ei):
            continue
        toks = [t for t in r[si].split() if not t.startswith("@")]
        if not toks:
            continue
        op = toks[0].split(".")[0]
        static[op] += 1
        dyn[op] += int(_num(r[ei]) or 0)
    total = sum(dyn.values()) or 1
    with open(os.path.join(PROFILES, name + "_sass.md"), "w") as f:
        f.write(f"# SASS opcode histogram: {kernel_name}\n\nFrom the source page of the report made by\n\n```\n{command}\n```\n\n")
        f.write("`static` = instructions in the binary, `executed` = warp instructions executed in the captured launch.\n"
                "UTCHMMA = tcgen05.mma, STTM / LDTM = tcgen05.st / ld, UTCBAR = tcgen05.commit, UBLKCP / UTMALDG = TMA bulk / tensor "
                "copies, SYNCS = mbarrier, FFMA2 / FADD2 / FMUL2 = packed FP32x2.\n\n| opcode | static | executed | share |\n|---|---|---|---|\n")
        for op, n in sorted(dyn.items(), key=lambda kv: -kv[1]):
            f.write(f"| {op} | {static[op]} | {n} | {100.0 * n / total:.2f} % |\n")


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("report")
    ap.add_argument("name")
    ap.add_argument("title")
    ap.add_argument("command")
    ap.add_argument("--kernel", default=None, help="regex on the kernel name (default: the first kernel of the report)")
    ap.add_argument("--sass", action="store_true", help="also write the SASS opcode histogram")
    a = ap.parse_args()
    out = summarise(a.report, a.name, a.title, a.command, a.kernel, a.sass)
    print(json.dumps({k: out[k] for k in ("kernel", "gpu_time_ms", "dram_bytes", "l2_hit_rate_pct", "utilisation_pct")}))


if __name__ == "__main__":
    main()
