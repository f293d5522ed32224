"""Turn an Nsight Compute raw page into the text summary kept under profiles/ and into the entry of
profiles/traffic.json that bench.py reports as roofline.traffic.

    ncu -i gpurun_out/prof.ncu-rep --page raw --csv > raw.csv
    python -m paper_2511_02328_b200.ncu_summary raw.csv --match lanes_kernel --kernel lanes --config fast \
        --command "<the full ncu command that made the report>" --md profiles/ncu_lanes_fast.md \
        --traffic profiles/traffic.json

Argument marshalling and table formatting only: every number is copied from the report; derived figures
(per-launch means, dram bytes = read + write, instructions per add) are labelled as derived.
"""
import argparse
import csv
import json
import os
import re
import sys

# metric -> label; any that the report lacks are skipped
METRICS = [
    ("gpu__time_duration.sum", "duration"),
    ("dram__bytes_read.sum", "dram bytes read"),
    ("dram__bytes_write.sum", "dram bytes written"),
    ("lts__t_bytes.sum", "L2 bytes"),
    ("launch__registers_per_thread", "registers / thread"),
    ("launch__grid_size", "grid"),
    ("launch__block_size", "block"),
    ("sm__cycles_elapsed.max", "SM cycles (max)"),
    ("smsp__cycles_active.avg", "SMSP cycles active (avg)"),
    ("sm__inst_executed.sum", "warp instructions executed"),
    ("smsp__thread_inst_executed.sum", "thread instructions executed"),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots busy %"),
    ("sm__inst_executed_pipe_alu.sum", "ALU pipe warp instr"),
    ("sm__inst_executed_pipe_fma.sum", "FMA pipe warp instr"),
    ("sm__inst_executed_pipe_lsu.sum", "LSU pipe warp instr"),
    ("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", "ALU pipe busy %"),
    ("sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active", "FMA pipe busy %"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "shared-memory wavefronts"),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed", "shared-memory wavefronts % of peak"),
    ("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "shared-memory bank conflicts"),
    ("smsp__inst_executed_op_local_ld.sum", "local loads (spills)"),
    ("smsp__inst_executed_op_local_st.sum", "local stores (spills)"),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "achieved occupancy %"),
]
STALL = re.compile(r"smsp__average_warps?_issue_stalled_(\w+?)_per_issue_active\.ratio|"
                   r"smsp__average_warp_latency_issue_stalled_(\w+?)\.ratio|"
                   r"smsp__warp_issue_stalled_(\w+?)_per_warp_active\.pct")


def to_float(s):
    try:
        return float(s.replace(",", ""))
    except (ValueError, AttributeError):
        return None


def read_raw(path):
    rows = list(csv.reader(open(path, newline="")))
    rows = [r for r in rows if r and not r[0].startswith("==")]
    header = rows[0]
    body = rows[1:]
    units = {}
    if body and (body[0][0] == "" or not body[0][0].strip().isdigit()):
        units = dict(zip(header, body[0]))
        body = body[1:]
    return header, units, [dict(zip(header, r)) for r in body]


def scale_to_base(value, unit):
    """ncu prints bytes / time with unit prefixes; bring them to bytes and seconds."""
    if value is None:
        return None
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12,
            "nsecond": 1e-9, "usecond": 1e-6, "msecond": 1e-3, "second": 1.0, "ns": 1e-9, "us": 1e-6, "ms": 1e-3, "s": 1.0}
    return value * mult.get(unit, 1.0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("raw_csv")
    ap.add_argument("--match", required=True, help="regex on the kernel name: the launches to summarise")
    ap.add_argument("--kernel", required=True, help="kernel name as bench.py reports it (direct / tiled / lanes)")
    ap.add_argument("--config", required=True, help="workload name (tiny / fast / wide / lowfreq / rfids)")
    ap.add_argument("--command", required=True, help="the full command that made the report")
    ap.add_argument("--adds-per-launch", type=float, default=None, help="nominal adds of one launch (for instr/add)")
    ap.add_argument("--md", default=None)
    ap.add_argument("--traffic", default=None)
    a = ap.parse_args()

    header, units, launches = read_raw(a.raw_csv)
    name_col = "Kernel Name" if "Kernel Name" in header else next(h for h in header if "ernel" in h)
    sel = [r for r in launches if re.search(a.match, r[name_col])]
    if not sel:
        sys.exit("no launch matches %r (kernels: %s)" % (a.match, sorted({r[name_col][:60] for r in launches})))

    def mean(metric):
        vals = [scale_to_base(to_float(r.get(metric)), units.get(metric, "")) for r in sel]
        vals = [v for v in vals if v is not None]
        return sum(vals) / len(vals) if vals else None

    lines = ["# ncu summary: kernel `%s`, workload `%s`" % (a.kernel, a.config), "",
             "Command: `%s`" % a.command, "",
             "Launches matched by `%s`: %d (kernel name: `%s`).  Values are means over those launches, copied from "
             "the report's raw page." % (a.match, len(sel), sel[0][name_col][:120]), "",
             "| metric | value | unit |", "|---|---|---|"]
    got = {}
    for metric, label in METRICS:
        v = mean(metric)
        if v is not None:
            got[metric] = v
            lines.append("| %s (`%s`) | %.6g | %s |" % (label, metric, v, units.get(metric, "")))
    stalls = []
    for h in header:
        m = STALL.match(h)
        if m:
            v = mean(h)
            if v:
                stalls.append((v, next(g for g in m.groups() if g), h))
    if stalls:
        lines += ["", "Stall reasons (largest first):", "", "| reason | value | metric |", "|---|---|---|"]
        for v, why, h in sorted(stalls, reverse=True)[:12]:
            lines.append("| %s | %.4g | `%s` |" % (why, v, h))
    rd, wr = got.get("dram__bytes_read.sum"), got.get("dram__bytes_write.sum")
    lines += ["", "Derived:", ""]
    if rd is not None and wr is not None:
        lines.append("- dram bytes per launch = read + write = %.6g" % (rd + wr))
    ti = got.get("smsp__thread_inst_executed.sum")
    if ti and a.adds_per_launch:
        lines.append("- executed thread instructions per nominal add = %.4f" % (ti / a.adds_per_launch))
    dur = got.get("gpu__time_duration.sum")
    if dur and a.adds_per_launch:
        lines.append("- nominal adds per second under the profiler (cold cache, serialised; NOT a bench value) = %.4g"
                     % (a.adds_per_launch / dur))
    text = "\n".join(lines) + "\n"
    if a.md:
        with open(a.md, "w") as f:
            f.write(text)
    else:
        sys.stdout.write(text)
    if a.traffic and rd is not None and wr is not None:
        table = {}
        if os.path.exists(a.traffic):
            table = json.load(open(a.traffic))
        table["%s/%s" % (a.kernel, a.config)] = {"dram_bytes_per_launch": rd + wr, "launches": len(sel),
                                                 "source": os.path.basename(a.md) if a.md else a.raw_csv,
                                                 "command": a.command}
        with open(a.traffic, "w") as f:
            json.dump(table, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
