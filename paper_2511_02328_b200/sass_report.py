"""Opcode histogram of the kernels' hot loops and their resource usage, read from the built library with cuobjdump
(no GPU needed).  The instruction budgets quoted in DESIGN.md section 6 are this report's numbers.

    python -m paper_2511_02328_b200.sass_report > profiles/sass_lanes_r02.md

The hot loop of a kernel is taken to be the innermost loop (a backward branch with no other backward branch
inside its range) that holds the most shared-memory loads.  Argument marshalling and counting only.
"""
import collections
import os
import re
import subprocess
import sys

from . import build as _build

CUOBJDUMP = os.path.join(os.path.dirname(_build._nvcc()), "cuobjdump") if os.path.isabs(_build._nvcc()) else "cuobjdump"
INSTR = re.compile(r"^\s*/\*([0-9a-f]{4,})\*/\s+(.*?);")
# nominal adds per iteration of the two-row loop body: 2 rows x 4 trials x 4 words x lanes per word
ADDS_PER_ITER = {"ddsp_lanes_kernel<0": 2 * 4 * 4 * 8, "ddsp_lanes_kernel<1": 2 * 4 * 4 * 8, "ddsp_lanes_kernel<2": 2 * 4 * 4 * 4,
                 "ddsp_tiled_u8_kernel": 2 * 8 * 4 * 4}
PIPE = [("LSU (shared loads)", r"^LDS"), ("ALU", r"^(IADD3|LOP3|PRMT|SHF|VIADD|ISETP|SEL|LEA|VIMNMX|PLOP3|IADD)\b"),
        ("FMA", r"^(IMAD|FADD|FFMA|FMUL)"), ("branch / sync", r"^(BRA|BSSY|BSYNC|WARPSYNC|SYNCS|NOP)")]


def demangle(names):
    out = subprocess.run(["c++filt"], input="\n".join(names), capture_output=True, text=True).stdout.split("\n")
    return dict(zip(names, out))


def functions(lib):
    text = subprocess.run([CUOBJDUMP, "-sass", lib], capture_output=True, text=True, check=True).stdout
    funcs, cur = {}, None
    for ln in text.splitlines():
        m = re.match(r"\s*Function : (\S+)", ln)
        if m:
            cur = m.group(1)
            funcs[cur] = []
            continue
        m = INSTR.match(ln)
        if m and cur:
            body = re.sub(r"^@!?U?P\d+\s+", "", m.group(2).strip())
            funcs[cur].append((int(m.group(1), 16), body))
    return funcs


def hot_loop(instrs):
    back = []
    for addr, body in instrs:
        m = re.match(r"BRA(?:\.U)?(?:\.ANY)?\s+(?:!?U?P\d+,\s*)?0x([0-9a-f]+)", body)
        if m and int(m.group(1), 16) <= addr:
            back.append((int(m.group(1), 16), addr))
    best = None
    for lo, hi in back:
        if any(l2 >= lo and h2 <= hi and (l2, h2) != (lo, hi) for l2, h2 in back):
            continue                                  # not innermost
        body = [b for a, b in instrs if lo <= a <= hi]
        nlds = sum(b.startswith("LDS") for b in body)
        if best is None or nlds > best[0]:
            best = (nlds, lo, hi, body)
    return best


def main():
    lib = _build.build()
    res = subprocess.run([CUOBJDUMP, "-res-usage", lib], capture_output=True, text=True, check=True).stdout
    funcs = functions(lib)
    names = demangle(list(funcs))
    print("# SASS report of %s (sm_100a)\n" % os.path.basename(lib))
    print("Command: `python -m paper_2511_02328_b200.sass_report` (cuobjdump -sass / -res-usage of the built library).\n")
    print("## Resource usage\n\n| kernel | registers | stack bytes | static shared | instructions |\n|---|---|---|---|---|")
    usage = {}
    cur = None
    for ln in res.splitlines():
        m = re.match(r"\s*Function (\S+):", ln)
        if m:
            cur = m.group(1)
        m = re.search(r"REG:(\d+) STACK:(\d+) SHARED:(\d+)", ln)
        if m and cur:
            usage[cur] = m.groups()
    for f in sorted(funcs, key=lambda f: names[f]):
        u = usage.get(f, ("?", "?", "?"))
        short = re.sub(r"\(anonymous namespace\)::", "", names[f])
        print("| `%s` | %s | %s | %s | %d |" % (short[:90], u[0], u[1], u[2], len(funcs[f])))
    copy_ops = collections.Counter()
    print("\n## Hot loops\n")
    for f in sorted(funcs, key=lambda f: names[f]):
        short = re.sub(r"\(anonymous namespace\)::", "", names[f])
        for b in (b for _, b in funcs[f]):
            op = b.split()[0]
            if op.startswith(("UBLKCP", "SYNCS", "UTMALDG", "LDGSTS", "REDG", "RED")):
                copy_ops[(short.split("(")[0], op.split(".")[0])] += 1
        key = next((k for k in ADDS_PER_ITER if k in short), None)
        if key is None:
            continue
        hl = hot_loop(funcs[f])
        if not hl or hl[0] < 8:
            continue
        nlds, lo, hi, body = hl
        hist = collections.Counter(re.sub(r"\.(U32|MOV|IADD|reuse|LUT)\b", lambda m: m.group(0), b.split()[0]) for b in body)
        adds = ADDS_PER_ITER[key]
        print("### `%s`\n" % short[:100])
        print("Loop 0x%x..0x%x: %d instructions per iteration, %d nominal adds per iteration (two channel rows) = "
              "**%.3f instructions per add**; local-memory accesses in the loop: %d.\n"
              % (lo, hi, len(body), adds, len(body) / adds, sum(b.startswith(("LDL", "STL")) for b in body)))
        print("| opcode | count | per add |\n|---|---|---|")
        for op, n in hist.most_common():
            print("| %s | %d | %.4f |" % (op, n, n / adds))
        print("\n| pipe (by opcode class) | instructions | per add | adds/clk/SM at that pipe's rate |\n|---|---|---|---|")
        for label, pat in PIPE:
            n = sum(bool(re.match(pat, b)) for b in body)
            rate = {"LSU (shared loads)": None, "ALU": 64.0, "FMA": 64.0, "branch / sync": None}[label]
            lim = "%.0f" % (rate * adds / n) if rate and n else "-"
            print("| %s | %d | %.4f | %s |" % (label, n, n / adds, lim))
        print("| all (issue: 128 thread-instr/clk/SM) | %d | %.4f | %.0f |\n" % (len(body), len(body) / adds, 128.0 * adds / len(body)))
    print("## Copy-engine, mbarrier and reduction instructions per kernel\n\n| kernel | opcode | count |\n|---|---|---|")
    for (k, op), n in sorted(copy_ops.items()):
        print("| `%s` | %s | %d |" % (k, op, n))


if __name__ == "__main__":
    main()
