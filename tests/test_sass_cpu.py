"""Properties of the generated machine code that can be checked without a GPU (cuobjdump on the built library):
the lanes kernels really use the copy engine and mbarriers (SASS UBLKCP / SYNCS, B200_PROFILING.md 'what proves a
Blackwell-native kernel'), their hot loops touch no local memory and keep the instruction budgets DESIGN.md 6.5
quotes, and every kernel fits the register file at its block size."""
import collections
import re
import shutil

import pytest

from paper_2511_02328_b200 import build, sass_report

pytestmark = pytest.mark.skipif(shutil.which(sass_report.CUOBJDUMP) is None, reason="cuobjdump not available")


@pytest.fixture(scope="module")
def funcs():
    f = sass_report.functions(build.build())
    names = sass_report.demangle(list(f))
    return {re.sub(r"\(anonymous namespace\)::", "", names[k]): v for k, v in f.items()}


def _kernel(funcs, prefix):
    hits = [k for k in funcs if prefix in k]
    assert len(hits) == 1, (prefix, hits)
    return funcs[hits[0]]


def _ops(instrs):
    return collections.Counter(b.split()[0].split(".")[0] for _, b in instrs)


@pytest.mark.parametrize("kind,adds,max_ipa", [(0, 256, 0.85), (1, 256, 0.45), (2, 128, 1.40)])
def test_lanes_hot_loop_budget(funcs, kind, adds, max_ipa):
    instrs = _kernel(funcs, "ddsp_lanes_kernel<%d," % kind)
    nlds, lo, hi, body = sass_report.hot_loop(instrs)
    assert nlds >= 32, "the two-row loop body holds the shared-memory loads of 2 rows x 4 trials x 4 words"
    assert not any(b.startswith(("LDL", "STL")) for b in body), "local memory in the hot loop"
    assert not any(b.startswith(("LDG", "STG", "RED", "ATOM", "BAR", "SYNCS")) for b in body), "global / barrier work in the hot loop"
    assert len(body) / adds <= max_ipa, (len(body), adds)
    if kind == 0:      # whole-word adds on the FMA pipe, odd bytes on the ALU pipe
        ops = collections.Counter(b.split()[0] for b in body)
        assert ops["LDS.64"] == 32 and ops["PRMT"] == 64 and ops["IADD3"] == 32 and ops["IMAD"] >= 64


def test_lanes_kernels_use_copy_engine_and_mbarriers(funcs):
    for kind in (0, 1, 2):
        ops = _ops(_kernel(funcs, "ddsp_lanes_kernel<%d," % kind))
        assert ops["UBLKCP"] >= 2 and ops["SYNCS"] >= 6, ops          # bulk copies; init / arrive / try_wait
        assert ops["BAR"] <= 1, "one __syncthreads (after barrier init), none in the pipeline"
        assert (ops["REDG"] > 0) == (kind != 2), "integer kinds flush with reductions, float32 stores once"
    for name, instrs in funcs.items():
        if "lanes_kernel" not in name:
            assert _ops(instrs)["UBLKCP"] == 0, name


def test_register_budgets():
    import subprocess
    res = subprocess.run([sass_report.CUOBJDUMP, "-res-usage", build.build()], capture_output=True, text=True, check=True).stdout
    regs = {}
    cur = None
    for ln in res.splitlines():
        m = re.match(r"\s*Function (\S+):", ln)
        if m:
            cur = m.group(1)
        m = re.search(r"REG:(\d+) STACK:(\d+)", ln)
        if m and cur:
            regs[cur] = (int(m.group(1)), int(m.group(2)))
    names = sass_report.demangle(list(regs))
    for k, (r, stack) in regs.items():
        n = names[k]
        if "lanes_kernel" in n or "tiled_u8" in n:
            assert r <= 128, (n, r)                     # 512 threads x 128 registers = the register file
        if "ddsp_lanes_kernel<0" in n:
            assert stack == 0, "the uint8 lanes kernel is spill-free"
