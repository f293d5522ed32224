"""Build the CPU emulation of the library's kernels (test infrastructure; see tests/test_emulated_cpu.py).

The product sources (ddsp_plan.cpp and every .cu) are compiled UNCHANGED except for three textual
substitutions that g++ cannot do without: the `<<<...>>>` launch becomes a call of emu_launch, the
`extern __shared__` array becomes a pointer to the emulated CTA's buffer, and the include of the PTX helper
header (ddsp_dev.cuh) is redirected to its host stand-in (emu_common.h).  <cuda_runtime.h> resolves to the
fake one here.

    python tests/emu/build_emu.py [--tsan]   ->  tests/emu/build/libddsp_emu.so  (or emu_tsan, an executable)
"""
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2511_02328_b200", "csrc")
BUILD = os.path.join(HERE, "build")
PRODUCT = ["ddsp_plan.cpp", "ddsp_lanes.cu", "ddsp_tiled.cu", "ddsp_direct.cu"]
LIB = os.path.join(BUILD, "libddsp_emu.so")
TSAN_EXE = os.path.join(BUILD, "emu_tsan")


def transform(text):
    # kernels without shared memory or barriers (the interleave pass): CUDA threads run one after another
    text, n0 = re.subn(r"(kPreKernels\[[^\]]*\])<<<\s*([^;]*?)\s*>>>\(", r"emu_launch_v(\1, \2, ", text)
    text, n1 = re.subn(r"(\w[\w\[\]\.]*)<<<\s*([^;]*?)\s*>>>\((\w+)\);", r"emu_launch(\1, \2, \3);", text)
    n1 += n0
    # launches with an argument list (template kernels of ddsp_direct.cu)
    text, n1b = re.subn(r"(\w+<[^;<>]*>)<<<\s*([^;]*?)\s*>>>\(", r"emu_launch_v(\1, \2, ", text)
    n1 += n1b
    text, n2 = re.subn(r"extern __shared__ __align__\(\d+\) uint8_t smem\[\];", "uint8_t* const smem = emu::smem();", text)
    text = text.replace('#include "ddsp_dev.cuh"', '#include "emu_common.h"')
    return text, n1, n2


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(tsan=False, mutate=None, defines=()):
    """mutate = (name, old, new): build emu_tsan_<name> with `old` replaced by `new` in the kernel sources --
    a deliberately broken protocol, to show that the race check can fail (negative control)."""
    os.makedirs(BUILD, exist_ok=True)
    target = TSAN_EXE if tsan else LIB
    if defines:         # a tuning-knob build (csrc/ddsp_lanes.cu): its own library
        assert not tsan and not mutate
        target = LIB.replace(".so", "_" + "_".join(d.replace("=", "") for d in defines) + ".so")
    if mutate:
        assert tsan
        target = TSAN_EXE + "_" + mutate[0]
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + \
           [os.path.join(HERE, f) for f in os.listdir(HERE) if f.endswith((".h", ".cpp", ".py"))]
    if not _stale(target, deps):
        return target
    srcs = []
    for name in PRODUCT:
        text, n1, n2 = transform(open(os.path.join(CSRC, name)).read())
        tag = "_emu"
        if mutate:
            tag = "_emu_" + mutate[0]
            if name == mutate[3]:
                assert text.count(mutate[1]) == 1, (name, mutate[1])
                text = text.replace(mutate[1], mutate[2])
        if name.endswith(".cu"):
            assert n1 >= 1 and (n2 >= 1 or name == "ddsp_direct.cu"), (name, n1, n2)
        out = os.path.join(BUILD, os.path.splitext(name)[0] + tag + ".cpp")
        with open(out, "w") as f:
            f.write(text)
        srcs.append(out)
    srcs += [os.path.join(HERE, "emu_runtime.cpp")]
    flags = ["-std=c++17", "-O1", "-g", "-fPIC", "-pthread", "-ffp-contract=off", "-fno-fast-math", "-w", "-DDDSP_TESTING"] + ["-D" + d for d in defines] + [
             "-I", HERE, "-I", CSRC, "-I", os.path.join(ROOT, "include")]
    if tsan:
        cmd = ["g++"] + flags + ["-fsanitize=thread"] + srcs + [os.path.join(HERE, "emu_tsan_main.cpp"), "-o", target]
    else:
        cmd = ["g++"] + flags + ["-shared"] + srcs + ["-o", target]
    subprocess.check_call(cmd)
    return target


if __name__ == "__main__":
    print(build(tsan="--tsan" in sys.argv))
