"""Build libddsp.so (the C-ABI library of include/ddsp.h) in-tree with nvcc for sm_100a.

    python -m paper_2511_02328_b200.build [--force] [--verbose] [--define NAME=VALUE ...]

nvcc cross-compiles without a GPU.  The .so lands next to this file so that it travels with the
repository snapshot to the GPU box; it is git-ignored.
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libddsp.so")
SOURCES = ["ddsp_plan.cpp", "ddsp_direct.cu", "ddsp_tiled.cu", "ddsp_lanes.cu"]
HEADERS = [os.path.join(CSRC, "ddsp_internal.h"), os.path.join(_ROOT, "include", "ddsp.h")]
NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math,-fvisibility=hidden",
    "--fmad=false",          # fp32 path must never contract add chains; integer code is unaffected
    "-x", "cu",
]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    deps += [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, defines=()):
    """Compile every CUDA source into libddsp.so; returns its path.  defines: compile-time tuning knobs
    ("NAME=VALUE", see csrc/ddsp_lanes.cu); a build with defines is always redone and is not what ships."""
    if not force and not defines and not _stale():
        return LIB
    objs = []
    bdir = os.path.join(_HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    procs = []
    for s in SOURCES:
        o = os.path.join(bdir, os.path.splitext(s)[0] + ".o")
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-D" + d for d in defines] + \
              ["-c", os.path.join(CSRC, s), "-o", o]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
        objs.append(o)
    for cmd, pr in procs:
        out = pr.communicate()[0].decode()
        if pr.returncode != 0:
            raise RuntimeError("nvcc failed: %s\n%s" % (" ".join(cmd), out))
        if verbose and out:
            sys.stderr.write(out)
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call([_nvcc(), "-shared", "-o", tmp] + objs + ["-cudart", "static"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    defs = [sys.argv[i + 1] for i, a in enumerate(sys.argv[:-1]) if a == "--define"]
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, defines=defs))
