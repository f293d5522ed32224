"""Per-SM issue-rate and shared-memory microbenchmark (csrc/ubench_pipes.cu): the measurement behind the
roofline denominator P_add of DESIGN.md section 6.6.

    python -m paper_2511_02328_b200.ubench [--build-only]      # prints one markdown table; needs a B200

Built in-tree with nvcc for sm_100a (cross-compiles without a GPU).  The table that bench.py's `peak_source`
refers to is the output of this command, kept under profiles/ with the command line beside it.
"""
import os
import subprocess
import sys

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "ubench_pipes.cu")
EXE = os.path.join(_HERE, "build", "ubench_pipes")


def build(force=False):
    os.makedirs(os.path.dirname(EXE), exist_ok=True)
    if not force and os.path.exists(EXE) and os.path.getmtime(EXE) >= os.path.getmtime(SRC):
        return EXE
    subprocess.check_call([_build._nvcc(), "-std=c++17", "-O3", "-lineinfo", "-gencode",
                           "arch=compute_100a,code=sm_100a", "-o", EXE, SRC])
    return EXE


if __name__ == "__main__":
    exe = build()
    if "--build-only" not in sys.argv:
        sys.exit(subprocess.call([exe]))
