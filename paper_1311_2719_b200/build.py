"""Build the CUDA library in-tree: paper_1311_2719_b200/liblqcd_b200.so (sm_100a only)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "liblqcd_b200.so")
SOURCES = [os.path.join(CSRC, "lqcd_api.cu"), os.path.join(CSRC, "lqcd_slab.cu"), os.path.join(CSRC, "lqcd_noalloc.cu")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17", "--threads", "3",   # the three translation units compile side by side
    "-Xcompiler", "-fPIC", "-shared",
    "-I", os.path.join(ROOT, "include"),
]


def _deps():
    out = [os.path.join(ROOT, "include", "lqcd.h"), os.path.join(ROOT, "include", "lqcd_slab.h"),
           os.path.join(ROOT, "include", "lqcd_noalloc.h"), os.path.abspath(__file__)]
    for f in os.listdir(CSRC):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    """Compile if the library is missing or older than any source.  Returns the .so path."""
    stale = force or not os.path.exists(SO) or any(os.path.getmtime(d) > os.path.getmtime(SO) for d in _deps())
    if stale:
        tmp = SO + ".tmp%d" % os.getpid()
        cmd = [nvcc(), *NVCC_FLAGS, *extra, "-o", tmp, *SOURCES]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
            print(" ".join(cmd), file=sys.stderr)
        subprocess.check_call(cmd)
        os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
