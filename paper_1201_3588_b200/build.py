"""In-tree build of the C-ABI library (csrc/mcrt.cu -> libmcrt.so) for sm_100a.

`python -m paper_1201_3588_b200.build` or `build_library()`.  nvcc cross-compiles without a
GPU; the built .so travels with the source tree and is never installed elsewhere.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB_PATH = os.path.join(_HERE, "libmcrt.so")
CHECKS_LIB_PATH = os.path.join(_HERE, "libmcrt_checks.so")      # same sources with -DMCRT_CHECKS

# -fmad=false: no implicit contraction of a*b+c into FMA.  Which products the compiler fuses differs from one
# template instance of the transport kernel to the next (it did between the swept and the unswept instance:
# one crossing in 2.3e8), and every knob of the library promises bit-identical results; the fused operations
# the kernels want are written as fmaf().
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
              "-Xcompiler", "-fPIC", "-shared"]


def _sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC)
                  if f.endswith((".cu", ".cuh", ".h"))) + [os.path.join(INCLUDE, "mcrt.h"), os.path.join(INCLUDE, "mcrt_dev.h")]


def needs_build(path: str = LIB_PATH) -> bool:
    if not os.path.exists(path):
        return True
    t = os.path.getmtime(path)
    return any(os.path.getmtime(s) > t for s in _sources())


def build_library(force: bool = False, verbose: bool = False, checks: bool = False) -> str:
    out = CHECKS_LIB_PATH if checks else LIB_PATH
    if not force and not needs_build(out):
        return out
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = out + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-DMCRT_CHECKS"] if checks else []) + \
        ["-I", INCLUDE, "-o", tmp, os.path.join(CSRC, "mcrt.cu")]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.check_call(cmd)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose=True))
