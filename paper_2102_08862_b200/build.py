"""In-tree build of the CUDA library (nvcc, sm_100a only) and of the input generator (g++)."""
from __future__ import annotations

import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(CSRC, "libtpctracker.so")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")

# --fmad=false: every decision is taken on fp32 values rounded operation by operation (BASELINE.json L5);
# default -prec-div=true -prec-sqrt=true -ftz=false are kept; never --use_fast_math.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--fmad=false", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(INCLUDE, "*.h")))


def build_cuda(force: bool = False, verbose: bool = False) -> str:
    """Compile ``csrc/tpc_tracker.cu`` into ``csrc/libtpctracker.so`` if missing or stale."""
    newest = max(os.path.getmtime(p) for p in _sources())
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("TPC_NVCC_EXTRA", "").split()      # build-time knobs (-DTPC_...); default: none
        cmd = [nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
               os.path.join(CSRC, "tpc_tracker.cu")]
        subprocess.check_call(cmd)
    return LIB


def build_all(force: bool = False) -> None:
    from . import gen
    gen.build(force)
    build_cuda(force)
