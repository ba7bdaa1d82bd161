"""Build the C-ABI CUDA library in-tree for sm_100a.

    python -m paper_2606_14480_b200.build [--force]

nvcc cross-compiles without a GPU.  -fmad=false: no multiply-add contraction, every float operation
rounds once in source order.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblhcb_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
         "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) + \
        [os.path.join(HERE, "..", "include", "lhcb.h")]


def build(force: bool = False, verbose: bool = False, stage_clocks: bool = False, checked: bool = False) -> str:
    """Compile the library (if the sources are newer).  Two diagnostic variants, never used by the timed path:
    stage_clocks=True builds liblhcb_b200_clk.so (-DLHCB_STAGE_CLOCKS: per-stage cycle counters read by
    lhcb_debug_stage_clocks; `bench.py --stage-clocks`); checked=True builds liblhcb_b200_chk.so (-DLHCB_CHECKED:
    index checks on the shared-memory queues, tables and searches, read by lhcb_debug_checks;
    tests/test_gpu_checked.py)."""
    lib, extra = LIB, []
    if stage_clocks:
        lib, extra = LIB.replace(".so", "_clk.so"), ["-DLHCB_STAGE_CLOCKS"]
    elif checked:
        lib, extra = LIB.replace(".so", "_chk.so"), ["-DLHCB_CHECKED"]
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in _deps()):
        return lib
    cmd = [NVCC, *FLAGS, *extra, *sources(), "-o", lib]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
