"""Build the CPU oracle (TEST INFRASTRUCTURE) as two shared libraries: f32 spec mode and f64.

    python -m oracle.build

-O2, no -ffast-math, -ffp-contract=off: every float operation rounds once, in source order.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.c")
FLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall", "-Wno-unused-function"]


def lib_path(mode: str) -> str:
    return os.path.join(HERE, f"liboracle_{mode}.so")


def build(force: bool = False) -> None:
    for mode, real in (("f32", "float"), ("f64", "double")):
        out = lib_path(mode)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
            continue
        subprocess.check_call(["gcc", *FLAGS, f"-DREAL={real}", SRC, "-o", out, "-lm"])


if __name__ == "__main__":
    build(force=True)
    print("built", lib_path("f32"), lib_path("f64"))
