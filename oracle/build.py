"""Build oracle/libovr.so from oracle/ovr.cpp (g++, no CUDA).  TEST INFRASTRUCTURE ONLY.

-ffp-contract=off: only the explicit std::fma calls fuse.
-mfma: std::fma compiles to one vfmadd instruction instead of a libm call.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ovr.cpp")
LIB = os.path.join(HERE, "libovr.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-fno-fast-math", "-fPIC", "-shared",
         "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "ovr.h")]
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["g++", *FLAGS, SRC, "-o", tmp], check=True, cwd=HERE)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
