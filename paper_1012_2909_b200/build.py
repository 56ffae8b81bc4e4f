"""Build paper_1012_2909_b200/libvr.so (the C-ABI library of include/vr.h) with nvcc for sm_100a.

--fmad=false: the kernels spell every fused multiply-add explicitly (__fmaf_rn / fma), nothing
else may be contracted.  No --use_fast_math.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvr.so")
SOURCES = ["vr_api.cu", "vr_cube.cu", "vr_march.cu", "vr_composite.cu", "vr_overlay.cu", "vr_pyramid.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--fmad=false", "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared",
              "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, "vr_internal.cuh"),
                   os.path.join(os.path.dirname(HERE), "include", "vr.h")]
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in deps)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    res = subprocess.run([_nvcc(), *NVCC_FLAGS, *srcs, "-o", tmp], capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libvr.so")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
