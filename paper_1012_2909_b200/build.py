"""Build paper_1012_2909_b200/libvr.so (the C-ABI library of include/vr.h) with nvcc for sm_100a.

--fmad=false: the kernels spell every fused multiply-add explicitly (__fmaf_rn / fma), nothing
else may be contracted.  No --use_fast_math.

Every .cu is compiled to its own object (in parallel, only if it or a header changed), then the
objects are linked into the shared library.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_obj")
LIB = os.path.join(HERE, "libvr.so")
SOURCES = ["vr_api.cu", "vr_cube.cu", "vr_march.cu", "vr_march_h.cu", "vr_setup.cu", "vr_touch.cu", "vr_mip_tiles.cu",
           "vr_composite.cu", "vr_composite_static.cu", "vr_overlay.cu", "vr_pyramid.cu"]
HEADERS = [os.path.join(CSRC, "vr_internal.cuh"), os.path.join(CSRC, "vr_sample.cuh"), os.path.join(CSRC, "vr_march.cuh"), os.path.join(CSRC, "vr_async.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "vr.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--fmad=false", "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-Xptxas", "-v"]


def _flags():
    """NVCC_FLAGS plus VR_NVCC_EXTRA from the environment (-D switches of A/B builds, e.g. "-DVR_LIST_CAP=128")."""
    return NVCC_FLAGS + os.environ.get("VR_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _sources():
    return [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = _sources()
    headers = [h for h in HEADERS if os.path.exists(h)]
    hdr_time = max(os.path.getmtime(h) for h in headers + [os.path.abspath(__file__)])
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    stale = []
    for s in srcs:
        src, obj = os.path.join(CSRC, s), os.path.join(OBJ, s[:-3] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_time):
            stale.append((src, obj))
    objs = [os.path.join(OBJ, s[:-3] + ".o") for s in srcs]
    if not stale and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(o) for o in objs):
        return LIB

    def compile_one(job):
        src, obj = job
        tmp = obj + f".tmp{os.getpid()}"
        res = subprocess.run([nvcc, *_flags(), "-c", src, "-o", tmp], capture_output=True, text=True)
        if res.returncode == 0:
            os.replace(tmp, obj)
            with open(obj[:-2] + ".log", "w") as f:        # ptxas -v: registers, spills, shared memory
                f.write(res.stdout + res.stderr)
        return src, res

    with ThreadPoolExecutor(max_workers=max(1, min(len(stale), os.cpu_count() or 1))) as pool:
        results = list(pool.map(compile_one, stale))
    failed = False
    for src, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(f"---- {os.path.basename(src)}\n" + res.stdout + res.stderr)
        failed |= res.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libvr.so")
    tmp = LIB + f".tmp{os.getpid()}"
    res = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *objs, "-o", tmp],
                         capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libvr.so")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
