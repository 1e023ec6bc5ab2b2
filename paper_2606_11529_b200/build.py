"""Build libxpr.so (the C-ABI CUDA library, include/xpr.h) in-tree for sm_100a.

    python -m paper_2606_11529_b200.build [--force]

nvcc cross-compiles without a GPU.  project.cu and ray.cu are compiled with -fmad=false (rule R1 of
DESIGN.md: no FMA contraction in anything that feeds depth bits, rectangles or tile counts).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libxpr.so")
OBJ_DIR = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

COMMON = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
          "-Xcompiler", "-fPIC,-ffp-contract=off", "-I", os.path.join(ROOT, "include"), "-I", CSRC]
COMMON += os.environ.get("XPR_NVCC_FLAGS", "").split()   # e.g. -DXPR_PBWD_MINB=3 for tuning experiments
SOURCES = {
    "api.cu": [],
    "project.cu": ["-fmad=false"],
    "binsort.cu": [],
    "rasterize.cu": [],
    "ray.cu": ["-fmad=false"],
    "rasterize_ray.cu": [],
    "rasterize_feat.cu": [],
    "rasterize_lin.cu": [],
}


def _newer(target: str, deps: list) -> bool:
    return os.path.exists(target) and all(os.path.getmtime(target) >= os.path.getmtime(d) for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ_DIR, exist_ok=True)
    headers = [os.path.join(CSRC, "common.cuh"), os.path.join(ROOT, "include", "xpr.h"), os.path.abspath(__file__)]
    objs = []
    procs = []
    for src, extra in SOURCES.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ_DIR, src.replace(".cu", ".o"))
        objs.append(o)
        if force or not _newer(o, [s] + headers):
            cmd = [NVCC, *COMMON, *extra, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if force or procs or not _newer(OUT, objs):
        # the CUDA runtime is linked dynamically (libcudart.so.12: the one PyTorch has already loaded, else the
        # toolkit's through the rpath), so the library carries no runtime entry points it never calls
        cmd = [NVCC, "-shared", "-o", OUT, *objs, "-cudart", "shared", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
        subprocess.run(cmd, check=True)
    return OUT


CUBCMP_OUT = os.path.join(HERE, "libxpr_cubcmp.so")


def build_cub_compare(force: bool = False) -> str:
    """libxpr_cubcmp.so: cub::DeviceRadixSort::SortPairs behind one C function, for `bench.py --sort-compare` only
    (BASELINE.json:north_star: "CUB is timed only as a comparison").  Never linked into or loaded by libxpr.so."""
    src = os.path.join(CSRC, "cub_compare.cu")
    if force or not _newer(CUBCMP_OUT, [src, os.path.abspath(__file__)]):
        cmd = [NVCC, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
               "-shared", "-o", CUBCMP_OUT, src, "-cudart", "shared", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]
        subprocess.run(cmd, check=True)
    return CUBCMP_OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--cub-compare" in sys.argv:
        print(build_cub_compare(force="--force" in sys.argv))
