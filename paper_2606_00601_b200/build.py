"""Builds libaffinescan.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_00601_b200.build [--force] [--verbose]

AFFINESCAN_NVCC_FLAGS (environment) is appended to the compile flags: the kernels' compile-time tuning
knobs (-DLR_PD=, -DLR_MIX_STAGES=, -DLR_TC=, -DLR_MIX_ORDER=; defaults in csrc/) for ablation builds.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG_DIR)
CSRC = os.path.join(PKG_DIR, "csrc")
LIB_PATH = os.path.join(PKG_DIR, "libaffinescan.so")
SOURCES = [os.path.join(CSRC, n) for n in
           ("affinescan_api.cu", "affinescan_affine.cu", "affinescan_selective.cu",
            "affinescan_bwd.cu", "affinescan_static_scratch.cu")]
NVCC_COMPILE_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC,-fvisibility=hidden",
]
NVCC_LINK_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-cudart", "static", "-shared", "-Xcompiler", "-fPIC,-fvisibility=hidden",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found (set NVCC=/path/to/nvcc)")


def _deps():
    deps = [os.path.join(ROOT, "include", "affinescan.h"), os.path.abspath(__file__)]
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            deps.append(os.path.join(CSRC, name))
    return deps


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    built = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(d) > built for d in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA extension if it is missing or older than its sources."""
    if not force and not is_stale():
        return LIB_PATH
    from concurrent.futures import ThreadPoolExecutor
    nvcc = _nvcc()
    objdir = os.path.join(PKG_DIR, "build", f"obj{os.getpid()}")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src) + ".o")
        cmd = [nvcc, *NVCC_COMPILE_FLAGS, *os.environ.get("AFFINESCAN_NVCC_FLAGS", "").split(),
               "-I", os.path.join(ROOT, "include"), "-c", "-o", obj, src]
        if verbose:
            cmd[1:1] = ["-Xptxas", "-v"]
            print(" ".join(cmd), file=sys.stderr)
        subprocess.check_call(cmd)
        return obj

    try:
        with ThreadPoolExecutor(len(SOURCES)) as pool:   # one nvcc per translation unit
            objs = list(pool.map(compile_one, SOURCES))
        tmp = LIB_PATH + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc, *NVCC_LINK_FLAGS, "-o", tmp, *objs])
        os.replace(tmp, LIB_PATH)
    finally:
        shutil.rmtree(objdir, ignore_errors=True)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
