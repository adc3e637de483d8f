"""Build step: nvcc -> paper_2607_03627_b200/libuc_pdhg.so (sm_100a only, in-tree so it ships with gpurun)."""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# UC_PDHG_LIB: load another build of the same sources instead (e.g. the -DUC_DEBUG_BOUNDS build for a checking run of
# the GPU tests); it is never built or rebuilt from here
LIB = os.environ.get("UC_PDHG_LIB") or os.path.join(HERE, "libuc_pdhg.so")
SOURCES = [os.path.join(CSRC, "uc_pdhg.cu")]
# everything the translation unit includes: every file under csrc/ plus the public header (a new .cuh is picked up
# without editing this list -- a stale library would let the GPU tests pass against old kernels)
DEPENDS = sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.hpp"))
                 + glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h")))
NVCC_FLAGS = ["-O3", "-std=c++17", "-fmad=false", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def stale() -> bool:
    if os.environ.get("UC_PDHG_LIB"):
        return False
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA extension if it is missing or older than its sources; returns the .so path."""
    if (force and not os.environ.get("UC_PDHG_LIB")) or stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *SOURCES]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
