"""Builds libhclooc_b200.so in-tree with nvcc for sm_100a (no JIT cache, no pip install).

`python -m paper_1808_05056_b200.build` or `build()`; the library is rebuilt when any source under
csrc/ or include/hclooc.h is newer than the .so.  cudart is linked statically and the driver API is
resolved at run time, so the .so also loads (for hclooc_plan / hclooc_schedule) on a box with no GPU.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhclooc_b200.so")
SOURCES = ["dgemm_sm100.cu", "dgemm_streamk_sm100.cu", "dgemm_direct_sm100.cu", "trsm_sm100.cu", "executor.cu", "fig2_pipeline.cu", "runtime.cu", "planner.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static", "-diag-suppress", "177"]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libhclooc_b200.so cannot be built (there is no CPU fallback)")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = glob.glob(os.path.join(CSRC, "*")) + [os.path.join(ROOT, "include", "hclooc.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
