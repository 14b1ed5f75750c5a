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
SOURCES = ["dgemm_sm100.cu", "dgemm_streamk_sm100.cu", "dgemm_direct_sm100.cu", "trsm_sm100.cu", "potrf_sm100.cu", "getrf_sm100.cu", "factor.cu", "lu.cu", "blas3_ooc.cu", "resident.cu", "executor.cu", "fig2_pipeline.cu", "runtime.cu", "planner.cpp"]
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
    """One object per source under _obj/ (git-ignored), compiled in parallel and only when the source, a header under
    csrc/ or include/hclooc.h is newer than it; then one link."""
    if not (force or stale()):
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    nvcc = _nvcc()
    objdir = os.path.join(HERE, "_obj")
    os.makedirs(objdir, exist_ok=True)
    headers = glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(ROOT, "include", "hclooc.h")]
    t_hdr = max(os.path.getmtime(h) for h in headers)
    cflags = [f for f in NVCC_FLAGS if f != "-shared"]

    def compile_one(src):
        obj = os.path.join(objdir, os.path.splitext(src)[0] + ".o")
        path = os.path.join(CSRC, src)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(t_hdr, os.path.getmtime(path)):
            subprocess.check_call([nvcc] + cflags + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, path])
        return obj

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.check_call([nvcc] + NVCC_FLAGS + ["-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
