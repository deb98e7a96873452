"""Builds libwd.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2407_00041_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libwd.so")
BENCH_SO = os.path.join(HERE, "libwdbench.so")  # measurement helpers of bench.py (include/wd_bench.h), not the product
SOURCES = ["wd_api.cu", "wd_kernels.cu", "wd_tma.cu", "wd_tmb.cu", "wd_tmw.cu", "wd_tmq.cu", "wd_pack.cu", "wd_clover.cu", "wd_gmres.cu", "wd_dd.cu", "wd_f32.cu"]
BENCH_SOURCES = [os.path.join("bench", "wd_peaks.cu")]
HEADERS = ["wd_internal.h", "wd_handle.h", "wd_math.cuh", "wd_tma.cuh", "wd_tma_common.cuh", "wd_tma_plan.cuh", "wd_smem_ops.cuh", "wd_ldg_kernels.cuh",
           os.path.join("..", "..", "include", "wd.h"), os.path.join("..", "..", "include", "wd_bench.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC,-fopenmp,-O2", "--expt-relaxed-constexpr"]


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    bsrcs = [os.path.join(CSRC, s) for s in BENCH_SOURCES]
    deps = srcs + bsrcs + [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    if (not force and os.path.exists(SO) and os.path.exists(BENCH_SO)
            and min(os.path.getmtime(SO), os.path.getmtime(BENCH_SO)) >= _newest(deps)):
        return SO
    os.makedirs(OBJDIR, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    if os.environ.get("WD_EXPERIMENTS"):  # tracing / policy knobs of the TMA kernels (never in the default build)
        extra += ["-DWD_EXPERIMENTS"]

    def compile_one(src):
        obj = os.path.join(OBJDIR, os.path.basename(src) + ".o")
        cmd = [NVCC, *FLAGS, *extra, "-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with concurrent.futures.ThreadPoolExecutor(max_workers=len(srcs) + len(bsrcs)) as ex:
        allobjs = list(ex.map(compile_one, srcs + bsrcs))
    objs, bobjs = allobjs[:len(srcs)], allobjs[len(srcs):]
    for so, oo in ((SO, objs), (BENCH_SO, bobjs)):
        cmd = [NVCC, "-shared", "-o", so, *oo, "-Xcompiler", "-fopenmp", "-lgomp", "-cudart", "static"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
