"""Build libfe_b200.so in-tree with nvcc for sm_100a (one object per .cu, compiled in parallel).

    python -m paper_2605_28800_b200.build [--force]

The shared library sits next to this file so that it travels with the repository snapshot to the
GPU box; it is git-ignored.  No CPU fallback exists: importing the binding without the library fails.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libfe_b200.so")
PEAKS_LIB = os.path.join(HERE, "libfe_peaks.so")      # bench.py's harness kernels (csrc/bench_peaks.cu), not the product
SOURCES = ["fe_api.cu", "fe_fft.cu", "fe_fft2_x.cu", "fe_fft2_axis.cu", "fe_fft2_z.cu", "fe_fft2_xy.cu", "fe_tensor.cu", "fe_local.cu", "fe_integ.cu"]
HEADERS = [os.path.join(CSRC, "fe_internal.h"), os.path.join(CSRC, "fe_fft2.cuh"), os.path.join(ROOT, "include", "fe.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC"]


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    objs, jobs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(HERE, "build", src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + HEADERS):
            cmd = [NVCC, *FLAGS, "-c", s, "-o", o] + (["-Xptxas", "-v"] if verbose else [])
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
        return r.stderr

    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            for out in ex.map(run, jobs):
                if verbose and out:
                    print(out)
    if jobs or not os.path.exists(LIB):
        run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs])
    peaks_src = os.path.join(CSRC, "bench_peaks.cu")
    if force or _stale(PEAKS_LIB, [peaks_src]):
        run([NVCC, *FLAGS, "-shared", peaks_src, "-o", PEAKS_LIB])
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv))
