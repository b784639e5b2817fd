"""Builds libtpctrack.so in-tree with nvcc for sm_100a (no torch involved: the library is a plain C ABI).

    python -m paper_2502_09138_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(_HERE, "libtpctrack.so")
SOURCES = ["api.cu", "a1_grid.cu", "a2_neighbours.cu", "a3_seeds.cu", "a4_follow.cu", "a4_phases.cu", "a5_select.cu", "a6_refit.cu",
           "a7_merge.cu", "a8_compress.cu", "a9_cluster.cu", "a10_rans.cu", "debug.cu"]
HEADERS = [os.path.join(CSRC, "tpc_internal.cuh"), os.path.join(CSRC, "kalman.cuh"), os.path.join(CSRC, "a4_search.cuh"), os.path.join(os.path.dirname(_HERE), "include", "tpc_track.h")]
# a4 only: fp32 division / sqrt / rsqrt as MUFU + one correction (2 ulp), denormals flushed.  Measured against
# the fp64 oracle on configs 0, 1, 2, 4: worst parameter error 9e-6 (bar 1e-4), hit tables unchanged; a4 -5 %.
EXTRA_FLAGS = {"a4_follow.cu": ["--use_fast_math"], "a4_phases.cu": ["--use_fast_math"], "a6_refit.cu": ["--use_fast_math"]}
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + HEADERS + [os.path.abspath(__file__)]
    if not force and os.path.exists(SO) and all(os.path.getmtime(d) <= os.path.getmtime(SO) for d in deps):
        return SO
    objs = []
    procs = []
    for s in srcs:
        o = os.path.join(CSRC, os.path.basename(s)[:-3] + ".o")
        objs.append(o)
        if not force and os.path.exists(o) and all(os.path.getmtime(d) <= os.path.getmtime(o) for d in [s] + HEADERS):
            continue
        cmd = ([_nvcc()] + NVCC_FLAGS + EXTRA_FLAGS.get(os.path.basename(s), [])
               + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o])
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for cmd, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + out)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-o", SO] + objs
    subprocess.check_call(link)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
