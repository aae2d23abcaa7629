"""Builds paper_1506_04553_b200/libp3t.so (the C-ABI library of include/p3t.h) for sm_100a.

    python -m paper_1506_04553_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is built in-tree (git-ignored) so that
it travels to the GPU box with the repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libp3t.so")
SOURCES = ["api.cu", "sort.cu", "build.cu", "moments.cu", "walk.cu", "direct.cu", "neighbours.cu", "calib.cu", "hard.cu", "hermite.cu", "static_direct.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC,-O3,-pthread", "-I", os.path.join(ROOT, "include"), "-I", CSRC]
# P3T_CHECKED=1: the kernels' own bounds checks (P3T_DEV_ASSERT of csrc/p3t_internal.cuh) are compiled in; use with --force
if os.environ.get("P3T_CHECKED") == "1":
    NVCC_FLAGS = NVCC_FLAGS + ["-DP3T_CHECKED"]
# tuning experiments: extra nvcc flags (e.g. P3T_NVCC_EXTRA="-DWALK_STACK_SMEM=1024"); use with --force
NVCC_FLAGS = NVCC_FLAGS + os.environ.get("P3T_NVCC_EXTRA", "").split()


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    headers = [os.path.join(CSRC, "p3t_internal.cuh"), os.path.join(ROOT, "include", "p3t.h"), os.path.abspath(__file__)]
    nvcc = _nvcc()
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        if force or _stale(o, [s] + headers):
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        return cmd, r

    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for cmd, r in ex.map(run, jobs):
            if verbose or r.returncode:
                sys.stderr.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
            if r.returncode:
                raise RuntimeError("nvcc failed for " + cmd[-3])
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    if force or jobs or _stale(LIB, objs):
        cmd = [nvcc, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a", "-lcudart", "-lpthread"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
