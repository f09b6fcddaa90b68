"""Builds libmhd_b200.so (the C-ABI library of include/mhd.h) in-tree with nvcc for sm_100a.

    python -m paper_2510_13965_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU. Objects and the shared library land next to this file (git-ignored).
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmhd_b200.so")
SOURCES = {"api.cu": [], "elementwise.cu": [], "c2p.cu": [], "ccz4.cu": [], "flux.cu": [], "m1.cu": [], "amr.cu": [], "les.cu": [], "noalloc.cu": []}
COMMON = ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC"]


def _newer(target, deps):
    return os.path.exists(target) and all(os.path.getmtime(target) >= os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    headers = [os.path.join(CSRC, "mhd_internal.cuh"), os.path.join(CSRC, "rootfind.cuh"), os.path.join(CSRC, "tma.cuh"), os.path.join(HERE, "..", "include", "mhd.h"), os.path.abspath(__file__)]
    objs, jobs = [], []
    for src, extra in SOURCES.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(o)
        if force or not _newer(o, [s] + headers):
            cmd = ["nvcc"] + COMMON + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
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
        run(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
