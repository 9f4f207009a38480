"""Build libgabsplat.so (the CUDA path) in-tree with nvcc for sm_100a.

    python -m paper_2508_05343_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library lands next to this file so that it travels with the
repository snapshot to the GPU box (it is git-ignored, not gpurun-ignored).

GABSPLAT_NVCC_FLAGS (environment, optional): extra nvcc flags, e.g. the -D switches of the measured design alternatives
kept in the sources (GS_FWD_STAGING_CPASYNC, GS_BWD_BRANCHFREE, GS_BWD_MINB, GS_BWD_REPLAY, GS_BWD_MAXROWS, GS_BWD_LOWPHASE: DESIGN.md 7.2, 7.4).
Use --force with it; the default build is what the tests and bench.py measure.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_obj")
LIB = os.path.join(HERE, "libgabsplat.so")
SOURCES = ["api.cu", "host_api.cu", "preprocess.cu", "binning.cu", "blend_forward.cu", "blend_backward.cu",
           "preprocess_backward.cu", "loss.cu", "peaks.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def _deps() -> float:
    inc = os.path.join(os.path.dirname(HERE), "include", "gabsplat.h")
    files = [inc] + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    return max(os.path.getmtime(f) for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    hdr_time = _deps()
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_time):
            cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("GABSPLAT_NVCC_FLAGS", "").split() + \
                  (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            jobs.append(cmd)

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
        return r.stderr

    with ThreadPoolExecutor(max_workers=min(8, max(1, len(jobs)))) as ex:
        for log in ex.map(run, jobs):
            if verbose and log:
                print(log, file=sys.stderr)
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    if jobs or not os.path.exists(LIB):
        run([_nvcc(), "-shared", "-o", LIB] + objs + ["-lcudart"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
