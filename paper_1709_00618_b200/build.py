"""Builds paper_1709_00618_b200/libtpctrk.so (the C-ABI library of include/tpc_tracker.h) in-tree with nvcc for sm_100a.

    python -m paper_1709_00618_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The neighbour-finder translation unit is compiled with -fmad=false on top of
its explicitly rounded intrinsics (bit-exact contract of S2).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libtpctrk.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
# extra nvcc flags for every translation unit, e.g. TPC_NVCC_FLAGS="-DTPC_FOLLOW_CTAS=8" (kernel tuning switches)
EXTRA = os.environ.get("TPC_NVCC_FLAGS", "").split()

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC,-Wall", "-Xptxas", "-v"]
SOURCES = {
    "tpc_tracker.cu": [],
    "k1_bin_rows.cu": [],
    "k2_neighbours.cu": ["-fmad=false"],
    "k34_links_chains.cu": [],
    "k5_follow.cu": [],
    "k6_select.cu": [],
    "k7_phase2.cu": [],
    "k8_vertex.cu": [],
    "k9_start_hits_static.cu": [],
    "host_pipeline.cu": [],
}


# bench-only helpers (not part of the C ABI of include/tpc_tracker.h): libtpcbench.so, loaded by bench.py
BENCH_SRC = os.path.join(HERE, "csrc_bench")
BENCH_LIB = os.path.join(HERE, "libtpcbench.so")


def _deps_mtime() -> float:
    paths = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    paths += [os.path.join(BENCH_SRC, f) for f in os.listdir(BENCH_SRC)]
    paths.append(os.path.join(os.path.dirname(HERE), "include", "tpc_tracker.h"))
    paths.append(os.path.abspath(__file__))
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.exists(BENCH_LIB)
            and min(os.path.getmtime(LIB), os.path.getmtime(BENCH_LIB)) >= _deps_mtime()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    objs = []
    log = []
    for src, extra in SOURCES.items():
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [NVCC, *ARCH, *COMMON, *extra, *EXTRA, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            sys.stderr.write(log[-1])
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    cmd = [NVCC, *ARCH, "-shared", "-o", LIB, *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        sys.stderr.write(log[-1])
        raise RuntimeError("link failed")
    cmd = [NVCC, *ARCH, "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC,-Wall", "-shared", "-o", BENCH_LIB,
           *[os.path.join(BENCH_SRC, f) for f in sorted(os.listdir(BENCH_SRC)) if f.endswith(".cu")]]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        sys.stderr.write(log[-1])
        raise RuntimeError("nvcc failed on the bench-only library")
    with open(os.path.join(OBJ, "build.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
