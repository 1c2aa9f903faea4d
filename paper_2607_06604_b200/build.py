"""Build libgramsci.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Usage: python -m paper_2607_06604_b200.build [--force]
The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
GRAMSCI_NVCC_DEFS adds compiler flags, e.g. the bounds-checked debug build (every dense-row gather and shared-memory
histogram address of the gather kernels checked, a violation traps):
    GRAMSCI_NVCC_DEFS=-DG3_BOUNDS=1 python -m paper_2607_06604_b200.build --force && python -m pytest tests -m gpu
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgramsci.so")
SOURCES = ["api.cu", "build_graph.cu", "dense.cu", "noalloc.cu", "query3.cu", "query3g.cu", "query4.cu", "tiler.cu"]
HEADERS = [os.path.join(CSRC, "internal.cuh"), os.path.join(HERE, "..", "include", "gramsci.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--fmad=false",                      # A-3/A-9: no FMA contraction anywhere in the device code
    "-Xcompiler", "-fPIC,-O2,-ffp-contract=off,-pthread",
    "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("GRAMSCI_NVCC_DEFS", "").split(), "-c", os.path.join(CSRC, s), "-o", o]
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(o)
    log = []
    for s, p in procs:
        out, _ = p.communicate()
        log.append(out)
        if p.returncode != 0:
            sys.stderr.write(out)
            raise RuntimeError(f"nvcc failed on {s}")
    cmd = [_nvcc(), "-shared", "-Wno-deprecated-gpu-targets", "-o", LIB, *objs, "-lcudart", "-lpthread"]
    subprocess.run(cmd, check=True)
    with open(os.path.join(CSRC, "ptxas_info.log"), "w") as f:
        f.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
