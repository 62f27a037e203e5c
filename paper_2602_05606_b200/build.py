"""Build libkappagen.so in-tree with nvcc for sm_100a (no torch headers: a plain C-ABI shared library).

    python -m paper_2602_05606_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libkappagen.so")
CU_SOURCES = ["kappagen_api.cu"]
CPP_SOURCES = ["host_params.cpp", "host_entropy.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC"]


def _newest_source_mtime() -> float:
    # compiled sources and their headers only (fit_polynomials.py prints constants, it is not compiled)
    paths = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh", ".cpp", ".hpp"))]
    paths += [os.path.join(HERE, "..", "include", "kappagen.h"), os.path.abspath(__file__)]
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(SO) and os.path.getmtime(SO) >= _newest_source_mtime():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    for src in CPP_SOURCES:
        obj = os.path.join(CSRC, src + ".o")
        subprocess.run(["g++", "-std=c++17", "-O2", "-fPIC", "-c", os.path.join(CSRC, src), "-o", obj], check=True)
        objs.append(obj)
    for src in CU_SOURCES:
        obj = os.path.join(CSRC, src + ".o")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
        subprocess.run(cmd, check=True)
        objs.append(obj)
    tmp = SO + ".tmp.%d" % os.getpid()
    subprocess.run([nvcc, "-shared", "-o", tmp] + objs + ["-lcudart_static", "-lpthread", "-ldl", "-lrt"], check=True)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
