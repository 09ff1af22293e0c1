"""Build libak.so (the C-ABI CUDA library of include/ak.h) in-tree with nvcc for sm_100a.

    python -m paper_2409_10384_b200.build [--force]

--fmad=false: every fp64 operation is a separate IEEE operation in the written order, which
makes the con2prim status and FOFC flag masks bit-reproducible.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libak.so")
SOURCES = ["ak_api.cu"]
HEADERS = ["ak_dev.cuh", "ak_flux.cuh", "ak_kernels.cuh", "ak_source.cuh", "ak_flux_tma.cuh", "ak_driver.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "--fmad=false", "-O3", "-lineinfo",
              "-std=c++17", "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _deps():
    d = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    d.append(os.path.join(os.path.dirname(HERE), "include", "ak.h"))
    d.append(os.path.abspath(__file__))
    return d


def build(force=False, verbose=False):
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(s) for s in _deps()):
        return SO
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
