"""Build libak.so (the C-ABI CUDA library of include/ak.h) in-tree with nvcc for sm_100a.

    python -m paper_2409_10384_b200.build [--force] [--fma]

libak.so, the product, is compiled --fmad=false: every fp64 operation is a separate IEEE operation
in the written order, which makes the con2prim status and FOFC flag masks bit-reproducible
(DESIGN.md §3).  --fma also builds libak_fma.so, the same sources with --fmad=true: the
FMA-contracted "perf build" of SURVEY.md §8(d), which bench.py times beside the product and
compares with it (BASELINE.json: "documented differences only where fp64 FMA contraction is
allowed"); load it with AK_LIBRARY or ak.use_library().
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libak.so")
SO_FMA = os.path.join(HERE, "libak_fma.so")
SOURCES = ["ak_api.cu"]
HEADERS = ["ak_dev.cuh", "ak_flux.cuh", "ak_kernels.cuh", "ak_source.cuh", "ak_flux_tma.cuh", "ak_flux_pencil.cuh",
           "ak_flux_static.cuh", "ak_driver.cuh"]
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


def build(force=False, verbose=False, fma=False):
    so = SO_FMA if fma else SO
    if not force and os.path.exists(so) and all(os.path.getmtime(so) >= os.path.getmtime(s) for s in _deps()):
        return so
    flags = ["--fmad=true" if (fma and f == "--fmad=false") else f for f in NVCC_FLAGS]
    cmd = [_nvcc()] + flags + (["-Xptxas", "-v"] if verbose else []) + ["-o", so] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--fma" in sys.argv:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, fma=True))
