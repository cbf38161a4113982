"""Build libr360.so in-tree with nvcc for sm_100a (no torch extension machinery needed:
the boundary is a plain C ABI loaded with ctypes)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(CSRC, "libr360.so")
BENCH_SO = os.path.join(CSRC, "libr360_bench.so")      # bench.py's measurement helper: not part of the product ABI
SOURCES = ["capi.cu", "render.cu", "sampler.cu", "mlp_fp32.cu", "mlp_tc.cu", "composite.cu", "assign.cu", "floorplan.cu", "fuse.cu"]
BENCH_SOURCES = ["microbench.cu"]
HEADERS = sorted(f for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))) + [os.path.join("..", "..", "include", "r360.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math,-Wall", "--shared", "-cudart", "static"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def build_bench(force: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in BENCH_SOURCES]
    if not force and os.path.exists(BENCH_SO) and os.path.getmtime(BENCH_SO) >= max(os.path.getmtime(d) for d in srcs):
        return BENCH_SO
    subprocess.check_call([_nvcc(), *NVCC_FLAGS, "-o", BENCH_SO, *srcs])
    return BENCH_SO


def build(force: bool = False, verbose: bool = False) -> str:
    build_bench(force)
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    if not force and os.path.exists(SO) and os.path.getmtime(SO) >= max(os.path.getmtime(d) for d in deps):
        return SO
    cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("R360_NVCC_FLAGS", "").split(), "-o", SO, *srcs]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
