"""Compiles libmlens.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libmlens.so")
BENCH_SO = os.path.join(HERE, "libmlens_bench.so")      # roofline micro-benchmarks (include/mlens_bench.h), bench.py only
SOURCES = ["api.cu", "tree.cu", "fmm.cu", "eval.cu", "shoot.cu", "consume.cu"]
HEADERS = ["common.cuh", "device.cuh", "tile.cuh", "deposit.cuh", os.path.join("..", "..", "include", "mlens.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-shared"]


def stale():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    bsrc = os.path.join(CSRC, "bench_kernels.cu")
    bhdr = os.path.join(HERE, "..", "include", "mlens_bench.h")
    if force or not os.path.exists(BENCH_SO) or max(os.path.getmtime(bsrc), os.path.getmtime(bhdr)) > os.path.getmtime(BENCH_SO):
        subprocess.run([NVCC] + FLAGS + ["-o", BENCH_SO, "bench_kernels.cu"], check=True, cwd=CSRC)
    if not force and not stale():
        return SO
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + SOURCES
    subprocess.run(cmd, check=True, cwd=CSRC)
    return SO


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(SO)
