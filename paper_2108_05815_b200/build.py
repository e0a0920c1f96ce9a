"""Builds paper_2108_05815_b200/csrc/libnecsim_b200.so for sm_100a with nvcc (in-tree).

    python -m paper_2108_05815_b200.build [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(CSRC, "libnecsim_b200.so")
SOURCES = ["necsim.cu"]
DEPS = ["necsim.cu", "device_prims.cuh", "sim_types.cuh", "sim_kernel.cuh", "tail_kernel.cuh", "aux_kernels.cuh", "neglog_tables.inc",
        os.path.join("..", "..", "include", "necsim.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=false",
              "-Xcompiler", "-fPIC", "-shared"]


def build(force=False, verbose=False):
    deps = [os.path.join(CSRC, d) for d in DEPS]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", OUT]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
