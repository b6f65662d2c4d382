"""Builds liblise.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "liblise.so")
SOURCES = ["lise.cu"]
HEADERS = ["common.cuh", "state_kernels.cuh", "grid_kernels.cuh", "plane_common.cuh", "split_lineop.cuh", "plane5_kernels.cuh", "peak_kernels.cuh", os.path.join("..", "..", "include", "lise.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def needs_build():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + SOURCES
    subprocess.run(cmd, check=True, cwd=CSRC)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
