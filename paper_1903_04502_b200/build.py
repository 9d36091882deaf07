"""Build the CUDA C-ABI library in-tree:  python -m paper_1903_04502_b200.build [--force]

nvcc cross-compiles sm_100a without a GPU; the resulting libpurify_op.so sits next to this file
(git-ignored, but shipped to the GPU box by gpurun)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpurify_op.so")
SOURCES = ["purify_op.cu", "wavelet.cu"]
DEPS = ["purify_op.cu", "kernels.cuh", "degrid.cuh", "grid.cuh", "batched.cuh", "kb_host.hpp", "ubench.cuh", "wavelet.cu", os.path.join("..", "..", "include", "purify_wavelet.h"),
        os.path.join("..", "..", "include", "purify_op.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(os.path.join(CSRC, d)) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB, "-lcufft"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
