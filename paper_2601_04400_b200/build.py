"""Build the CUDA library (paper_2601_04400_b200/libjxs.so) for sm_100a, in-tree.

    python -m paper_2601_04400_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libjxs.so")
SOURCES = [os.path.join(CSRC, "jxs_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("stage_kernel.cuh", "stage1d_kernel.cuh", "tangent1d_kernel.cuh", "adjoint1d_kernel.cuh", "mlp1d_kernel.cuh", "deriv2d_kernels.cuh", "aux_kernels.cuh", "flux_mlp_kernel.cuh", "flux_cnn_kernel.cuh")] + [
    os.path.join(ROOT, "include", "jxs.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)):
        return LIB
    cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB, *SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
