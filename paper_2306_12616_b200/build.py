"""Build the CUDA library (csrc/cheb_dm.cu -> libcheb_dm.so) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The resulting .so is git-ignored but travels to the GPU box.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "cheb_dm.cu")
LIB_PATH = os.path.join(_HERE, "libcheb_dm.so")
_DEPS = [os.path.join(_HERE, "csrc", f) for f in ("cheb_dm.cu", "common.cuh", "gemm_dmma.cuh", "gemm_epi.cuh", "giant_resident.cuh", "aux_kernels.cuh", "ozaki.cuh")]
_DEPS.append(os.path.join(os.path.dirname(_HERE), "include", "cheb_dm.h"))

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(d) > t for d in _DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB_PATH, SRC]
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB_PATH


if __name__ == "__main__":
    build(force=True, verbose=True)
