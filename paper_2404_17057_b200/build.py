"""Build libmpm_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2404_17057_b200.build [--force]

nvcc cross-compiles without a GPU.  The static CUDA runtime is linked so that the library is self-contained;
the built .so travels to the GPU box with the repository snapshot (it is git-ignored, not gpurun-ignored).
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmpm_b200.so")
LIB_CHECKED = os.path.join(HERE, "libmpm_b200_checked.so")      # -DMPM_CHECKED=1: own bounds checks, traps on a violation
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "--shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "mpm.h")]


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    lib = LIB_CHECKED if checked else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= max(os.path.getmtime(p) for p in _deps()):
        return lib
    cmd = [NVCC] + FLAGS + (["-DMPM_CHECKED=1"] if checked else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + sources()
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
