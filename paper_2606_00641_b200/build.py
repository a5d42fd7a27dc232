"""Builds the C-ABI CUDA library in-tree for sm_100a with nvcc (no torch in the build)."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(_HERE, "liblbmhd.so")
SRC = os.path.join(_HERE, "csrc", "lbmhd_api.cu")
DEPS = [SRC, os.path.join(_HERE, "csrc", "lbmhd_kernels.cuh"), os.path.join(_HERE, "csrc", "lbmhd_lattice.cuh"),
        os.path.join(_HERE, "csrc", "lbmhd_tma.cuh"),
        os.path.join(os.path.dirname(_HERE), "include", "lbmhd.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--split-compile", "0",
              "-shared", "-Xcompiler", "-fPIC"]


def needs_build():
    return (not os.path.exists(SO)) or os.path.getmtime(SO) < max(os.path.getmtime(d) for d in DEPS)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [SRC, "-o", SO]
    subprocess.run(cmd, check=True, cwd=os.path.join(_HERE, "csrc"))
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
