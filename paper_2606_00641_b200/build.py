"""Builds the C-ABI CUDA library in-tree for sm_100a with nvcc (no torch in the build).

The kernel templates are instantiated once per (lattice, precision, scheme group) in csrc/lbmhd_inst.cu; those twenty translation units and
csrc/lbmhd_api.cu and csrc/lbmhd_noalloc.cu compile in parallel into build/*.o and link into liblbmhd.so."""
import os
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(_HERE, "liblbmhd.so")
OBJ_DIR = os.path.join(_HERE, "build")
DEPS = [os.path.join(_CSRC, f) for f in ("lbmhd_api.cu", "lbmhd_inst.cu", "lbmhd_noalloc.cu", "lbmhd_host.h", "lbmhd_ops.cuh", "lbmhd_kernels.cuh",
                                         "lbmhd_lattice.cuh", "lbmhd_tma.cuh", "lbmhd_resident.cuh")] + \
       [os.path.join(os.path.dirname(_HERE), "include", "lbmhd.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]
LATTICES = (3, 2, 5, 4, 1)          # heaviest first: D3Q19, D2Q9, D3Q7, D2Q5, D1Q3
PRECISIONS = (64, 32)


def needs_build():
    return (not os.path.exists(SO)) or os.path.getmtime(SO) < max(os.path.getmtime(d) for d in DEPS)


def _units():
    units = [("api", os.path.join(_CSRC, "lbmhd_api.cu"), []), ("noalloc", os.path.join(_CSRC, "lbmhd_noalloc.cu"), [])]
    for lat in LATTICES:
        for bits in PRECISIONS:
            for grp in (1, 0):      # RESIST / FULL first: the heavier half
                units.append(("inst_%d_%d_g%d" % (lat, bits, grp), os.path.join(_CSRC, "lbmhd_inst.cu"),
                              ["-DLBMHD_INST_LAT=%d" % lat, "-DLBMHD_INST_BITS=%d" % bits, "-DLBMHD_INST_GROUP=%d" % grp]))
    return units


def build(force=False, verbose=False, jobs=None, extra_flags=(), out=None):
    """extra_flags: more nvcc flags for every unit; out: path of the library to write (default: the in-tree liblbmhd.so)"""
    out = out or SO
    if out == SO and not force and not needs_build():
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    obj_dir = OBJ_DIR if out == SO else out + ".build"
    os.makedirs(obj_dir, exist_ok=True)
    jobs = jobs or int(os.environ.get("LBMHD_BUILD_JOBS", "0")) or min(os.cpu_count() or 1, 22)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(unit):
        name, src, defs = unit
        obj = os.path.join(obj_dir, name + ".o")
        subprocess.run([nvcc] + NVCC_FLAGS + extra + list(extra_flags) + defs + ["-c", src, "-o", obj], check=True, cwd=_CSRC)
        return obj

    with ThreadPoolExecutor(max_workers=jobs) as pool:
        objs = list(pool.map(compile_one, _units()))
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-o", out], check=True, cwd=_CSRC)
    shutil.rmtree(obj_dir, ignore_errors=True)      # intermediates only: every unit depends on the same headers
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
