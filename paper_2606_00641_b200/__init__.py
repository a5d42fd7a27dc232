"""B200-native vectorial lattice Boltzmann step for MHD (arxiv/paper_2606_00641).

`lbmhd` is the ctypes binding of the C-ABI CUDA library (include/lbmhd.h); importing this package does
not load it, so the input generators in `workloads` stay usable on a CPU-only box.
"""
__all__ = ["lbmhd", "workloads", "build"]
