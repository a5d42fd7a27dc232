"""CPU oracle for the vectorial LBM MHD step — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2606_00641_b200 (the CUDA path) and never imports it.
"""
from .oracle import Oracle, OracleParams, build, lattice, flux, equilibrium  # noqa: F401
