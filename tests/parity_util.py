"""Shared helpers of the GPU parity tests: drive the oracle and the CUDA library on the same arrays."""
import numpy as np

from oracle import oracle as orc

LAT_ORC = orc.LATTICES
ORC_SCHEME = orc.SCHEMES
TOL64 = 1e-11      # BASELINE.json north_star: max relative error on all macroscopic fields, fp64
TOL32 = 1e-5       # fp32


def oracle_from_workload(w, mask=None):
    return orc.from_workload(w, mask=mask)


def field_errors(Q, Qref):
    """reading A15: per field max|dQ| / max|Qref|; fields identically 0 in the oracle must be exactly 0"""
    errs = []
    for k in range(Qref.shape[0]):
        ref = np.abs(Qref[k]).max()
        d = np.abs(Q[k] - Qref[k]).max()
        errs.append(d if ref == 0.0 else d / ref)
    return np.array(errs)


def diag_errors(dg, dgref, K):
    """global sums against sum|Q_k|; maxima and minima relative"""
    e_sum = np.abs(dg[:K] - dgref[:K]) / np.maximum(dgref[K:2 * K], 1e-300)
    e_abs = np.abs(dg[K:2 * K] - dgref[K:2 * K]) / np.maximum(dgref[K:2 * K], 1e-300)
    e_max = np.abs(dg[2 * K:3 * K] - dgref[2 * K:3 * K]) / np.maximum(dgref[2 * K:3 * K], 1e-300)
    return e_sum, e_abs, e_max
