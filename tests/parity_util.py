"""Shared helpers of the GPU parity tests: drive the oracle and the CUDA library on the same arrays."""
import numpy as np

from oracle import oracle as orc

LAT_ORC = {"D1Q3": orc.D1Q3, "D2Q9": orc.D2Q9, "D3Q19": orc.D3Q19, "D2Q5": orc.D2Q5, "D3Q7": orc.D3Q7}
ORC_SCHEME = {"IDEAL": orc.IDEAL, "INCRES": orc.INCRES, "IDEAL_DIVB": orc.IDEAL_DIVB, "RESIST": orc.RESIST, "FULL": orc.FULL}
TOL64 = 1e-11      # BASELINE.json north_star: max relative error on all macroscopic fields, fp64
TOL32 = 1e-5       # fp32


def oracle_from_workload(w, mask=None):
    p = orc.make_params(ORC_SCHEME[w["scheme"]], LAT_ORC[w["lattice"]], w["shape"],
                        gamma=w["gamma"] or 1.4, c0sq=w["c0sq"], nu=w["nu"], eta=w["eta"], tau=w["tau"],
                        powell=w["powell"], bc=w["bc"], tau_relax=w.get("tau_relax", 0.0), eta_jc=w.get("eta_jc", 0.0))
    o = orc.Oracle(p, mask=mask)
    if w.get("sphere"):
        s = w["sphere"]
        o.set_sphere(s["centre"], s["radius"], s["u_solid"], s["dipole_dir"], s["B_surface"])
        if s.get("width"):
            o.set_sphere_width(s["width"])
        if s.get("omega") is not None:
            o.set_sphere_rotation(s["omega"])
        if s.get("dipoles"):
            dp = s["dipoles"]
            o.set_sphere_dipoles(dp["offsets"], dp["dirs"], dp["B_surface"], dp["cores"])
    return o


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
