"""Small runs of every step-kernel family for compute-sanitizer (SURVEY.md §5 aux row "race / memory checking"):

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py

The places where a mis-indexed slot would be a silent race or an out-of-bounds access: the in-place (AA) kernels in both
step types with x-edge, general and sphere tiles; the 2-CTA cluster exchange through distributed shared memory
(step_kernel_cl); the multi-cell and cell-per-thread kernels with their vector accesses and shuffled stores; the cooperative
many-step launch; the register-resident cluster kernel of the 1D lattices; the slab halo pack / unpack with the in-place return exchange.  Each case is also compared with the
oracle, so a run that passes the tool but computes garbage still fails.  On this project's GPU pool compute-sanitizer is
closed (profiles/r2_sanitizer.md records the refusal); there tests/test_guard_gpu.py runs these same cases with guard bands
around every workspace instead.  Not collected by pytest (no test_ prefix)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def main():
    from paper_2606_00641_b200 import slab
    from parity_util import TOL64, TOL32, field_errors
    from test_parity_gpu import compare, random_workload, resist_workload, full_workload, gpu_from_workload
    mh = np.array([0.3, -0.5, 0.8]) / np.linalg.norm([0.3, -0.5, 0.8])
    sph = dict(centre=np.array([40.3, 9.1, 6.2]), radius=4.0, u_solid=np.array([-0.25, 0.0, 0.0]), dipole_dir=mh, B_surface=0.03)

    def case(name, env, fn):
        saved = dict(os.environ)
        os.environ.update(env)
        try:
            fn()
        finally:
            os.environ.clear()
            os.environ.update(saved)
        print("ok", name, flush=True)

    base = {"LBMHD_PERSIST": "0"}
    # one thread per (cell, variable): A/B and both in-place step types, all tile classes, the moving sphere
    w3 = random_workload("IDEAL", "D3Q19", (100, 18, 12), (2, 1, 0, 0, 0, 0), seed=301, sphere=sph)
    for streaming in (0, 1):
        case("step_kernel D3Q19 streaming %d" % streaming, base, lambda: (compare(w3, 5, streaming=streaming), compare(w3, 4, streaming=streaming)))
    w2 = random_workload("IDEAL", "D2Q9", (150, 37), (1, 1, 1, 1, 0, 0), seed=302)
    case("step_kernel D2Q9 in place, zero-gradient box", base, lambda: compare(w2, 5, streaming=1))
    # several cells per thread (vector loads, shuffled fp32 pull-push stores)
    wm = random_workload("IDEAL", "D3Q19", (292, 6, 5), (2, 1, 0, 0, 0, 0), seed=303)
    for prec, tol in ((64, TOL64), (32, TOL32)):
        case("step_kernel_multi fp%d in place and A/B" % prec, dict(base, LBMHD_MULTI="1"),
             lambda: (compare(wm, 5, tol=tol, precision=prec, streaming=1), compare(wm, 4, tol=tol, precision=prec, streaming=0)))
    wq = random_workload("IDEAL", "D3Q7", (292, 6, 5), (0, 0, 1, 1, 0, 0), seed=304)
    case("step_kernel_multi D3Q7 fp32 (four cells per thread) in place", dict(base, LBMHD_MULTI="1", LBMHD_CELL="0"),
         lambda: compare(wq, 5, tol=TOL32, precision=32, streaming=1))
    case("step_kernel_cell D3Q7 in place and A/B", dict(base, LBMHD_CELL="2"), lambda: (compare(wq, 5, streaming=1), compare(wq, 4, streaming=0)))
    # variable rows split over a 2-CTA cluster (distributed shared memory)
    wr = resist_workload("D3Q19", (100, 12, 9), (2, 1, 0, 0, 0, 0), seed=305)
    for streaming in (0, 1):
        case("step_kernel_cl RESIST streaming %d" % streaming, base, lambda: compare(wr, 5, streaming=streaming))
    wf = full_workload("D3Q19", (64, 8, 6), (1, 1, 1, 1, 1, 1), seed=306)
    case("step_kernel FULL (26 rows) in place", base, lambda: compare(wf, 4, streaming=1))
    # many steps in one cooperative launch
    wp = random_workload("IDEAL", "D2Q9", (90, 21), (1, 1, 2, 1, 0, 0), seed=307)
    for streaming in (0, 1):
        case("step_kernel_persist streaming %d" % streaming, {"LBMHD_PERSIST": "2"}, lambda: compare(wp, 7, streaming=streaming))

    # 1D lattices, populations resident in registers: one cluster, halo cells through distributed shared memory; both in-place
    # layouts read and written (7 steps from P0 end in P1, 6 more from P1 end in P1 ... ), ragged last CTA, every face kind
    def resident(w, streaming):
        from paper_2606_00641_b200 import lbmhd
        from parity_util import oracle_from_workload
        o = oracle_from_workload(w)
        o.init(w["fields"])
        o.step(18)
        g = gpu_from_workload(w, streaming=streaming)
        g.init(w["fields"])
        for n in (7, 6, 5):
            g.step(n)
            assert g.step_path == lbmhd.PATH_RESIDENT
        Q = g.moments()[0]
        g.close()
        assert (field_errors(Q, o.moments(diag=False)) <= TOL64).all()
        o.close()
    for nx, bc in ((800, (1, 1)), (131, (2, 1)), (100, (0, 0)), (20, (1, 2))):
        w1 = random_workload("IDEAL", "D1Q3", (nx,), bc + (0, 0, 0, 0), seed=308)
        for streaming in (0, 1):
            case("step_kernel_resident nx %d bc %s streaming %d" % (nx, bc, streaming), {"LBMHD_RESIDENT": "1", "LBMHD_PERSIST": "0"},
                 lambda: resident(w1, streaming))
    # dependent launches (griddepcontrol) are on in every case above (LBMHD_PDL default)

    # slabs: halo pack / unpack, in-place return exchange, overlapped schedule
    def slabs(streaming):
        w = random_workload("IDEAL", "D3Q19", (70, 9, 12), (2, 1, 1, 1, 0, 0), seed=309)
        ref = gpu_from_workload(w, streaming=streaming)
        ref.init(w["fields"])
        ref.step(5)
        Qr = ref.moments()[0]
        ref.close()
        grp = slab.LocalSlabGroup(w, 3, streaming=streaming, overlap=True)
        grp.init(w["fields"])
        grp.step(5)
        Qs = grp.moments()[0]
        grp.close()
        assert (field_errors(Qs, Qr) <= 1e-13).all()
    for streaming in (0, 1):
        case("slabs overlapped streaming %d" % streaming, base, lambda: slabs(streaming))
    print("all sanitizer cases ran")


if __name__ == "__main__":
    main()
