#!/usr/bin/env python
"""bench.py — MLUPS and achieved HBM GB/s of the fused VLBM MHD step (BASELINE.json metric).

  python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload C5]

One "step" = one pass of the whole hot path (one lbmhd_step launch) over the resident workload.
N = 1 runs BASELINE config 5 (3D ideal MHD, D3Q19 x 8 sets, fp64, 384x256x256, moving magnetised sphere):
the configuration the north_star target is quoted on.  N > 1 (torchrun): every rank runs the same
workload on its own GPU with no data-path collective ("scaling": "weak").
Prints ONE JSON line on rank 0.  --impl reference times the CPU oracle (oracle/) on the host cores.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "MLUPS (fused VLBM MHD stream-collide step)"
SAMPLE_SHAPE = (96, 64, 64)      # bounded sample of the same workload for the CPU oracle legs


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons of one GPU during the timed region (NVML)"""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.sm_max = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap", nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.05)

    def result(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons)}


def max_over_ranks(values, world, device=None):
    """element-wise MAX of a list of floats over all ranks (the contract's max-over-ranks timing); identity at world 1"""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_mlups(cells_per_rank, steps, ms, world):
    """whole-job throughput: every rank advanced its own replica `steps` times in `ms` (max over ranks)"""
    return world * cells_per_rank * steps / (ms * 1e-3) / 1e6


def oracle_leg(workload_name, steps, warmup, budget_s=None, scheme=None, lattice=None):
    """the CPU oracle, as it stands, on a bounded sample of the workload; -> (MLUPS, cores, sample text, ms/step)"""
    from oracle import oracle as orc
    from paper_2606_00641_b200 import workloads as W
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity_util import oracle_from_workload
    w = W.config5(shape=SAMPLE_SHAPE) if workload_name == "C5" else W.get(workload_name, small=True)
    w = W.variant(w, scheme=scheme, lattice=lattice)
    o = oracle_from_workload(w)
    o.init(w["fields"])
    o.step(max(warmup, 1))
    N = int(np.prod(w["shape"]))
    t0 = time.perf_counter()
    done = 0
    while done < steps:
        o.step(1)
        done += 1
        if budget_s is not None and done >= 3 and time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    sample = "%s at %s (same recipe, reduced size), %d steps after %d warm-up" % (
        workload_name, "x".join(str(s) for s in w["shape"]), done, max(warmup, 1))
    return N * done / dt / 1e6, orc.get_threads(), sample, dt / done * 1e3, w


def run_reference(args, rank):
    if rank != 0:
        return
    mlups, cores, sample, ms, w = oracle_leg(args.workload, args.steps, args.warmup, scheme=args.scheme, lattice=args.lattice)
    line = {"impl": "reference", "metric": METRIC, "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s (CPU oracle on a bounded sample)" % args.workload, "sample": sample},
            "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_native(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2606_00641_b200 import lbmhd, workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    local_rank = local_rank % torch.cuda.device_count()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(args.backend)
    if args.decomp == "slab" and world > 1:
        return run_slab(args, rank, world, local_rank, dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    w = W.variant(W.get(args.workload), scheme=args.scheme, lattice=args.lattice)
    N = int(np.prod(w["shape"]))
    prec = args.precision
    sim = lbmhd.from_workload(w, precision=prec, device=local_rank, streaming=1 if args.streaming == "inplace" else 0)
    K, Q = sim.K, sim.Q
    bytes_per_cell = 2 * K * Q * (8 if prec == 64 else 4) + (0 if w.get("sphere") else 0)
    st = sim.stream

    # ---- device-resident timing: inputs already in HBM -------------------------------------------------
    F_dev = torch.as_tensor(w["fields"]).to(dev)
    sim.init(F_dev)
    sim.step(args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    sim.step(args.steps)
    e1.record(st)
    barrier()
    launches = sim.launch_count - l0
    sampler.stop_flag = True
    sampler.join()
    ms_total = e0.elapsed_time(e1)
    _, dg = sim.moments(want_fields=False)
    if dg[-1] != 0:
        raise SystemExit("bench.py: numerical failure flag %g after the timed run" % dg[-1])

    # ---- end to end through the C ABI with HOST buffers: init (H2D) + K steps + moments (D2H) ----------
    F_host = torch.as_tensor(w["fields"]).pin_memory()
    out_host = torch.empty_like(F_host).pin_memory()
    diag_host = torch.empty(3 * K + 4, dtype=torch.float64).pin_memory()
    del F_dev
    sim.init(F_host)               # warm the path once
    sim.moments(out_host, diag_host)
    barrier()
    t0 = torch.cuda.Event(enable_timing=True)
    t1 = torch.cuda.Event(enable_timing=True)
    t0.record(st)
    sim.init(F_host)
    sim.step(args.steps)
    sim.moments(out_host, diag_host)
    t1.record(st)
    barrier()
    ms_e2e = t0.elapsed_time(t1)
    h2d = F_host.numel() * 8
    d2h = out_host.numel() * 8 + diag_host.numel() * 8

    ms_total, ms_e2e = max_over_ranks([ms_total, ms_e2e], world, dev)
    own_copy = lbmhd.copy_probe(1 << 27, reps=5, device=local_rank) if rank == 0 else None   # fp64 copy, this library's grid style
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = load_peaks()
    ms_step = ms_total / args.steps
    value = aggregate_mlups(N, args.steps, ms_total, world)
    achieved = N * bytes_per_cell / (ms_step * 1e-3) / 1e9
    e2e_val = aggregate_mlups(N, args.steps, ms_e2e, world)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")      # dram__bytes_read/write.sum of one ncu --set full capture
    if os.path.exists(tpath) and prec == 64 and args.streaming == "ab" and args.scheme is None and args.lattice is None:
        with open(tpath) as f:
            for row in f.read().splitlines()[1:]:
                cols = row.split(",")
                if cols[0] == args.workload:
                    traffic = float(cols[1]) + float(cols[2])
    line = {
        "metric": METRIC, "value": value, "unit": "MLUPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if prec == 64 else "f32", "data": "synthetic",
        "config": {"workload": "%s: %s %s x %d sets, %s, %s, %d B/cell/step; replicas per GPU, no collective" % (
                       w["name"], w["scheme"], w["lattice"], K, "x".join(str(s) for s in w["shape"]),
                       "fp64" if prec == 64 else "fp32", bytes_per_cell),
                   "cells": N, "streaming": "in-place AA pattern, one copy" if args.streaming == "inplace" else "A/B double buffer",
                   "workspace_GB": round(sim.workspace.numel() / 1e9, 2),
                   "l2": "populations %.1f GB >> 126 MB L2, no flush needed" % (
                       (1 if args.streaming == "inplace" else 2) * N * bytes_per_cell / 2 / 1e9)},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "peak_source": peak_src,
                     "kernel": {0: "step_kernel", 1: "step_kernel_multi", 2: "step_kernel_cl", 3: "step_kernel_tma"}.get(sim.step_path, "?"),
                     "frac_of_nominal_8TBs": achieved / 8000.0,
                     "own_fp64_copy_GBs": own_copy, "frac_of_own_copy": achieved / own_copy,
                     "paper_context": "98.9% (2D) / 75.8% (3D) of 680 GB/s BabelStream, RTX A5000 fp32 (PAPER.md:269)"},
        "e2e": {"value": e2e_val, "unit": "MLUPS", "h2d_bytes_per_step": h2d / args.steps,
                "d2h_bytes_per_step": d2h / args.steps,
                "what": "lbmhd_init(pinned host fields) + %d x lbmhd_step + lbmhd_moments(pinned host out)" % args.steps},
        "gpu_launches": int(launches), "clocks": sampler.result(),
    }
    if world == 1 and not args.no_cpu_baseline:
        mlups, cores, sample, _, _ = oracle_leg(args.workload, 10 ** 9, 1, budget_s=args.cpu_seconds, scheme=args.scheme, lattice=args.lattice)
        line["cpu_baseline"] = {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_slab(args, rank, world, local_rank, dev):
    """N > 1 with a real exchange: ONE lattice, config 5 stacked `world` times along z (weak scaling: 384x256x256 owned
    cells per rank), cut into z-slabs with one ghost plane per cut face; per step one paired send/recv of the 5 x 8
    crossing populations per face.  Opt-in: this path could not be run on more than one GPU here."""
    import torch
    import torch.distributed as dist
    from paper_2606_00641_b200 import slab, workloads as W
    nx, ny, nz1 = (384, 256, 256) if args.shape is None else tuple(int(v) for v in args.shape.split("x"))
    shape = (nx, ny, nz1 * world)
    meta = W.config5(shape=(nx, ny, 4), planes=[0])          # parameters only; the fields are built per slab below
    meta["shape"] = shape
    meta["sphere"]["centre"] = np.array([nx / 3.0, ny / 2.0, shape[2] / 2.0])
    geo = slab.local_geometry(shape, meta["bc"], rank, world)
    local = W.config5(shape=shape, planes=geo["take"])
    meta["sphere"] = local["sphere"]
    sl = slab.Slab(meta, rank, world, precision=args.precision, device=local_rank)
    via_host = args.backend != "nccl"
    F = torch.as_tensor(local["fields"]).to(dev)
    sl.init_local(F)
    for _ in range(args.warmup):
        slab.exchange_distributed(sl, dist, via_host=via_host)
        sl.sim.step(1)
    dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = sl.sim.launch_count
    st = sl.sim.stream
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(args.steps):
        slab.exchange_distributed(sl, dist, via_host=via_host)
        sl.sim.step(1)
    e1.record(st)
    dist.barrier()
    torch.cuda.synchronize(dev)
    sampler.stop_flag = True
    sampler.join()
    launches = sl.sim.launch_count - l0
    ms_total = max_over_ranks([e0.elapsed_time(e1)], world, dev if args.backend == "nccl" else None)[0]
    slab.exchange_distributed(sl, dist, full=True, via_host=via_host)
    _, dg = sl.sim.moments(want_fields=False)
    flag = max_over_ranks([float(dg[-1])], world, dev if args.backend == "nccl" else None)[0]
    if rank == 0:
        if flag != 0:
            raise SystemExit("bench.py: numerical failure flag %g after the timed run" % flag)
        N = nx * ny * nz1
        K, Q = sl.sim.K, sl.sim.Q
        bpc = 2 * K * Q * (8 if args.precision == 64 else 4)
        peak, peak_src = load_peaks()
        ms_step = ms_total / args.steps
        halo = int(sl.sim.lib.lbmhd_halo_bytes(sl.sim.h, 0))
        line = {"metric": METRIC, "value": aggregate_mlups(N, args.steps, ms_total, world), "unit": "MLUPS", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic",
                "config": {"workload": "C5 stacked %d x along z: one %dx%dx%d lattice in %d z-slabs, halo exchange of %d B per face "
                                       "per step (%s)" % (world, nx, ny, shape[2], world, halo, args.backend),
                           "cells": N * world, "streaming": "A/B double buffer"},
                "roofline": {"bound": "hbm", "achieved": N * bpc / (ms_step * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                             "frac": N * bpc / (ms_step * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                             "kernel": "step_kernel (per rank, exchange included in the step time)"},
                "e2e": {"value": None, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                        "what": "not measured in slab mode"},
                "gpu_launches": int(launches), "clocks": sampler.result()}
        print(json.dumps(line), flush=True)
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--scheme", default=None, choices=["IDEAL_DIVB", "RESIST", "FULL"],
                    help="run the ideal-MHD workload on a scheme with transported gradient sets (DESIGN.md A19, A22, A23)")
    ap.add_argument("--lattice", default=None, choices=["D2Q5", "D3Q7"], help="the paper's own lattice instead of D2Q9 / D3Q19")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--streaming", default="ab", choices=["ab", "inplace"])
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default) or one lattice in z-slabs with halo exchange")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="gloo + host staging is for tests only")
    ap.add_argument("--shape", default=None, help="slab mode: per-rank owned shape nx x ny x nz (default 384x256x256)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "native" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_native(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
