#!/usr/bin/env python
"""bench.py — MLUPS and achieved HBM GB/s of the fused VLBM MHD step (BASELINE.json metric).

  python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload C5]

One "step" = one pass of the whole hot path (one lbmhd_step) over the resident workload.
N = 1 runs BASELINE config 5 (3D ideal MHD, D3Q19 x 8 sets, fp64, 384x256x256, moving magnetised sphere), the configuration
the north_star target is quoted on, with in-place (AA pattern) streaming — north_star's population storage — as the headline
and the A/B double-buffer layout measured beside it in the same run ("other_layout").  The timed region (exactly K steps,
CUDA events on the launching stream) is repeated 3 times: `value` / `ms_per_step` are the MEDIAN repeat, the minimum is
reported too (SURVEY.md:555-557).
N > 1 (torchrun): ONE lattice cut into z-slabs, one per rank, halo exchange over torch.distributed (NCCL) overlapped with the
interior update; `--decomp replicas` runs N independent replicas instead.
--impl reference times the CPU oracle (oracle/) on the host cores; the native arm's `cpu_baseline` is that same command run
as a child process BEFORE any GPU work (clean process, threads bound to cores), so the two agree.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "MLUPS (fused VLBM MHD stream-collide step)"
HALF_C5 = (192, 128, 128)      # the oracle's sample of config 5 (half-scale domain when the full one is too slow)
REPEATS = 3
KERNEL_NAMES = {0: "step_kernel", 1: "step_kernel_multi", 2: "step_kernel_cl", 3: "step_kernel_tma", 4: "step_kernel_persist", 5: "step_kernel_cell",
                6: "step_kernel_resident"}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


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
            time.sleep(0.02)

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
    """whole-job throughput: every rank advanced its own cells `steps` times in `ms` (max over ranks)"""
    return world * cells_per_rank * steps / (ms * 1e-3) / 1e6


def bench_workload(args, small=False):
    from paper_2606_00641_b200 import workloads as W
    w = W.get(args.workload, small=small)
    return W.variant(w, scheme=args.scheme, lattice=args.lattice)


# ---------------------------------------------------------------------------------------------------------
# the oracle arm (--impl reference; also the native arm's cpu_baseline, as a child process)
# ---------------------------------------------------------------------------------------------------------
def oracle_sample(args):
    """the bounded sample of the workload the oracle is timed on: C5 at half scale, C1-C4 at their own size"""
    from paper_2606_00641_b200 import workloads as W
    if args.workload == "C5":
        w = W.config5(shape=HALF_C5)
        what = "C5 at half scale 192x128x128, R = 12 (same recipe; the full 384x256x256 needs 61 GB and ~3 s per oracle step)"
    else:
        w = W.get(args.workload)
        what = "%s at its full size %s" % (args.workload, "x".join(str(s) for s in w["shape"]))
    return W.variant(w, scheme=args.scheme, lattice=args.lattice), what


def time_oracle(o, N, steps, warmup, budget_s=None):
    o.step(max(warmup, 1))
    t0 = time.perf_counter()
    done = 0
    while done < steps:
        o.step(1)
        done += 1
        if budget_s is not None and done >= 3 and time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return N * done / dt / 1e6, dt / done * 1e3, done


def run_reference(args, rank):
    """the CPU oracle, as it stands, on the host cores: all cores (the line's value) and one thread"""
    if rank != 0:
        return
    if os.environ.get("OMP_PROC_BIND") is None or os.environ.get("OMP_PLACES") is None:
        # bind the OpenMP threads to cores: the binding is read when libgomp loads, so re-exec with it set
        env = dict(os.environ, OMP_PROC_BIND="close", OMP_PLACES="cores")
        os.execve(sys.executable, [sys.executable] + sys.argv, env)
    from oracle import oracle as orc
    w, what = oracle_sample(args)
    N = int(np.prod(w["shape"]))
    o = orc.from_workload(w)
    o.init(w["fields"])
    cores = orc.get_threads()
    mlups, ms, done = time_oracle(o, N, args.steps, args.warmup, budget_s=args.cpu_seconds)
    orc.set_threads(1)
    mlups1, ms1, done1 = time_oracle(o, N, 3, 1)
    orc.set_threads(0)
    o.close()
    sample = "%s; all cores: %d steps after %d warm-up; one thread: %d steps after 1 warm-up" % (what, done, max(args.warmup, 1), done1)
    cpu = {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample,
           "single_thread": {"value": mlups1, "unit": "MLUPS", "ms_per_step": ms1},
           "ms_per_step": ms, "cpu_model": cpu_model(), "host_cores": os.cpu_count(),
           "omp": {"OMP_PROC_BIND": os.environ.get("OMP_PROC_BIND"), "OMP_PLACES": os.environ.get("OMP_PLACES")}}
    line = {"impl": "reference", "metric": METRIC, "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
            "steps": done, "warmup": max(args.warmup, 1), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s (CPU oracle on a bounded sample)" % args.workload, "sample": sample, "cells": N},
            "cpu_baseline": cpu,
            "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline_child(args):
    """run `bench.py --impl reference` on the same workload in a clean child process (no torch, no pinned memory, no NVML
    thread; threads bound to cores) and return its cpu_baseline object"""
    cmd = [sys.executable, os.path.abspath(__file__), "--impl", "reference", "--workload", args.workload, "--steps", "20",
           "--warmup", "1", "--cpu-seconds", str(min(args.cpu_seconds, 12.0))]
    if args.scheme:
        cmd += ["--scheme", args.scheme]
    if args.lattice:
        cmd += ["--lattice", args.lattice]
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=900)
    for ln in r.stdout.splitlines():
        if ln.startswith("{"):
            return json.loads(ln)["cpu_baseline"]
    return {"value": None, "unit": "MLUPS", "kind": "oracle", "error": (r.stderr or "no output")[-300:]}


# ---------------------------------------------------------------------------------------------------------
# the native arm
# ---------------------------------------------------------------------------------------------------------
def timed_steps(sim, steps, repeats, barrier, torch):
    """`repeats` timed regions of exactly `steps` steps each, CUDA events on the launching stream -> list of ms"""
    out = []
    for _ in range(repeats):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(sim.stream)
        sim.step(steps)
        e1.record(sim.stream)
        barrier()
        out.append(e0.elapsed_time(e1))
    return out


def traffic_from_profiles(args, streaming):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture of this configuration, with
    its source: a constant of that capture, NOT a quantity measured in this run"""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path) or args.scheme or args.lattice:
        return None, None
    key = "%s%s%s" % (args.workload, "" if args.precision == 64 else "_fp32", "" if streaming == "ab" else "_inplace")
    with open(path) as f:
        rows = [r.split(",") for r in f.read().splitlines()[1:] if r and not r.startswith("#")]
    for cols in rows:
        if cols[0] == key:
            return float(cols[1]) + float(cols[2]), "profiles/traffic.csv row %s (ncu --set full capture %s; not re-measured in this run)" % (key, cols[3] if len(cols) > 3 else "r1")
    return None, None


def run_native(args, rank, world, local_rank):
    # the oracle first, in a child process, before this process touches CUDA
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_child(args)

    import torch
    import torch.distributed as dist
    from paper_2606_00641_b200 import lbmhd

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

    w = bench_workload(args)
    N = int(np.prod(w["shape"]))
    prec = args.precision
    es = 8 if prec == 64 else 4
    F_dev = torch.as_tensor(w["fields"]).to(dev)

    def leg(streaming):
        """device-resident timing of one streaming layout: inputs already in HBM"""
        # no per-cell solid field or porosity in these workloads: the workspace leaves that optional storage out
        sim = lbmhd.from_workload(w, precision=prec, device=local_rank, streaming=1 if streaming == "inplace" else 0, solid_fields=False)
        sim.init(F_dev)
        sim.step(args.warmup)
        sampler = ClockSampler(local_rank)
        sampler.start()
        l0 = sim.launch_count
        ms = timed_steps(sim, args.steps, REPEATS, barrier, torch)
        launches = sim.launch_count - l0
        sampler.stop_flag = True
        sampler.join()
        _, dg = sim.moments(want_fields=False)
        if dg[-1] != 0:
            raise SystemExit("bench.py: numerical failure flag %g after the timed run (%s)" % (dg[-1], streaming))
        return sim, ms, launches, sampler.result()

    head = args.streaming
    other = "ab" if head == "inplace" else "inplace"
    sim, ms_list, launches, clocks = leg(head)
    K, Q = sim.K, sim.Q
    bytes_per_cell = 2 * K * Q * es
    kernel = KERNEL_NAMES.get(sim.step_path, "?")
    ws_gb = round(sim.workspace.numel() / 1e9, 2)

    # ---- end to end through the C ABI with HOST buffers: init (H2D) + K steps + moments (D2H), on the headline layout ----
    F_host = torch.as_tensor(w["fields"]).pin_memory()
    out_host = torch.empty_like(F_host).pin_memory()
    diag_host = torch.empty(3 * K + 4, dtype=torch.float64).pin_memory()
    st = sim.stream
    sim.init(F_host)               # warm the path once
    sim.moments(out_host, diag_host)
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(st)
    sim.init(F_host)
    sim.step(args.steps)
    sim.moments(out_host, diag_host)
    t1.record(st)
    barrier()
    ms_e2e = t0.elapsed_time(t1)
    h2d = F_host.numel() * 8
    d2h = out_host.numel() * 8 + diag_host.numel() * 8
    sim.close()
    del sim, F_host, out_host

    other_res = None
    if not args.single_layout:
        sim2, ms2, _, _ = leg(other)
        other_res = (sorted(ms2), KERNEL_NAMES.get(sim2.step_path, "?"), round(sim2.workspace.numel() / 1e9, 2))
        sim2.close()
        del sim2
    del F_dev

    ms_sorted = sorted(ms_list)
    ms_med, ms_min = ms_sorted[len(ms_sorted) // 2], ms_sorted[0]
    ms_med, ms_min, ms_e2e = max_over_ranks([ms_med, ms_min, ms_e2e], world, dev)
    probes = None
    if rank == 0:
        probes = {"fp64_copy_GBs": lbmhd.copy_probe(1 << 27, reps=5, device=local_rank),
                  "fp64_triad_GBs": lbmhd.triad_probe(1 << 27, reps=5, device=local_rank)}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = load_peaks()
    ms_step = ms_med / args.steps
    value = aggregate_mlups(N, args.steps, ms_med, world)
    achieved = N * bytes_per_cell / (ms_step * 1e-3) / 1e9
    traffic, traffic_src = traffic_from_profiles(args, head)
    lay = {"inplace": "in-place AA pattern, one population copy", "ab": "A/B double buffer"}
    line = {
        "metric": METRIC, "value": value, "unit": "MLUPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if prec == 64 else "f32", "data": "synthetic",
        "config": {"workload": "%s: %s %s x %d sets, %s, %s, %d B/cell/step%s" % (
                       w["name"], w["scheme"], w["lattice"], K, "x".join(str(s) for s in w["shape"]),
                       "fp64" if prec == 64 else "fp32", bytes_per_cell, "; replicas per GPU, no collective" if world > 1 else ""),
                   "cells": N, "streaming": lay[head], "workspace_GB": ws_gb,
                   "l2": "populations %.2f GB vs 126 MB L2%s" % (
                       (1 if head == "inplace" else 2) * N * bytes_per_cell / 2 / 1e9,
                       ": no flush needed" if N * bytes_per_cell / 2 > 4 * 126e6 else ": the working set is (partly) L2 resident, the fraction is against HBM bandwidth all the same")},
        "repeats": {"n": REPEATS, "ms_per_step_median": ms_step, "ms_per_step_min": ms_min / args.steps,
                    "ms_per_step_all": [m / args.steps for m in ms_list], "value_at_min": aggregate_mlups(N, args.steps, ms_min, world)},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src, "kernel": kernel,
                     "algorithmic_bytes_per_launch": N * bytes_per_cell,
                     "frac_at_min": N * bytes_per_cell / (ms_min / args.steps * 1e-3) / 1e9 / peak,
                     "frac_of_nominal_8TBs": achieved / 8000.0,
                     "own_probes": probes, "frac_of_own_copy": achieved / probes["fp64_copy_GBs"],
                     "frac_of_own_triad": achieved / probes["fp64_triad_GBs"],
                     "paper_context": "98.9% (2D) / 75.8% (3D) of 680 GB/s BabelStream, RTX A5000 fp32 (PAPER.md:269)"},
        "e2e": {"value": aggregate_mlups(N, args.steps, ms_e2e, world), "unit": "MLUPS", "h2d_bytes_per_step": h2d / args.steps,
                "d2h_bytes_per_step": d2h / args.steps,
                "what": "lbmhd_init(pinned host fields) + %d x lbmhd_step + lbmhd_moments(pinned host out), %s" % (args.steps, lay[head])},
        "gpu_launches": int(launches), "gpu_launches_what": "%d timed regions x %d steps" % (REPEATS, args.steps),
        "clocks": clocks,
    }
    if other_res is not None:
        ms2, k2, ws2 = other_res
        m2 = ms2[len(ms2) // 2] / args.steps
        line["other_layout"] = {"streaming": lay[other], "ms_per_step": m2, "ms_per_step_min": ms2[0] / args.steps,
                                "value": N / (m2 * 1e-3) / 1e6 * world, "unit": "MLUPS",
                                "frac": N * bytes_per_cell / (m2 * 1e-3) / 1e9 / peak, "kernel": k2, "workspace_GB": ws2}
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_slab(args, rank, world, local_rank, dev):
    """N > 1: ONE lattice, config 5 stacked `world` times along z (weak scaling: 384x256x256 owned cells per rank), cut into
    z-slabs with one ghost plane per cut face.  Per step: the two boundary planes are updated first, their crossing
    populations (5 of 19 directions x 8 sets) packed and exchanged on a side stream while the interior planes are updated
    (DESIGN.md §8).  This path has not run on more than one GPU in this repo's history (no multi-GPU box was available)."""
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
    via_host = args.backend != "nccl"
    sl = slab.Slab(meta, rank, world, precision=args.precision, device=local_rank,
                   streaming=1 if args.streaming == "inplace" else 0)
    ex = slab.DistributedExchange(sl, dist, via_host=via_host, overlap=not args.no_overlap)
    F = torch.as_tensor(local["fields"]).to(dev)
    sl.init_local(F)
    ex.prime()
    for _ in range(args.warmup):
        ex.step()

    def barrier():
        dist.barrier()
        torch.cuda.synchronize(dev)

    red_dev = dev if args.backend == "nccl" else None
    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = sl.sim.launch_count
    st = sl.sim.stream
    ms_list = []
    for _ in range(REPEATS):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(args.steps):
            ex.step()
        ex.join()
        e1.record(st)
        barrier()
        ms_list.append(e0.elapsed_time(e1))
    sampler.stop_flag = True
    sampler.join()
    launches = sl.sim.launch_count - l0
    ms_sorted = sorted(ms_list)
    ms_med, ms_min = max_over_ranks([ms_sorted[len(ms_sorted) // 2], ms_sorted[0]], world, red_dev)
    dg = ex.diagnostics()
    flag = max_over_ranks([float(dg[-1])], world, red_dev)[0]
    if rank == 0:
        if flag != 0:
            raise SystemExit("bench.py: numerical failure flag %g after the timed run" % flag)
        N = nx * ny * nz1
        K, Q = sl.sim.K, sl.sim.Q
        bpc = 2 * K * Q * (8 if args.precision == 64 else 4)
        peak, peak_src = load_peaks()
        ms_step = ms_med / args.steps
        halo = int(sl.sim.lib.lbmhd_halo_bytes(sl.sim.h, 0))
        ach = N * bpc / (ms_step * 1e-3) / 1e9
        line = {"metric": METRIC, "value": aggregate_mlups(N, args.steps, ms_med, world), "unit": "MLUPS", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic",
                "config": {"workload": "C5 stacked %d x along z: one %dx%dx%d lattice in %d z-slabs, halo exchange of %d B per face "
                                       "per step (%s, %s)" % (world, nx, ny, shape[2], world, halo, args.backend,
                                                              "serial" if args.no_overlap else "overlapped with the interior update"),
                           "cells": N * world, "streaming": "in-place AA pattern" if args.streaming == "inplace" else "A/B double buffer",
                           "decomposition": "z-slabs, one ghost plane per cut face, paired send/recv per face and step"},
                "repeats": {"n": REPEATS, "ms_per_step_median": ms_step, "ms_per_step_min": ms_min / args.steps},
                "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                             "peak_source": peak_src,
                             "kernel": "%s per rank; exchange inside the timed step" % KERNEL_NAMES.get(sl.sim.step_path, "?")},
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
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C2i", "C3", "C4", "C5"])
    ap.add_argument("--scheme", default=None, choices=["IDEAL_DIVB", "RESIST", "FULL"],
                    help="run the ideal-MHD workload on a scheme with transported gradient sets (DESIGN.md A19, A22, A23)")
    ap.add_argument("--lattice", default=None, choices=["D2Q5", "D3Q7"], help="the paper's own lattice instead of D2Q9 / D3Q19")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--streaming", default="inplace", choices=["ab", "inplace"],
                    help="headline population storage: in-place AA pattern (north_star's layout, default) or A/B double buffer")
    ap.add_argument("--single-layout", action="store_true", help="do not measure the other streaming layout beside the headline")
    ap.add_argument("--decomp", default="slab", choices=["replicas", "slab"],
                    help="N > 1: one lattice in z-slabs with halo exchange (default) or independent replicas")
    ap.add_argument("--no-overlap", action="store_true", help="slab mode: serial exchange-then-step schedule")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="gloo + host staging is for tests only")
    ap.add_argument("--shape", default=None, help="slab mode: per-rank owned shape nx x ny x nz (default 384x256x256)")
    ap.add_argument("--cpu-seconds", type=float, default=60.0, help="time budget of the oracle's all-core leg (it stops after >= 3 steps once over it)")
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
