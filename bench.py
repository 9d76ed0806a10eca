#!/usr/bin/env python
"""bench.py -- throughput of the viscoelastic FDTD step on B200, in BASELINE.json's metric.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one full FDTD time step (S1 inject -> S2 velocity -> S3 stress + S4 sensor) over the
whole grid of the workload (default: config 2, 300x300x450, the configuration the metric is quoted
on).  Prints ONE JSON line.  See DESIGN.md "Measurement" for the definitions:

  value       Gcell-updates/s = cells * K / device time (CUDA events, max over ranks), inputs and
              state resident in HBM; 2.4 GB of state per step >> 126 MB L2, so no flush is needed.
  e2e         the same metric through the public API with HOST buffers: bvfdtd_create (H2D of the
              index map and tables) + bvfdtd_set_source + bvfdtd_step(K) + bvfdtd_read_peak_pressure
              into pinned host memory, wall clock around the whole sequence.
  roofline    the dominant kernel (stress + sensor): algorithmic bytes per launch / mean launch
              duration measured live with CUDA events on the context's stream.
  cpu_baseline the fp64 oracle, as it stands, timed on this box's host cores on a bounded sample.

Multi-GPU (torchrun): the path does not shard in this build ("replicas only"): every rank
advances its own replica of the workload; value = N * cells * K / max-over-ranks time.
--impl reference times the oracle (the only "reference" there is: the paper ships no code).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gcell-updates/s per FDTD step (fp32)"
UNIT = "Gcell-updates/s"
HBM_FALLBACK_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic_bytes(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu summary."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(path):
            parts = [p.strip() for p in line.split(",")]
            if parts and parts[0] == kernel:
                return float(parts[1]) + float(parts[2])
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------------
# distributed plumbing (one process per GPU; the data path has no collective)
# ---------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), \
        int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def reduce_max(value, device="cpu"):
    """max over ranks of a python float (device timing -> whole-job time)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(cells_per_rank, steps, ms_local, world, device="cpu"):
    """Whole-job Gcell-updates/s: all ranks' cell-steps / the slowest rank's time."""
    ms = reduce_max(ms_local, device)
    return world * cells_per_rank * steps / (ms * 1e-3) / 1e9, ms


# ---------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = os.path.join("/tmp", f"bvfdtd_clocks_{os.getpid()}.csv")

    def start(self):
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in open(self.path):
            p = [x.strip() for x in line.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[1]))
                mx.append(float(p[2]))
            except ValueError:
                continue
            for n, v in zip(names, p[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        try:
            os.remove(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------------
# the oracle legs (the only places bench.py executes oracle/)
# ---------------------------------------------------------------------------------------------
def crop_workload(w, nx, ny, nz):
    """Centred sub-box of the workload's index map (same materials, PML, dt); the source is the
    part of the source list that falls in the box.  Used to bound the oracle's CPU time."""
    from paper_2301_12727_b200 import workloads as wl
    x0, y0 = (w.nx - nx) // 2, (w.ny - ny) // 2
    idx = np.ascontiguousarray(w.index_map[:nz, y0:y0 + ny, x0:x0 + nx])
    c = w.src_cell
    i, j, k = c % w.nx, (c // w.nx) % w.ny, c // (w.nx * w.ny)
    P = w.pml
    keep = (i >= x0 + P) & (i < x0 + nx - P) & (j >= y0 + P) & (j < y0 + ny - P) & (k >= P) & (k < nz - P)
    cells = ((i - x0) + nx * ((j - y0) + ny * k))[keep].astype(np.int64)
    return wl.Workload(f"{w.name}_crop{nx}x{ny}x{nz}", nx, ny, nz, P, w.dx, w.dt, w.f0, w.spp, w.steps,
                       w.table, idx, cells, w.src_amp[keep], w.src_delay[keep], w.waveform, w.f_src,
                       w.n_cycles, w.peak_begin, w.rms_begin, w.sensor_end, w.pml_R)


def oracle_rate(w, steps, warmup=0):
    """Gcell-updates/s of the oracle on workload w, wall clock around the step loop."""
    from oracle import fdtd_oracle as orc
    o = orc.Oracle.from_workload(w)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    return w.cells * steps / dt / 1e9, dt


def oracle_threads():
    n = os.environ.get("OMP_NUM_THREADS")
    return int(n) if n else (os.cpu_count() or 1)


def cpu_baseline_leg(w, budget_s=12.0):
    """The oracle on the full grid of the workload for as many of its first steps as fit the
    budget (calibrated on one step)."""
    from oracle import fdtd_oracle as orc
    o = orc.Oracle.from_workload(w)
    o.step(1)                                   # first touch of the arrays, untimed
    t0 = time.perf_counter()
    o.step(2)
    t1 = (time.perf_counter() - t0) / 2.0
    n = int(max(1, min(400, budget_s / max(t1, 1e-4))))
    t0 = time.perf_counter()
    o.step(n)
    dt = time.perf_counter() - t0
    o.close()
    return {"value": w.cells * n / dt / 1e9, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
            "sample": f"full {w.nx}x{w.ny}x{w.nz} grid of the workload, steps 4..{n + 3} of {w.steps} "
                      f"({dt:.1f} s wall, fp64, gcc -O2 -fopenmp)"}


def reference_arm(args):
    """--impl reference: the oracle timed on the host cores on a bounded sample of the workload."""
    from paper_2301_12727_b200 import workloads as wl
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    K, W = args.steps, args.warmup
    w = wl.make(args.config)
    # size the sample so that K + W steps take about a minute: calibrate on a small crop first
    lim = 2 * w.pml + 8
    cal = crop_workload(w, min(w.nx, 96), min(w.ny, 96), min(w.nz, 96))
    rate, _ = oracle_rate(cal, 3, warmup=1)                       # Gcell/s
    target_cells = rate * 1e9 * 60.0 / max(1, K + W)
    n = int(round(target_cells ** (1.0 / 3.0)))
    sx, sy, sz = (int(min(full, max(lim, n))) for full in (w.nx, w.ny, w.nz))
    s = crop_workload(w, sx, sy, sz)
    from oracle import fdtd_oracle as orc
    o = orc.Oracle.from_workload(s)
    o.step(W)
    t0 = time.perf_counter()
    o.step(K)
    dt = time.perf_counter() - t0
    o.close()
    value = s.cells * K / dt / 1e9
    sample = (f"centred {sx}x{sy}x{sz} sub-box of {w.name} (same materials, PML {w.pml}, dt), "
              f"{K} steps, fp64 oracle, gcc -O2 -fopenmp")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": K, "warmup": W, "ms_per_step": dt * 1e3 / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "pml": w.pml,
                   "sample_grid": [sx, sy, sz]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def kernel_bytes(w, rms_on):
    """Algorithmic bytes per launch: per cell 49 B (S2) and
    109 B + 8 (peak) + 8 (sumsq when on) (S3+S4), plus 24 B per PML mask bit in each pass."""
    bits = w.mean_mask_bits()
    vel = (49.0 + 24.0 * bits) * w.cells
    st = (109.0 + 8.0 + (8.0 if rms_on else 0.0) + 24.0 * bits) * w.cells
    return vel, st


def ours(args):
    import torch
    from paper_2301_12727_b200 import build as bv_build
    from paper_2301_12727_b200 import workloads as wl

    rank, local_rank, world = dist_env()
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("launch with torchrun --nproc-per-node N for --gpus N")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist_init("nccl")
    if rank == 0:
        bv_build.build()
    barrier()
    from paper_2301_12727_b200 import binding as bv

    K, W = args.steps, args.warmup
    w = wl.make(args.config)
    total = W + K
    # sensor windows follow the run length: running peak throughout, steady-state amplitude over
    # the last 3 periods of the timed run (config 2's "last 3 periods")
    w.steps = total
    w.rms_begin = max(0, total - 3 * w.spp) if args.config in (1, 2, 3) else -1
    flags = bv.FLAG_REFERENCE_KERNELS if args.reference_kernels else 0
    if args.dense:
        flags |= bv.FLAG_DENSE

    # ---- device-resident timing -----------------------------------------------------------
    sim = bv.Simulation.from_workload(w, flags=flags, device=dev)
    sim.step(W)
    sim.synchronize()
    sim.enable_kernel_timing(True)
    clocks = ClockSampler(local_rank)
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record()
    sim.step(K)
    e1.record()
    torch.cuda.synchronize()
    barrier()
    ms_local = e0.elapsed_time(e1)
    clk = clocks.stop()
    kt = sim.kernel_times()
    value, ms = aggregate_rate(w.cells, K, ms_local, world, dev)
    peak_dev, _ = sim.read_peak_pressure_device()
    finite = bool(torch.isfinite(peak_dev).all()) and float(peak_dev.max()) > 0.0
    del peak_dev
    sim.close()
    del sim
    torch.cuda.empty_cache()

    # ---- end to end through the C ABI with host buffers -------------------------------------
    nbytes = bv.workspace_bytes(w.nx, w.ny, w.nz, w.pml)
    pinned_idx = torch.from_numpy(w.index_map.copy()).pin_memory()
    pinned_peak = torch.empty(w.index_map.shape, dtype=torch.float32).pin_memory()
    idx_np, peak_np = pinned_idx.numpy(), pinned_peak.numpy()
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    sim = bv.Simulation(w.nx, w.ny, w.nz, w.pml, w.dx, w.dt, w.table, idx_np, w.f0, w.pml_R,
                        w.peak_begin, w.rms_begin, w.sensor_end, flags=flags, device=dev)
    sim.set_source(w.src_cell, w.src_amp, w.src_delay, w.waveform, w.f_src, w.n_cycles)
    sim.step(total)
    sim.read_peak_pressure(peak=True, rms=False, out_peak=peak_np)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_ms = reduce_max(e2e_s * 1e3, dev)
    h2d = w.index_map.nbytes + 256 * 32 + 4 * 4 * (w.nx + w.ny + w.nz) + w.src_cell.size * 16
    d2h = peak_np.nbytes
    e2e_value = world * w.cells * total / (e2e_ms * 1e-3) / 1e9
    sim.close()

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel -----------------------------------------------------
    peak_gbs, peak_src = measured_hbm_peak()
    vel_b, st_b_off = kernel_bytes(w, False)
    _, st_b_on = kernel_bytes(w, True)
    n_rms = min(K, max(0, total - max(w.rms_begin, W))) if w.rms_begin >= 0 else 0
    st_b = (st_b_on * n_rms + st_b_off * (K - n_rms)) / K
    kern = {}
    for name, b in (("velocity", vel_b), ("stress_sensor", st_b)):
        n = max(1, kt[name]["launches"])
        avg_ms = kt[name]["ms"] / n
        kern[name] = {"avg_ms": avg_ms, "launches": kt[name]["launches"],
                      "algorithmic_bytes": b, "achieved_gbs": b / (avg_ms * 1e-3) / 1e9 if avg_ms > 0 else None}
    kern["inject"] = {"avg_ms": kt["inject"]["ms"] / max(1, kt["inject"]["launches"]),
                      "launches": kt["inject"]["launches"]}
    dom = "stress_sensor"
    ach_dense = kern[dom]["achieved_gbs"]
    step_bytes = vel_b + st_b
    step_gbs = step_bytes / (ms / K * 1e-3) / 1e9
    min_step_bytes = w.min_bytes_per_cell_step(rms_frac=n_rms / K) * w.cells
    have_ncu = args.config == 2 and not args.dense and not args.reference_kernels
    step_traffic = dom_traffic = None
    if have_ncu:
        tv, ts = ncu_traffic_bytes("velocity"), ncu_traffic_bytes("stress_sensor")
        if tv and ts:
            # the capture had both sensor maps on: take the sum-of-squares map (8 B per cell, read + write)
            # off for the timed steps outside the rms window, so bytes and times describe the same launches
            dom_traffic = ts - 8.0 * w.cells * (1.0 - n_rms / K)
            step_traffic = tv + dom_traffic
    # SURVEY.md 8(d) "reporting rule (no inflation)": the achieved rate never credits bytes the kernel
    # skipped: min(B_dense rate, measured DRAM rate).  Without an ncu capture of this workload the
    # class-aware minimum B_min (what the data forces the pass to move) stands in for the traffic.
    if args.dense or args.reference_kernels:
        ach, rule = ach_dense, "B_dense bytes / CUDA-event time (the dense sweep moves every array)"
    elif dom_traffic:
        ach = min(ach_dense, dom_traffic / (kern[dom]["avg_ms"] * 1e-3) / 1e9)
        rule = "min(B_dense bytes, ncu-measured DRAM bytes of this kernel on this workload) / CUDA-event time"
    else:
        ach = ach_dense * min(1.0, min_step_bytes / step_bytes)
        rule = "B_dense bytes scaled by the step's class-aware minimum B_min / B_dense (no ncu capture of this workload) / CUDA-event time"
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak_gbs, "unit": "GB/s",
                "frac": ach / peak_gbs if ach else None,
                "traffic": dom_traffic,
                "rule": rule,
                "bytes_definition": "B_dense of SURVEY.md 8(d): every array of every cell once per pass; the default "
                                    "path moves fewer bytes where shear stresses / memory variables are identically "
                                    "zero (traffic = ncu-measured DRAM bytes of the same kernel, profiles/traffic.md)",
                "algorithmic_bytes_per_launch": st_b,
                "achieved_b_dense": ach_dense, "frac_b_dense": ach_dense / peak_gbs if ach_dense else None,
                "class_aware_min_bytes_per_step": min_step_bytes,
                "peak_source": peak_src + ", burst copy figure",
                "step": {"algorithmic_bytes": step_bytes, "achieved_gbs": step_gbs,
                         "frac_of_measured": step_gbs / peak_gbs, "frac_of_8TBs": step_gbs / 8000.0,
                         # SURVEY.md 8(d) reporting rule: min(B_dense rate, measured DRAM rate) / 8 TB/s
                         "measured_dram_gbs": step_traffic / (ms / K * 1e-3) / 1e9 if step_traffic else None,
                         "frac_of_measured_min_rule": min(step_gbs, step_traffic / (ms / K * 1e-3) / 1e9) / peak_gbs
                         if step_traffic else None,
                         "frac_of_8TBs_min_rule": min(step_gbs, step_traffic / (ms / K * 1e-3) / 1e9) / 8000.0
                         if step_traffic else None},
                "kernels": kern}

    cpu = cpu_baseline_leg(wl.make(args.config)) if (world == 1 and not args.no_cpu_baseline) else None

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "pml": w.pml, "cells": w.cells,
                   "materials": int(w.table.shape[0]), "source_cells": int(w.src_cell.size),
                   "parallelism": f"replicas x{world} (no sharding)",
                   "l2": "state 2.4 GB per step >> 126 MB L2: inputs larger than L2, no flush",
                   "kernels": "reference (one thread per cell)" if args.reference_kernels else
                              ("tiled, dense sweep" if args.dense else "tiled, tile-class skipping"),
                   "result_finite_nonzero": finite},
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d / total,
                "d2h_bytes_per_step": d2h / total, "steps": total, "seconds": e2e_ms * 1e-3,
                "what": "bvfdtd_create + set_source + step(W+K) + read_peak_pressure to pinned host"},
        "gpu_launches": int(sum(kt[k]["launches"] for k in kt)),
        "roofline": roofline,
    }
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--reference-kernels", action="store_true",
                    help="debug: time the one-thread-per-cell kernels")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dense", action="store_true",
                    help="BVFDTD_FLAG_DENSE: sweep every array everywhere (no tile-class skipping)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return reference_arm(args)
    return ours(args)


if __name__ == "__main__":
    sys.exit(main())
