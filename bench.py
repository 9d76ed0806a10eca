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


TRAFFIC_CSV = os.path.join(ROOT, "profiles", "traffic.csv")
KERNEL_CLASSES = (("fused", "k_fluid_fused"), ("velocity", "k_velocity_tiled"), ("stress_sensor", "k_stress_tiled"))


def kernel_source_hash():
    """sha256 over the hot-path kernel sources and the nvcc flags of the library being timed: profiles/traffic.csv names
    the hash it was captured for, and a capture of other code is refused."""
    import hashlib
    from paper_2301_12727_b200 import build as bv_build
    h = hashlib.sha256()
    for f in ("device_params.hpp", "kernels_tiled.cuh", "kernels_fused.cuh"):      # the hot kernels and their work lists
        h.update(f.encode())
        h.update(open(os.path.join(bv_build.CSRC, f), "rb").read())
    h.update(" ".join(bv_build.NVCC_FLAGS).encode())
    return h.hexdigest()[:16]


def ncu_traffic(config):
    """({kernel: dram read + write bytes per launch}, source note) from the committed ncu summary of THIS build
    on workload `config`; ({}, why) when the capture belongs to other kernel sources or another workload."""
    want = kernel_source_hash()
    try:
        lines = [ln.strip() for ln in open(TRAFFIC_CSV)]
    except OSError:
        return {}, "no profiles/traffic.csv"
    have = None
    out = {}
    for ln in lines:
        if ln.startswith("#"):
            if "kernel_hash=" in ln:
                have = ln.split("kernel_hash=")[1].split()[0]
            continue
        parts = [p.strip() for p in ln.split(",")]
        if len(parts) >= 4 and parts[0] == str(config):
            out[parts[1]] = float(parts[2]) + float(parts[3])
    if have != want:
        return {}, f"profiles/traffic.csv is a capture of kernel hash {have}; the library timed here is {want}: refused"
    if not out:
        return {}, f"profiles/traffic.csv (kernel hash {have}) holds no capture of config {config}"
    return out, f"profiles/traffic.csv, ncu --set full capture of this build (kernel hash {have}), config {config}"


def traffic_from_ncu(raw_csv, config):
    """`bench.py --traffic-from <ncu -i x.ncu-rep --page raw --csv> --config C`: average dram__bytes_read.sum /
    dram__bytes_write.sum per launch of each hot kernel into profiles/traffic.csv, stamped with the kernel hash."""
    import csv
    rows = list(csv.reader(open(raw_csv)))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[hdr], rows[hdr + 1]
    col = {n: i for i, n in enumerate(names)}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    acc = {}
    for r in rows[hdr + 2:]:
        if len(r) <= col["dram__bytes_write.sum"]:
            continue
        for cls, pat in KERNEL_CLASSES:
            if pat in r[col["Kernel Name"]]:
                rd = float(r[col["dram__bytes_read.sum"]]) * scale[units[col["dram__bytes_read.sum"]]]
                wr = float(r[col["dram__bytes_write.sum"]]) * scale[units[col["dram__bytes_write.sum"]]]
                a = acc.setdefault(cls, [0.0, 0.0, 0])
                a[0] += rd; a[1] += wr; a[2] += 1
                break
    want = kernel_source_hash()
    keep = []
    try:
        old = [ln.rstrip("\n") for ln in open(TRAFFIC_CSV)]
        if any(ln.startswith("#") and f"kernel_hash={want}" in ln for ln in old):
            keep = [ln for ln in old if not ln.startswith("#") and ln.strip() and ln.split(",")[0].strip() != str(config)]
    except OSError:
        pass
    with open(TRAFFIC_CSV, "w") as f:
        f.write(f"# kernel_hash={want}  columns: config, kernel, dram__bytes_read.sum, dram__bytes_write.sum (bytes per launch, mean), launches\n")
        for ln in keep:
            f.write(ln + "\n")
        for cls, (rd, wr, n) in sorted(acc.items()):
            f.write(f"{config},{cls},{rd / n:.0f},{wr / n:.0f},{n}\n")
    print(open(TRAFFIC_CSV).read())
    return 0


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
    """SM clock and clock-event reasons sampled DURING the timed region: NVML in-process every 2 ms (a 20-step
    run lasts ~15 ms, too short for nvidia-smi's own loop), `nvidia-smi -lms` as the fallback."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index, uuid=None):
        self.index, self.uuid = index, uuid
        self.proc = self.thread = None
        self.path = os.path.join("/tmp", f"bvfdtd_clocks_{os.getpid()}.csv")
        self.sm, self.reasons, self.sm_max, self.power = [], set(), None, []

    def _nvml_loop(self, nv, h):
        names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksEventReasonHwPowerBrakeSlowdown: "hw_power_brake_slowdown"}
        while not self._stop:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                for bit, n in names.items():
                    if r & bit:
                        self.reasons.add(n)
                self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        try:
            import threading
            import pynvml as nv
            nv.nvmlInit()
            h = None
            if self.uuid:
                try:
                    h = nv.nvmlDeviceGetHandleByUUID(("GPU-" + str(self.uuid)).encode())
                except Exception:
                    h = None
            if h is None:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                ids = [v for v in vis.split(",") if v.strip().isdigit()]
                h = nv.nvmlDeviceGetHandleByIndex(int(ids[self.index]) if self.index < len(ids) else self.index)
            self.sm_max = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            self._stop = False
            self.thread = threading.Thread(target=self._nvml_loop, args=(nv, h), daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                 "-i", str(self.index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.thread is not None:
            self._stop = True
            self.thread.join(timeout=2)
            if self.sm:
                out.update(sm_mhz=float(np.median(self.sm)), sm_max_mhz=self.sm_max, reasons=sorted(self.reasons),
                           samples=len(self.sm), power_w_max=max(self.power) if self.power else None,
                           how="NVML in-process, 2 ms period, over the timed region")
            return out
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
                       reasons=sorted(reasons), samples=len(sm), how="nvidia-smi -lms 20")
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
# the kernels beyond the hot path: `--next`, and "next_rows" of the default line
# ---------------------------------------------------------------------------------------------
def next_rows(dev):
    """One row per NEXT kernel, timed with CUDA events after warm-up.
    NEXT-1 k_rayleigh: config 2's focused bowl (aperture 64 mm, F# 1) decomposed at lambda/4 on the
    whole 300 x 300 entry plane; SFU-bound, 3 MUFU operations (rsqrt, sin, cos) per (source, receiver) pair: peak =
    the MUFU rate measured by bvfdtd_probe_mufu on this device / 3.
    NEXT-4 k_bhte: thermal step on config 2's grid; HBM-bound, 21 B per cell-step (rise read + write, Q, dose read +
    write, material byte), 29 B with the running maximum; peak = the measured copy bandwidth."""
    import math
    import torch
    from paper_2301_12727_b200 import binding as bv
    from paper_2301_12727_b200 import workloads as wl
    rows = []
    f, c0, rho0 = 500e3, 1500.0, 1000.0
    pos, area = wl.bowl_elements(64e-3, 64e-3, c0 / f / 4)
    dx = 1e-3 / 3.0
    xs = (np.arange(300) - 149.5) * dx
    X, Y = np.meshgrid(xs, xs)
    rcv = np.stack([X.ravel(), Y.ravel(), np.full(X.size, 15e-3)], axis=1)
    s = torch.from_numpy(pos.astype(np.float32)).to(dev)
    wg = torch.from_numpy(np.stack([0.01 * area, np.zeros_like(area)], axis=1).astype(np.float32)).to(dev)
    r = torch.from_numpy(rcv.astype(np.float32)).to(dev)
    out = torch.empty((4, r.shape[0]), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream

    def launch():
        bv._check(bv.lib().bvfdtd_rayleigh(s.shape[0], s.data_ptr(), wg.data_ptr(), r.shape[0], r.data_ptr(), f, c0, rho0,
                                           out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), out[3].data_ptr(),
                                           stream), "bvfdtd_rayleigh")
    for _ in range(40):                 # (the GPU idled through the CPU baseline: let the clocks come back up)
        launch()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    reps = 20
    e0.record()
    for _ in range(reps):
        launch()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    pairs = float(s.shape[0]) * float(r.shape[0])
    mufu = bv.probe_mufu(dev)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    rows.append({"kernel": "k_rayleigh", "workload": f"{s.shape[0]} bowl elements x {r.shape[0]} receivers", "ms": ms,
                 "value": pairs / (ms * 1e-3) / 1e9, "unit": "Gpair/s",
                 "roofline": {"bound": "alu", "achieved": pairs / (ms * 1e-3) / 1e9, "peak": mufu / 3.0 / 1e9, "unit": "Gpair/s",
                              "frac": pairs / (ms * 1e-3) / (mufu / 3.0),
                              "peak_source": f"MUFU rate measured by bvfdtd_probe_mufu ({mufu / 1e12:.2f} Top/s = "
                                             f"{mufu / sms / 1.965e9:.1f} per SM per clock at 1965 MHz) / 3 MUFU per pair"}})
    del s, wg, r, out
    hbm, _ = measured_hbm_peak()
    tw = wl.thermal_config2()
    cells = tw["nx"] * tw["ny"] * tw["nz"]
    for track_max in (False, True):
        th = bv.Bhte(tw["nx"], tw["ny"], tw["nz"], tw["dx"], tw["dt"], tw["table"], tw["index_map"], track_max=track_max, device=dev)
        th.set_heat(tw["Q"])
        th.step(5, tw["duty"])
        torch.cuda.synchronize()
        reps = 50
        e0.record()
        th.step(reps, tw["duty"])
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        b = 29.0 if track_max else 21.0
        gbs = cells * b / (ms * 1e-3) / 1e9
        rows.append({"kernel": "k_bhte<%s>" % ("true" if track_max else "false"),
                     "workload": "thermal step on config 2's grid (300x300x450, 128 materials), %d launches" % reps,
                     "ms": ms, "value": cells / (ms * 1e-3) / 1e9, "unit": "Gcell-updates/s",
                     "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
                                  "bytes_per_cell_step": b}})
        th.close()
        del th
        torch.cuda.empty_cache()
    return rows


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
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

    # ---- device-resident timing: the call a user makes, bvfdtd_step(K) (CUDA-graph replay) ------
    sim = bv.Simulation.from_workload(w, flags=flags, device=dev, tuning=args.tuning)
    kernels_desc = sim.kernel_mode()
    mode_bits = sim.mode_bits()
    coverage = sim.fused_coverage()
    sim.step(W)
    sim.synchronize()
    try:
        uuid = torch.cuda.get_device_properties(dev).uuid
    except Exception:
        uuid = None
    clocks = ClockSampler(local_rank, uuid)
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
    value, ms = aggregate_rate(w.cells, K, ms_local, world, dev)
    peak_dev, _ = sim.read_peak_pressure_device()
    finite = bool(torch.isfinite(peak_dev).all()) and float(peak_dev.max()) > 0.0
    del peak_dev
    sim.close()
    del sim

    # ---- the same W + K steps once more, kernel by kernel with CUDA events between the launches (the
    #      library's own events on the context's stream): per-kernel durations for the roofline ----
    sim = bv.Simulation.from_workload(w, flags=flags, device=dev, tuning=args.tuning)
    sim.step(W)
    sim.synchronize()
    sim.enable_kernel_timing(True)
    t0e, t1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0e.record()
    sim.step(min(K, 4096))
    t1e.record()
    torch.cuda.synchronize()
    kt = sim.kernel_times()
    ms_timed_pass = t0e.elapsed_time(t1e) / min(K, 4096)
    sim.close()
    del sim
    torch.cuda.empty_cache()

    # ---- end to end through the C ABI with host buffers -------------------------------------
    nbytes = bv.workspace_bytes(w.nx, w.ny, w.nz, w.pml)
    pinned_idx = torch.from_numpy(w.index_map.copy()).pin_memory()
    pinned_peak = torch.empty(w.index_map.shape, dtype=torch.float32).pin_memory()
    idx_np, peak_np = pinned_idx.numpy(), pinned_peak.numpy()
    def e2e_pass():
        barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sim = bv.Simulation(w.nx, w.ny, w.nz, w.pml, w.dx, w.dt, w.table, idx_np, w.f0, w.pml_R,
                            w.peak_begin, w.rms_begin, w.sensor_end, flags=flags, device=dev, tuning=args.tuning)
        sim.set_source(w.src_cell, w.src_amp, w.src_delay, w.waveform, w.f_src, w.n_cycles)
        sim.step(total)
        sim.read_peak_pressure(peak=True, rms=False, out_peak=peak_np)
        torch.cuda.synchronize()
        dt_s = time.perf_counter() - t0
        sim.close()
        return dt_s

    e2e_cold_s = e2e_pass()          # first pass: the allocator's cudaMalloc of the workspace, first graph instantiation
    e2e_s = e2e_pass()               # timed pass (the warm-up rule applies to this leg too)
    e2e_ms = reduce_max(e2e_s * 1e3, dev)
    h2d = w.index_map.nbytes + 256 * 32 + 4 * 4 * (w.nx + w.ny + w.nz) + w.src_cell.size * 16
    d2h = peak_np.nbytes
    e2e_value = world * w.cells * total / (e2e_ms * 1e-3) / 1e9

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel -----------------------------------------------------
    # Algorithmic bytes.  The two passes: B_dense of SURVEY.md 8(d) (49 B + 109 B + sensors +
    # psi per cell) over the cells they process.  The fused sweep: what ONE sweep over an all-fluid cell must move:
    # sigma_xx and v read + write 32 B, index 1 B, r_xx 8 B in lossy cells, 8 B per active sensor map, 16 B per PML
    # mask bit (one psi per pass direction).  traffic = ncu-measured DRAM bytes of the same kernel on the same
    # workload with this build (profiles/traffic.csv, refused unless its kernel hash matches).  achieved never
    # credits bytes that were not moved: min(algorithmic, traffic) / CUDA-event time.
    peak_gbs, peak_src = measured_hbm_peak()
    n_rms = min(K, max(0, total - max(w.rms_begin, W))) if w.rms_begin >= 0 else 0
    rms_frac = n_rms / K
    bits = w.mean_mask_bits()
    fluid = w.table[w.index_map, 2] == 0
    lossy_fluid_frac = float(((w.table[w.index_map, 3] > 0) & fluid).sum() / max(1, fluid.sum()))
    cells_f = coverage * w.cells                        # cells of the fused tile columns (tile-plane fraction x cells)
    cells_2 = w.cells - cells_f
    alg = {"fused": (33.0 + 8.0 * lossy_fluid_frac + 8.0 + 8.0 * rms_frac + 16.0 * bits) * cells_f,
           "velocity": (49.0 + 24.0 * bits) * cells_2,
           "stress_sensor": (109.0 + 8.0 + 8.0 * rms_frac + 24.0 * bits) * cells_2}
    if args.dense or args.reference_kernels:
        traffic, traffic_source = {}, "dense / per-cell kernels: B_dense is what moves"
    elif args.tuning:
        traffic, traffic_source = {}, "experiment (--tuning): the committed capture describes the default launch plan, not used"
    else:
        traffic, traffic_source = ncu_traffic(args.config)
    kern = {}
    for name in ("fused", "velocity", "stress_sensor"):
        n = kt[name]["launches"]
        avg_ms = kt[name]["ms"] / n if n else 0.0
        tr = traffic.get(name)
        if tr is not None and name != "velocity":
            # the capture had both sensor maps on: take the sum-of-squares map (8 B per cell) off for the timed
            # steps outside the rms window, so that bytes and times describe the same launches
            tr -= 8.0 * (cells_f if name == "fused" else cells_2) * (1.0 - rms_frac)
        moved = min(alg[name], tr) if tr else alg[name]
        kern[name] = {"avg_ms": avg_ms, "launches": n, "algorithmic_bytes": alg[name] if n else 0.0, "traffic": tr if n else None,
                      "achieved_gbs": moved / (avg_ms * 1e-3) / 1e9 if n and avg_ms > 0 else None,
                      "dram_gbs": tr / (avg_ms * 1e-3) / 1e9 if n and tr and avg_ms > 0 else None}
    kern["inject"] = {"avg_ms": kt["inject"]["ms"] / max(1, kt["inject"]["launches"]), "launches": kt["inject"]["launches"]}
    dom = max(("fused", "velocity", "stress_sensor"), key=lambda k: kt[k]["ms"])
    step_alg = sum(kern[k]["algorithmic_bytes"] for k in ("fused", "velocity", "stress_sensor"))
    have_all = all(kern[k]["traffic"] is not None for k in ("fused", "velocity", "stress_sensor") if kern[k]["launches"])
    step_traffic = sum(kern[k]["traffic"] for k in ("fused", "velocity", "stress_sensor") if kern[k]["launches"]) if (traffic and have_all) else None
    step_s = ms / K * 1e-3
    b_dense_step = (166.0 + 8.0 * rms_frac + 48.0 * bits) * w.cells      # what a plain dense two-pass sweep would move
    min_step_bytes = w.min_bytes_per_cell_step(rms_frac=rms_frac) * w.cells
    step_moved = min(step_alg, step_traffic) if step_traffic else step_alg
    if not traffic and not (args.dense or args.reference_kernels) and coverage == 0.0:
        # two passes with tile-class skipping and no capture: the class-aware minimum stands in for the traffic
        scale = min(1.0, min_step_bytes / step_alg)
        for k in ("velocity", "stress_sensor"):
            if kern[k]["achieved_gbs"]:
                kern[k]["achieved_gbs"] *= scale
        step_moved = step_alg * scale
    rule = ("min(algorithmic bytes, ncu-measured DRAM bytes of this kernel on this workload and build) / CUDA-event time"
            if traffic else "algorithmic bytes (class-aware minimum where tile classes are skipped: no ncu capture) / CUDA-event time")
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["achieved_gbs"], "peak": peak_gbs, "unit": "GB/s",
                "frac": kern[dom]["achieved_gbs"] / peak_gbs if kern[dom]["achieved_gbs"] else None,
                "traffic": kern[dom]["traffic"], "traffic_source": traffic_source, "rule": rule,
                "dram_frac": kern[dom]["dram_gbs"] / peak_gbs if kern[dom]["dram_gbs"] else None,
                "algorithmic_bytes_per_launch": kern[dom]["algorithmic_bytes"],
                "peak_source": peak_src + ", burst copy figure",
                "kernel_times": "CUDA events of the library on the context's stream, second pass of the same W + K steps "
                                "launched kernel by kernel (the timed pass replays CUDA graphs)",
                "step": {"ms_graph_replay": ms / K, "ms_kernel_by_kernel": ms_timed_pass,
                         "algorithmic_bytes": step_alg, "traffic": step_traffic,
                         "achieved_gbs": step_moved / step_s / 1e9,
                         "frac_of_measured": step_moved / step_s / 1e9 / peak_gbs,
                         "frac_of_8TBs": step_moved / step_s / 1e9 / 8000.0,
                         "measured_dram_gbs": step_traffic / step_s / 1e9 if step_traffic else None,
                         "b_dense_bytes": b_dense_step,
                         "b_dense_equivalent_gbs": b_dense_step / step_s / 1e9,
                         "note": "frac_of_8TBs counts bytes really moved (north_star's bar by SURVEY 8(d)'s no-inflation rule); "
                                 "b_dense_equivalent is the rate a dense two-pass sweep would need for the same throughput"},
                "class_aware_min_bytes_per_step_two_pass": min_step_bytes,
                "kernels": kern}

    cpu = cpu_baseline_leg(wl.make(args.config)) if (world == 1 and not args.no_cpu_baseline) else None
    nxt = next_rows(dev) if (world == 1 and args.config == 2 and not args.no_next and not args.no_cpu_baseline) else None

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "pml": w.pml, "cells": w.cells,
                   "materials": int(w.table.shape[0]), "source_cells": int(w.src_cell.size),
                   "parallelism": f"replicas x{world} (no sharding)",
                   "l2": "state 2.4 GB per step >> 126 MB L2: inputs larger than L2, no flush",
                   "kernels": kernels_desc, "cuda_graph": bool(mode_bits & bv.MODE_GRAPH),
                   "fused_tile_plane_fraction": coverage,
                   "result_finite_nonzero": finite},
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d / total,
                "d2h_bytes_per_step": d2h / total, "steps": total, "seconds": e2e_ms * 1e-3,
                "seconds_first_pass": e2e_cold_s,
                "what": "bvfdtd_create + set_source + step(W+K) + read_peak_pressure to pinned host, wall clock; "
                        "second of two identical passes (the first also pays the workspace cudaMalloc)"},
        "gpu_launches": int(round(sum(kt[k]["launches"] for k in kt) * K / max(1, min(K, 4096)))),
        "ms_per_step_kernel_by_kernel": ms_timed_pass,
        "roofline": roofline,
    }
    if cpu is not None:
        line["cpu_baseline"] = cpu
    if nxt is not None:
        line["next_rows"] = nxt            # SURVEY.md 8(f) kernels beyond the hot path (also: bench.py --next)
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
    ap.add_argument("--next", action="store_true", help="time only the kernels beyond the hot path (SURVEY.md 8(f)), one JSON line")
    ap.add_argument("--no-next", action="store_true", help="leave next_rows out of the default line")
    ap.add_argument("--tuning", type=int, default=0, help="bvfdtd_opts.tuning bits (BVFDTD_TUNE_*), experiments")
    ap.add_argument("--traffic-from", default=None,
                    help="ncu `--page raw --csv` export of a --set full capture of this build: write profiles/traffic.csv")
    ap.add_argument("--dense", action="store_true",
                    help="BVFDTD_FLAG_DENSE: sweep every array everywhere (no tile-class skipping)")
    args = ap.parse_args()
    if args.traffic_from:
        return traffic_from_ncu(args.traffic_from, args.config)
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return reference_arm(args)
    if args.next:
        import torch
        from paper_2301_12727_b200 import build as bv_build
        bv_build.build()
        print(json.dumps({"next_rows": next_rows(torch.device("cuda", 0))}), flush=True)
        return 0
    return ours(args)


if __name__ == "__main__":
    sys.exit(main())
