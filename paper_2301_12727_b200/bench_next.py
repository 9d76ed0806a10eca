"""Timing of the kernels beyond the hot path: one JSON line per kernel.

    python -m paper_2301_12727_b200.bench_next

NEXT-1 Rayleigh-Sommerfeld: config 2's focused bowl (aperture 64 mm, F# 1) decomposed at lambda/4
(elements of lambda^2/16) evaluated on the whole 300 x 300 entry plane.  The kernel is
SFU-bound: 3 MUFU operations (rsqrt, sin, cos) per (source, receiver) pair; peak = SMs x 16 MUFU
lanes per SM x SM clock / 3 (16 lanes per SM = 4 per scheduler is the figure assumed for sm_100).
NEXT-2 plane intensity: one read of the sum-of-squares map and the index map of config 2 (HBM-bound).
NEXT-4 thermal step on config 2's grid: HBM-bound, algorithmic bytes per cell-step = rise read + write,
Q read, dose read + write, material byte (21 B) + running maximum read + write (29 B); peak = the
measured copy bandwidth of MEASURED_PEAKS.json.
"""
from __future__ import annotations

import json
import math

import numpy as np


def main():
    import torch
    from . import binding as bv
    from . import build as bv_build
    from . import workloads as wl
    bv_build.build()
    dev = torch.device("cuda", 0)
    f, c0, rho0 = 500e3, 1500.0, 1000.0
    lam = c0 / f
    pos, area = wl.bowl_elements(64e-3, 64e-3, lam / 4)
    dx = 1e-3 / 3.0
    xs = (np.arange(300) - 149.5) * dx
    X, Y = np.meshgrid(xs, xs)
    rcv = np.stack([X.ravel(), Y.ravel(), np.full(X.size, 15e-3)], axis=1)
    s = torch.from_numpy(pos.astype(np.float32)).to(dev)
    w = torch.from_numpy(np.stack([0.01 * area, np.zeros_like(area)], axis=1).astype(np.float32)).to(dev)
    r = torch.from_numpy(rcv.astype(np.float32)).to(dev)
    out = torch.empty((4, r.shape[0]), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream

    def launch():
        bv._check(bv.lib().bvfdtd_rayleigh(s.shape[0], s.data_ptr(), w.data_ptr(), r.shape[0], r.data_ptr(), f, c0, rho0,
                                           out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), out[3].data_ptr(),
                                           stream), "bvfdtd_rayleigh")
    for _ in range(3):
        launch()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 20
    e0.record()
    for _ in range(reps):
        launch()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    pairs = float(s.shape[0]) * float(r.shape[0])
    props = torch.cuda.get_device_properties(dev)
    clk = 1.965e9
    peak = props.multi_processor_count * 16 * clk / 3.0
    print(json.dumps({"kernel": "k_rayleigh", "workload": f"{s.shape[0]} bowl elements x {r.shape[0]} receivers",
                      "ms": ms, "value": pairs / (ms * 1e-3) / 1e9, "unit": "Gpair/s",
                      "roofline": {"bound": "alu", "achieved": pairs / (ms * 1e-3) / 1e9, "peak": peak / 1e9,
                                   "unit": "Gpair/s", "frac": pairs / (ms * 1e-3) / peak,
                                   "peak_source": "SMs x 16 MUFU lanes x 1.965 GHz / 3 MUFU per pair (assumed lane count)"}}))

    wk = wl.make(2, steps=40)
    wk.rms_begin = 10
    sim = bv.Simulation.from_workload(wk, device=dev)
    sim.step(40)
    sim.plane_intensity()
    torch.cuda.synchronize()
    import time
    t0 = time.perf_counter()
    for _ in range(5):
        sim.plane_intensity()
    dt = (time.perf_counter() - t0) / 5
    bytes_ = wk.cells * 5.0
    print(json.dumps({"kernel": "k_plane_intensity", "workload": wk.name, "ms": dt * 1e3,
                      "value": bytes_ / dt / 1e9, "unit": "GB/s (sumsq + index map, wall clock incl. the 7 KB read-back)"}))
    sim.close()
    del sim
    torch.cuda.empty_cache()

    import os
    peaks = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    hbm = json.load(open(peaks))["hbm_gbs"] if os.path.exists(peaks) else 6400.0
    tw = wl.thermal_config2()
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
        cells = tw["nx"] * tw["ny"] * tw["nz"]
        b = 29.0 if track_max else 21.0
        gbs = cells * b / (ms * 1e-3) / 1e9
        print(json.dumps({"kernel": "k_bhte<%s>" % ("true" if track_max else "false"),
                          "workload": "thermal step on config 2's grid (300x300x450, 128 materials), %d launches" % reps,
                          "ms": ms, "value": cells / (ms * 1e-3) / 1e9, "unit": "Gcell-updates/s",
                          "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
                                       "bytes_per_cell_step": b}}))
        th.close()
        del th
        torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
