"""Full-length parity of configs 3 and 4 on sampled planes, in three steps that need not run on one machine.

The oracle needs about an hour per configuration for the 5000 / 6000 steps (fp64, 171-173 M cells, 16 cores) and a
GPU call of this build environment is limited to one hour: `test_gpu_full_runs.py::test_config34_full_length`
checkpoints and resumes the oracle across calls; this script is the other way round it -- the oracle leg can run
anywhere, without a GPU.  The tier's rule for full sizes is "on sampled outputs the oracle can compute": the comparison runs on
whole planes of every field.

    python tests/full_length_sampled.py oracle  CFG OUT.npz     # CPU only: calls nothing but oracle/ and the inputs
    python tests/full_length_sampled.py gpu     CFG OUT.npz     # B200: default path through the C ABI; also checks
                                                                # the run bit for bit against the two-pass path
    python tests/full_length_sampled.py compare CFG ORACLE.npz GPU.npz [REPORT.json]

Sampled: two x-y planes (one third and two thirds of the depth), the x-z plane through the axis and the y-z plane
through the axis, of all 15 state arrays, the pressure, the running peak and (where the config has an rms window)
the rms amplitude.  Bars as in north_star: relative L2 <= 1e-4 per field over the sampled cells (fields whose oracle
norm is below 1e-6 of their group's largest are compared against that largest), peak / rms max relative error
<= 1e-3 over the sampled cells above 10 % of the sampled maximum; plus max abs error <= 1e-3 of the group's largest
value.  No expected value comes from the CUDA path: ORACLE.npz is written by the `oracle` step alone.
"""
from __future__ import annotations

import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FIELDS = ("vx", "vy", "vz", "sxx", "syy", "szz", "sxy", "sxz", "syz", "rxx", "ryy", "rzz", "rxy", "rxz", "ryz")
GROUPS = (("vx", "vy", "vz"), ("sxx", "syy", "szz", "sxy", "sxz", "syz"), ("rxx", "ryy", "rzz", "rxy", "rxz", "ryz"))


def planes(w):
    return {"xy1": (w.nz // 3, None, None), "xy2": (2 * w.nz // 3, None, None), "xz": (None, w.ny // 2, None),
            "yz": (None, None, w.nx // 2)}


def sample(a, w):
    out = {}
    for tag, (k, j, i) in planes(w).items():
        out[tag] = np.ascontiguousarray(a[k] if k is not None else a[:, j] if j is not None else a[:, :, i])
    return out


def run_oracle(cfg, out):
    from oracle import fdtd_oracle as orc
    from paper_2301_12727_b200 import workloads as wl
    w = wl.make(cfg)
    o = orc.Oracle.from_workload(w)
    t0 = time.perf_counter()
    done = 0
    while done < w.steps:
        n = min(100, w.steps - done)
        o.step(n)
        done += n
        el = time.perf_counter() - t0
        print(f"oracle cfg {cfg}: step {done}/{w.steps}, {el:.0f} s, {w.cells * done / el / 1e6:.1f} Mcell/s", flush=True)
    res = {"steps": np.int64(w.steps), "seconds": np.float64(time.perf_counter() - t0), "rms_count": np.int64(o.rms_count)}
    names = FIELDS + ("p", "peak") + (("rms_amp",) if 0 <= w.rms_begin < w.steps else ())
    for n in names:
        for tag, v in sample(o.get(n), w).items():
            res[f"{n}:{tag}"] = v
    np.savez_compressed(out, **res)
    print("wrote", out)


def run_gpu(cfg, out):
    from paper_2301_12727_b200 import binding as bv
    from paper_2301_12727_b200 import build as bv_build
    from paper_2301_12727_b200 import workloads as wl
    bv_build.build()
    w = wl.make(cfg)
    res = {}
    keep = {}
    for tuning in (0, bv.TUNE_NO_FUSED | bv.TUNE_NO_GRAPH):
        sim = bv.Simulation.from_workload(w, tuning=tuning)
        mode = sim.kernel_mode()
        sim.step(w.steps)
        peak, rms = sim.read_peak_pressure()
        if tuning == 0:
            res.update(steps=np.int64(w.steps), rms_count=np.int64(sim.rms_count), fused_fraction=np.float64(sim.fused_coverage()))
            res["kernel_mode"] = np.array(mode)
            for n in FIELDS + ("p",):
                a = sim.read_fields(n)
                keep[n] = a if n in ("p", "vz", "rxx", "sxy") else None
                for tag, v in sample(a, w).items():
                    res[f"{n}:{tag}"] = v
            for tag, v in sample(peak, w).items():
                res[f"peak:{tag}"] = v
            if 0 <= w.rms_begin < w.steps:
                for tag, v in sample(rms, w).items():
                    res[f"rms_amp:{tag}"] = v
            keep["peak"] = peak
            assert sim.padding_nonzeros() == 0
        else:
            same = all(np.array_equal(keep[n], sim.read_fields(n)) for n in ("p", "vz", "rxx", "sxy")) and np.array_equal(keep["peak"], peak)
            res["bit_identical_to_two_pass_path"] = np.bool_(same)
            assert same, "default path differs from the two-pass path"
        print(f"gpu cfg {cfg}: {mode}: {w.steps} steps done", flush=True)
        sim.close()
    np.savez_compressed(out, **res)
    print("wrote", out, os.path.getsize(out) / 1e6, "MB")


def compare(cfg, f_oracle, f_gpu, report=None):
    o, g = np.load(f_oracle), np.load(f_gpu)
    assert int(o["steps"]) == int(g["steps"]) and int(o["rms_count"]) == int(g["rms_count"])
    tags = ("xy1", "xy2", "xz", "yz")
    cat = lambda z, n: np.concatenate([z[f"{n}:{t}"].astype(np.float64).ravel() for t in tags])
    rep = {"config": cfg, "steps": int(o["steps"]), "oracle_seconds": float(o["seconds"]), "kernel_mode": str(g["kernel_mode"]),
           "fused_tile_plane_fraction": float(g["fused_fraction"]), "bit_identical_to_two_pass_path": bool(g["bit_identical_to_two_pass_path"]),
           "sampled_cells": int(cat(o, "p").size), "fields": {}}
    ok = True
    for group in GROUPS:
        ref = {n: cat(o, n) for n in group}
        gn = max(np.linalg.norm(v) for v in ref.values())
        ga = max(np.abs(v).max() for v in ref.values())
        for n in group:
            d = cat(g, n) - ref[n]
            nrm = np.linalg.norm(ref[n])
            denom = nrm if nrm > 1e-6 * gn else gn
            l2 = float(np.linalg.norm(d) / denom) if denom > 0 else float(np.linalg.norm(d))
            mx = float(np.abs(d).max() / ga) if ga > 0 else float(np.abs(d).max())
            rep["fields"][n] = {"rel_l2": l2, "max_abs_over_group_max": mx}
            ok &= l2 <= 1e-4 and mx <= 1e-3
    for n in ("peak", "rms_amp"):
        if f"{n}:xy1" not in o.files:
            continue
        r, v = cat(o, n), cat(g, n)
        m = r > 0.1 * r.max()
        e = float(np.abs(v[m] / r[m] - 1.0).max())
        rep[n + "_max_rel"] = e
        ok &= e <= 1e-3
    rep["worst_rel_l2"] = max(v["rel_l2"] for v in rep["fields"].values())
    rep["pass"] = bool(ok)
    print(json.dumps(rep, indent=1))
    if report:
        with open(report, "w") as f:
            json.dump(rep, f, indent=1)
    return 0 if ok else 1


if __name__ == "__main__":
    mode, cfg = sys.argv[1], int(sys.argv[2])
    if mode == "oracle":
        run_oracle(cfg, sys.argv[3])
    elif mode == "gpu":
        run_gpu(cfg, sys.argv[3])
    else:
        sys.exit(compare(cfg, sys.argv[3], sys.argv[4], sys.argv[5] if len(sys.argv) > 5 else None))
