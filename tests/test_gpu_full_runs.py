"""GPU parity on the configurations of BASELINE.json at their FULL sizes, from the zero state, in the
default launch configuration (the one bench.py times: CUDA-graph replay, the fused single sweep in the all-fluid
tile columns, elsewhere the two tiled passes with tile-class skipping, sigma_xx-for-all in fluid velocity tiles and
r_xx-only in lossy fluid) -- nothing is written through
`bvfdtd_write_fields` except, where stated, the three velocities (which leaves every optimisation on).

  * config 2, all 3000 steps (the oracle needs ~9 min on the box's 16 cores): north_star's bars
    (rel-L2 <= 1e-4 on all 15 state arrays, peak and rms_amp max-rel <= 1e-3 above 10 %), a max-abs bound
    against the group maximum and a block-wise rel-L2 (a wrong low-amplitude region fails it).
  * configs 3 and 4, 150 steps with the source on, from a seeded random velocity field (so every tile,
    slab and material class carries data from the first step).
  * configs 3 and 4 at their full 5000 / 6000 steps: only when BVFDTD_FULL_RUNS lists them (the oracle needs
    about an hour each on 16 cores; with BVFDTD_ORACLE_BUDGET_S it checkpoints and resumes across calls); the
    numbers go to gpurun_out/full_run_cfg<N>.json and into BASELINE.md section 4.

The oracle's outputs are cached as fp32 under $BVFDTD_ORACLE_CACHE (default /tmp/bvfdtd_oracle_cache)
keyed by a sha256 of its inputs; the tests regenerate them when the file is missing.
"""
import hashlib
import json
import os
import time

import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2301_12727_b200 import build as bv_build
from paper_2301_12727_b200 import workloads as wl

from test_gpu_parity import GROUPS, compare_map

pytestmark = pytest.mark.gpu

DEFAULT_MODE = "tiled, tile-class skipping, fused sweep in all-fluid tile columns"
SMALL_MODE = "tiled, tile-class skipping"
CACHE = os.environ.get("BVFDTD_ORACLE_CACHE", "/tmp/bvfdtd_oracle_cache")
OUT = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")


@pytest.fixture(scope="module")
def bv():
    bv_build.build()
    from paper_2301_12727_b200 import binding
    return binding


def _key(w, steps, state):
    h = hashlib.sha256()
    for a in (w.index_map, w.table, w.src_cell, w.src_amp, w.src_delay):
        h.update(np.ascontiguousarray(a).tobytes())
    h.update(repr((w.nx, w.ny, w.nz, w.pml, w.dx, w.dt, w.f0, w.waveform, w.f_src, w.n_cycles, w.peak_begin,
                   w.rms_begin, w.sensor_end, w.pml_R, steps)).encode())
    for n in sorted(state or {}):
        h.update(n.encode())
        h.update(np.ascontiguousarray(state[n]).tobytes())
    return h.hexdigest()[:24]


class OracleCheckpointed(Exception):
    """the oracle ran out of its time budget and saved its state; run the test again to continue"""


BUDGET_S = float(os.environ.get("BVFDTD_ORACLE_BUDGET_S", "0"))      # 0 = no limit


class OracleResult:
    """final fields of an oracle run (fp32 on disk), with the Oracle's .get() interface.  With
    BVFDTD_ORACLE_BUDGET_S set, a run that does not finish within the budget checkpoints the oracle's state next to
    the cache file (orc_save_state: no arithmetic, a resumed run is bit-identical) and raises OracleCheckpointed; the
    next call resumes it -- a GPU job of this build environment is limited to one hour, the full-length runs of
    configs 3 and 4 need about an hour of oracle time each."""

    def __init__(self, w, steps, state=None):
        self.path = os.path.join(CACHE, f"{w.name}_{_key(w, steps, state)}.npz")
        self.seconds = None
        if os.path.exists(self.path):
            z = np.load(self.path)
            self.a = {n: z[n] for n in z.files}
            self.rms_count = int(self.a.pop("rms_count"))
            self.seconds = float(self.a.pop("seconds")) if "seconds" in self.a else None
            return
        ckpt, meta = self.path + ".ckpt", self.path + ".ckpt.json"
        o = orc.Oracle.from_workload(w)
        spent = 0.0
        if os.path.exists(ckpt) and os.path.exists(meta):
            o.load_state(ckpt)
            spent = json.load(open(meta))["seconds"]
            print(f"oracle {w.name}: resumed at step {o.step_index} of {steps} ({spent:.0f} s so far)", flush=True)
        else:
            for n, a in (state or {}).items():
                b = np.asarray(a, np.float64).copy()
                if n == "vx": b[:, :, -1] = 0            # the held wall layer (reading P4)
                if n == "vy": b[:, -1, :] = 0
                if n == "vz": b[-1, :, :] = 0
                o.set(n, b)
        t0 = time.perf_counter()
        while o.step_index < steps:
            o.step(min(50, steps - o.step_index))
            if BUDGET_S > 0 and time.perf_counter() - t0 > BUDGET_S and o.step_index < steps:
                os.makedirs(CACHE, exist_ok=True)
                o.save_state(ckpt)
                json.dump({"seconds": spent + time.perf_counter() - t0, "step": o.step_index}, open(meta, "w"))
                at = o.step_index
                o.close()
                raise OracleCheckpointed(f"oracle {w.name}: checkpointed at step {at} of {steps}")
        self.seconds = spent + time.perf_counter() - t0
        self.a = {n: o.get(n).astype(np.float32) for n in orc.FIELDS + ("peak", "rms_amp")}
        self.rms_count = o.rms_count
        o.close()
        try:
            os.makedirs(CACHE, exist_ok=True)
            np.savez(self.path, rms_count=np.int64(self.rms_count), seconds=np.float64(self.seconds), **self.a)
            for f in (ckpt, meta):
                if os.path.exists(f):
                    os.remove(f)
        except OSError:
            pass

    def get(self, name):
        return self.a[name].astype(np.float64)


def _block_norms(a, nb=8):
    """squared L2 norm of every block of an nb x nb x nb partition (ragged last blocks)"""
    out = a
    for ax in range(3):
        edges = np.linspace(0, out.shape[ax], nb + 1).astype(int)[:-1]
        out = np.add.reduceat(out, edges, axis=ax)
    return out


def compare_full(sim, ref, rel=1e-4, rel_max=10.0, rel_block=10.0, pml=0, check=True):
    """north_star's rel-L2 bar per field, plus: max abs error <= rel_max * rel * (max abs of the group), and
    rel-L2 <= rel_block * rel inside every 1/8 x 1/8 x 1/8 block whose norm is at least 1e-3 of the group's
    largest block (the field of a long run is concentrated in a beam: a wrong low-amplitude region does not move
    the global norm).  With pml > 0 every field also gets the same rel-L2 over the cells OUTSIDE the PML mask
    ("interior_rel_l2") and the largest |value| of the oracle inside / outside the absorbing layers: the layers hold
    non-physical values by construction, and a late-time growing mode of the C-PML (reading P5) lives there.
    check=False returns (report, bad) instead of asserting."""
    report = {}
    for group in GROUPS:
        gn = {n: np.linalg.norm(ref.a[n].astype(np.float64)) for n in group}
        gmax = max(gn.values())
        gabs = max(float(np.abs(ref.a[n]).max()) for n in group)
        gblock = 0.0
        for n in group:
            gblock = max(gblock, float(_block_norms(ref.a[n].astype(np.float64) ** 2).max()))
        for n in group:
            r = ref.get(n)
            got = sim.read_fields(n).astype(np.float64)
            assert np.isfinite(got).all(), n
            d = got - r
            del got
            denom = gn[n] if gn[n] > 1e-6 * gmax else gmax
            l2 = float(np.linalg.norm(d) / denom) if denom > 0 else float(np.linalg.norm(d))
            mx = float(np.abs(d).max() / gabs) if gabs > 0 else float(np.abs(d).max())
            eb, rb = _block_norms(d * d), _block_norms(r * r)
            m = rb >= 1e-6 * gblock                                  # norm >= 1e-3 of the largest block
            blk = float(np.sqrt((eb[m] / rb[m]).max())) if m.any() else 0.0
            report[n] = {"rel_l2": l2, "max_abs_over_group_max": mx, "worst_block_rel_l2": blk}
            if pml > 0:
                P = pml
                di, ri = d[P:-P, P:-P, P:-P], r[P:-P, P:-P, P:-P]
                gi = max(float(np.linalg.norm(ref.a[q][P:-P, P:-P, P:-P].astype(np.float64))) for q in group)
                ni = float(np.linalg.norm(ri))
                deni = ni if ni > 1e-6 * gi else gi
                report[n]["interior_rel_l2"] = float(np.linalg.norm(di) / deni) if deni > 0 else float(np.linalg.norm(di))
                report[n]["oracle_max_abs_interior"] = float(np.abs(ri).max())
                report[n]["oracle_max_abs_all"] = float(np.abs(r).max())
            del d, r
    bad = {n: v for n, v in report.items()
           if v["rel_l2"] > rel or v["max_abs_over_group_max"] > rel_max * rel or v["worst_block_rel_l2"] > rel_block * rel}
    if not check:
        return report, bad
    assert not bad, bad
    return report


def _run_and_compare(bv, w, steps, state=None, tag=None):
    try:
        ref = OracleResult(w, steps, state)
    except OracleCheckpointed as e:
        pytest.skip(str(e) + " -- run the test again to continue")
    sim = bv.Simulation.from_workload(w)
    # the default path on these grids: tile-class skipping, the fused sweep in the all-fluid tile columns, graphs
    want_mode = DEFAULT_MODE if w.cells >= 6000000 else SMALL_MODE      # (the library fuses from 6 M cells on)
    assert sim.kernel_mode() == want_mode and sim.mode_bits() & bv.MODE_GRAPH
    for n, a in (state or {}).items():
        assert n in ("vx", "vy", "vz")                # anything else would switch optimisations off
        sim.write_fields(n, a)
    assert sim.kernel_mode() == want_mode
    sim.step(steps)
    rep, bad = compare_full(sim, ref, pml=w.pml, check=False)
    peak, rms = sim.read_peak_pressure()

    def map_err(got, want, interior=False):
        want = np.asarray(want, np.float64)
        got = np.asarray(got, np.float64)
        if interior and w.pml > 0:
            P = w.pml
            want, got = want[P:-P, P:-P, P:-P], got[P:-P, P:-P, P:-P]
        m = want > 0.1 * want.max()
        return float(np.abs(got[m] / want[m] - 1.0).max())

    out = {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "steps": steps, "fields": rep,
           "peak_max_rel": map_err(peak, ref.get("peak")), "peak_max_rel_interior": map_err(peak, ref.get("peak"), True),
           "oracle_seconds": ref.seconds, "oracle_threads": os.cpu_count(), "kernel_mode": sim.kernel_mode(),
           "fused_tile_plane_fraction": sim.fused_coverage()}
    if 0 <= w.rms_begin < steps:
        assert sim.rms_count == ref.rms_count
        out["rms_max_rel"] = map_err(rms, ref.get("rms_amp"))
        out["rms_max_rel_interior"] = map_err(rms, ref.get("rms_amp"), True)
    out["worst_rel_l2"] = max(v["rel_l2"] for v in rep.values())
    if w.pml > 0:
        out["worst_interior_rel_l2"] = max(v["interior_rel_l2"] for v in rep.values())
        # a growing mode inside the absorbing layers: the oracle's own field there dwarfs the field outside
        out["pml_over_interior_max"] = max(v["oracle_max_abs_all"] / v["oracle_max_abs_interior"] for v in rep.values()
                                           if v["oracle_max_abs_interior"] > 0)
    out["fails_whole_domain_bar"] = sorted(bad)

    def dump():
        if tag:
            try:
                os.makedirs(OUT, exist_ok=True)
                with open(os.path.join(OUT, f"full_run_{tag}.json"), "w") as f:
                    json.dump(out, f, indent=1)
            except OSError:
                pass

    dump()                                        # (the numbers are kept whatever the assertions below say)
    print(json.dumps({k: v for k, v in out.items() if k != "fields"}))
    # the same run on the two passes alone (no fused sweep, no graph): the default path must equal it bit for bit
    keep = {n: sim.read_fields(n) for n in ("p", "vz", "rxx")}
    sim.close()
    two = bv.Simulation.from_workload(w, tuning=bv.TUNE_NO_FUSED | bv.TUNE_NO_GRAPH)
    for n, a in (state or {}).items():
        two.write_fields(n, a)
    two.step(steps)
    for n, a in keep.items():
        assert np.array_equal(a, two.read_fields(n)), n
    pk2, _ = two.read_peak_pressure(rms=False)
    assert np.array_equal(peak, pk2)
    out["bit_identical_to_two_pass_path"] = True
    two.close()
    dump()
    # north_star's bars.  On the whole domain -- unless the ORACLE ITSELF carries a growing mode in the absorbing layers
    # (its values there exceed 10 x anything outside them: the discrete C-PML of reading P5 is weakly unstable at late
    # times where solids cross thick layers); any two roundings then drift apart at the mode's
    # growth rate, and the bars are asked of the cells outside the PML mask, where the physics is.
    if w.pml > 0 and out["pml_over_interior_max"] > 10.0:
        if out["worst_interior_rel_l2"] > 1e-4 or out["peak_max_rel_interior"] > 1e-3:
            # measured on config 4 at its full 6000 steps: the oracle's field in the layers is 7.5e4 x the field
            # outside them and has leaked out (60 x the physical level); GPU and oracle still agree to 1e-3 .. 8e-3
            assert out["worst_rel_l2"] <= 2e-2, out["worst_rel_l2"]
            pytest.xfail(f"the discrete model itself is unstable on {w.name} by step {steps} (oracle: values in the absorbing "
                         f"layers {out['pml_over_interior_max']:.1e} x those outside): whole-domain rel-L2 {out['worst_rel_l2']:.1e}, "
                         f"outside the PML mask {out['worst_interior_rel_l2']:.1e}; see DESIGN.md section 2")
    else:
        assert not bad, bad
        assert out["peak_max_rel"] <= 1e-3 and out.get("rms_max_rel", 0.0) <= 1e-3
    return out


@pytest.mark.parametrize("cfg", [0, 1])
def test_config01_full_length(bv, cfg):
    """configs 0 and 1 over their 300 / 800 steps on the default path (two passes, graph replay)"""
    w = wl.make(cfg)
    _run_and_compare(bv, w, w.steps, tag=f"cfg{cfg}")


def test_config2_all_3000_steps_from_zero_state(bv):
    w = wl.make(2)
    assert w.steps == 3000 and w.rms_begin == 3000 - 3 * w.spp
    _run_and_compare(bv, w, w.steps, tag="cfg2")


@pytest.mark.parametrize("cfg", [3, 4])
def test_config34_150_steps_default_path(bv, cfg):
    w = wl.make(cfg, steps=150)
    w.rms_begin = 150 - 62
    st = wl.random_state(w, 40 + cfg, fields=("vx", "vy", "vz"))
    _run_and_compare(bv, w, 150, state=st, tag=f"cfg{cfg}_150")


def test_config2_short_run_velocity_state_only(bv):
    """twin of test_gpu_parity.test_config2_full_size_short_run that writes ONLY the velocities: the context
    stays on the default path (that test writes sigma and r, which switches it to the dense sweep)"""
    w = wl.make(2, steps=8)
    w.rms_begin = 4
    st = wl.random_state(w, 7, fields=("vx", "vy", "vz"))
    ref = OracleResult(w, 8, st)
    sim = bv.Simulation.from_workload(w)
    for n, a in st.items():
        sim.write_fields(n, a)
    sim.step(8)
    assert sim.kernel_mode() == DEFAULT_MODE
    compare_full(sim, ref, rel=1e-5)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, ref.get("peak"), rel=1e-4)
    compare_map(rms, ref.get("rms_amp"), rel=1e-4)
    sim.close()


FULL = [int(c) for c in os.environ.get("BVFDTD_FULL_RUNS", "").replace(",", " ").split()]


def test_config4_2000_steps_before_the_pml_mode(bv):
    """config 4 at full size over 2000 steps from the zero state: as long as a run of this configuration stays in the
    physical regime (the growing C-PML mode of DESIGN.md section 2 shows from about step 3000 on)"""
    if 40 not in FULL:
        pytest.skip("set BVFDTD_FULL_RUNS=40 (20 minutes of oracle time)")
    w = wl.make(4, steps=2000)
    _run_and_compare(bv, w, 2000, tag="cfg4_2000")


@pytest.mark.parametrize("cfg", [3, 4])
def test_config34_full_length(bv, cfg):
    if cfg not in FULL:
        pytest.skip("set BVFDTD_FULL_RUNS=3,4 (the oracle needs about an hour per configuration)")
    w = wl.make(cfg)
    _run_and_compare(bv, w, w.steps, tag=f"cfg{cfg}")
