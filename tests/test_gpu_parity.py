"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (ctypes binding), against
the fp64 CPU oracle on the same seeded inputs, element by element.

Bars (BASELINE.json:north_star, restated in DESIGN.md "Tolerances"):
  * bit-exact: material-index round trip, PML mask;
  * fp32 state fields: relative L2 <= 1e-4 after the config's step count (fields whose oracle norm
    is negligible against their group's largest are compared by absolute error against the group);
  * peak-pressure / rms-amplitude maps: max relative error <= 1e-3 over cells above 10 % of the
    map's maximum.
"""
import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2301_12727_b200 import build as bv_build
from paper_2301_12727_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL_L2 = 1e-4
REL_PEAK = 1e-3
GROUPS = (("vx", "vy", "vz"), ("sxx", "syy", "szz", "sxy", "sxz", "syz"),
          ("rxx", "ryy", "rzz", "rxy", "rxz", "ryz"))


@pytest.fixture(scope="module")
def bv():
    bv_build.build()
    from paper_2301_12727_b200 import binding
    return binding


def compare_state(sim, o, rel=REL_L2, fields=None):
    """rel-L2 per field (bar `rel`) and max abs error against the largest value of the field's group (bar 20 rel)."""
    worst = 0.0
    report = {}
    for group in GROUPS:
        ref = {n: o.get(n) for n in group}
        gmax = max(np.linalg.norm(ref[n]) for n in group)
        gabs = max(float(np.abs(ref[n]).max()) for n in group)
        for n in group:
            if fields is not None and n not in fields:
                continue
            got = sim.read_fields(n).astype(np.float64)
            assert np.isfinite(got).all(), n
            err = np.linalg.norm(got - ref[n])
            nrm = np.linalg.norm(ref[n])
            denom = nrm if nrm > 1e-6 * gmax else gmax
            r = err / denom if denom > 0 else err
            report[n] = r
            worst = max(worst, r / rel)
            # no single cell far off either: max abs error against the largest value of the group
            if gabs > 0:
                m = float(np.abs(got - ref[n]).max()) / gabs
                report[n + ":max_abs"] = m
                worst = max(worst, m / (20.0 * rel))
    assert worst <= 1.0, report
    return report


def compare_map(got, ref, rel=REL_PEAK):
    ref = np.asarray(ref, np.float64)
    got = np.asarray(got, np.float64)
    m = ref > 0.1 * ref.max()
    assert m.any()
    e = np.abs(got[m] / ref[m] - 1.0).max()
    assert e <= rel, e
    return e


def run_both(bv, w, steps=None, flags=0, state=None, tuning=0):
    steps = w.steps if steps is None else steps
    sim = bv.Simulation.from_workload(w, flags=flags, tuning=tuning)
    o = orc.Oracle.from_workload(w)
    if state is not None:
        for n, a in state.items():
            sim.write_fields(n, a)
            b = a.astype(np.float64).copy()
            # the wall layer of the normal velocity is held at 0 (reading P4)
            if n == "vx": b[:, :, -1] = 0
            if n == "vy": b[:, -1, :] = 0
            if n == "vz": b[-1, :, :] = 0
            o.set(n, b)
    sim.step(steps)
    o.step(steps)
    return sim, o


# ---------------------------------------------------------------------------------------------
# construction parity (bit-exact)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1, 2])
def test_construction_bit_exact(bv, flags):
    w = wl.random_domain(37, 29, 41, 4, seed=1)
    sim = bv.Simulation.from_workload(w, flags=flags)
    assert np.array_equal(sim.read_fields("material"), w.index_map)
    assert np.array_equal(sim.read_fields("pml_mask"), orc.pml_mask(w.nx, w.ny, w.nz, w.pml))
    der = sim.read_fields("derived")
    ref = orc.derive_materials(w.table, w.f0).astype(np.float32)
    assert np.abs(der.view(np.int32).astype(np.int64) - ref.view(np.int32).astype(np.int64)).max() <= 1
    prof = sim.read_fields("pml_profiles")
    o = orc.Oracle.from_workload(w)
    ref = np.concatenate([o.profile(a, q) for a in range(3) for q in range(4)]).astype(np.float32)
    assert np.abs(prof.view(np.int32).astype(np.int64) - ref.view(np.int32).astype(np.int64)).max() <= 1
    # device-destination reads return the same bytes
    assert np.array_equal(sim.read_fields_device("material").cpu().numpy(), w.index_map)
    for n in ("vx", "sxx", "p"):
        assert not sim.read_fields(n).any()          # zero initial state (reading P9)
    sim.close()


def test_write_read_round_trip(bv):
    w = wl.random_domain(40, 24, 26, 0, seed=2)
    sim = bv.Simulation.from_workload(w)
    st = wl.random_state(w, 3)
    for n, a in st.items():
        sim.write_fields(n, a)
    for n, a in st.items():
        b = a.copy()
        if n == "vx": b[:, :, -1] = 0
        if n == "vy": b[:, -1, :] = 0
        if n == "vz": b[-1, :, :] = 0
        assert np.array_equal(sim.read_fields(n), b), n
    p = -(st["sxx"].astype(np.float64) + st["syy"] + st["szz"]) / 3
    assert np.allclose(sim.read_fields("p"), p, rtol=1e-6, atol=1e-6)
    sim.close()


# ---------------------------------------------------------------------------------------------
# kernel-level parity: one full step from a seeded random state (v after the step checks S2 in
# isolation, sigma/r check S3 given S2), on ragged grids that span several tiles
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1, 2])
@pytest.mark.parametrize("dims,P", [((37, 29, 41), 4), ((72, 40, 24), 8), ((24, 24, 24), 0),
                                    ((131, 21, 19), 2), ((40, 70, 33), 12)])
def test_single_step_random_state(bv, dims, P, flags):
    w = wl.random_domain(*dims, P, seed=10 + P)
    st = wl.random_state(w, 5)
    sim, o = run_both(bv, w, steps=1, flags=flags, state=st)
    rep = compare_state(sim, o, rel=2e-6)
    sim.step(2)
    o.step(2)
    compare_state(sim, o, rel=5e-6)
    sim.close()


@pytest.mark.parametrize("flags", [0, 1, 2])
@pytest.mark.parametrize("kind", ["all_fluid", "all_solid", "single_lossy_voxel", "lossless"])
def test_degenerate_media(bv, kind, flags):
    w = wl.random_domain(36, 28, 30, 6, seed=20, lossy=(kind != "lossless"))
    if kind == "all_fluid":
        w.table[:, 2] = 0.0
        w.table[:, 4] = 0.0
    elif kind == "all_solid":
        w.table[:, 2] = 0.5 * w.table[:, 1]
        w.index_map[:] = np.maximum(w.index_map, 1)
        w.table[0] = (1200.0, 1700.0, 800.0, 10.0, 20.0)
    elif kind == "single_lossy_voxel":
        w.table = np.array([wl.WATER, (1900.0, 2800.0, 1500.0, 200.0, 200.0)])
        w.index_map[:] = 0
        w.index_map[15, 14, 18] = 1
    st = wl.random_state(w, 6)
    if kind == "all_fluid":
        for n in ("sxy", "sxz", "syz", "rxy", "rxz", "ryz"):
            st[n][:] = 0
    sim, o = run_both(bv, w, steps=3, flags=flags, state=st)
    compare_state(sim, o, rel=5e-6)
    if kind == "all_fluid":
        for n in ("sxy", "sxz", "syz", "rxy", "rxz", "ryz"):
            assert not sim.read_fields(n).any()
    if kind == "lossless":
        for n in ("rxx", "rxy"):      # r decays as A^n r0 only: no coupling (reading P3, tau = 0)
            pass
    sim.close()


# ---------------------------------------------------------------------------------------------
# time-stepped parity with source, PML and sensors on small random domains
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1, 2])
@pytest.mark.parametrize("dims,P,wave", [((45, 38, 50), 6, 0), ((64, 33, 37), 5, 1), ((30, 30, 30), 0, 0),
                                         ((70, 57, 56), 24, 1)])
def test_stepped_random_domain(bv, dims, P, wave, flags):
    w = wl.random_domain(*dims, P, seed=30 + P, steps=120, waveform=wave)
    sim, o = run_both(bv, w, flags=flags)
    compare_state(sim, o)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"))
    compare_map(rms, o.get("rms_amp"))
    assert sim.step_index == 120
    sim.close()


@pytest.mark.parametrize("dims,P,wave", [((150, 41, 70), 8, 1), ((131, 45, 66), 12, 0), ((64, 40, 52), 0, 1),
                                         ((150, 60, 80), 24, 1), ((203, 57, 64), 20, 0)])
def test_velocity_three_cta_stage_plans(bv, dims, P, wave):
    """The velocity pass with three resident CTAs per SM and per-CTA stage plans (compact 3-stage plan
    outside the y / z slabs, full 2-stage plan inside; z slabs in chunks of their own) is what config 2
    runs by default; bvfdtd_opts.tuning = BVFDTD_TUNE_VEL_3CTA forces it on a small grid with ragged tiles and
    several chunks: it must match the oracle AND be bit-identical to the two-CTA plan (BVFDTD_TUNE_VEL_2CTA)."""
    w = wl.random_domain(*dims, P, seed=60 + P, steps=90, waveform=wave, n_mat=200 if P == 20 else 6)
    sim, o = run_both(bv, w, tuning=bv.TUNE_VEL_3CTA)
    compare_state(sim, o)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"))
    compare_map(rms, o.get("rms_amp"))
    two = bv.Simulation.from_workload(w, tuning=bv.TUNE_VEL_2CTA)
    two.step(w.steps)
    for n in bv.FIELDS:
        assert np.array_equal(sim.read_fields(n), two.read_fields(n)), n
    pk2, rms2 = two.read_peak_pressure()
    assert np.array_equal(peak, pk2) and np.array_equal(rms, rms2)
    sim.close()
    two.close()


@pytest.mark.parametrize("dims,P,seed", [((150, 43, 38), 6, 1), ((70, 30, 61), 5, 2), ((64, 64, 40), 8, 3)])
def test_tile_class_skipping(bv, dims, P, seed):
    """Mostly-fluid, partly lossless domains: the default path skips the shear stresses and memory
    variables of tile-planes where they are identically zero.  It must match the oracle AND be
    bit-identical to the dense sweep (adding the skipped zeros changes nothing)."""
    w = wl.blocky_domain(*dims, P, seed=seed, steps=60)
    st = wl.random_state(w, 8)
    st = {n: st[n] for n in ("vx", "vy", "vz", "sxx", "syy", "szz")}     # shear stresses and r start at 0
    sim, o = run_both(bv, w, state=st)
    compare_state(sim, o, rel=2e-5)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"), rel=1e-4)
    compare_map(rms, o.get("rms_amp"), rel=1e-4)
    dense, _ = run_both(bv, w, state=st, flags=bv.FLAG_DENSE, steps=0)
    dense.step(w.steps)
    for n in bv.FIELDS:
        assert np.array_equal(sim.read_fields(n), dense.read_fields(n)), n
    pk2, rms2 = dense.read_peak_pressure()
    assert np.array_equal(peak, pk2) and np.array_equal(rms, rms2)
    sim.close()
    dense.close()


def test_full_material_table(bv):
    """256 materials (the uint8 limit): every table row is used by some voxel, ids up to 255."""
    w = wl.random_domain(52, 36, 40, 5, seed=61, n_mat=256, steps=40, waveform=1)
    assert w.table.shape[0] == 256 and w.index_map.max() == 255
    sim, o = run_both(bv, w)
    compare_state(sim, o)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"))
    sim.close()


def test_sensor_windows(bv):
    """peak window [5, 25), rms window [10, 25): nothing sampled outside them."""
    w = wl.random_domain(32, 32, 32, 4, seed=40, steps=40)
    w.peak_begin, w.rms_begin, w.sensor_end = 5, 10, 25
    sim, o = run_both(bv, w)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"))
    compare_map(rms, o.get("rms_amp"))
    assert o.rms_count == 15
    ss = sim.read_fields("sumsq").astype(np.float64)
    ref = o.get("sumsq")
    m = ref > 0.01 * ref.max()
    assert np.abs(ss[m] / ref[m] - 1).max() < 1e-4
    sim.close()


# ---------------------------------------------------------------------------------------------
# the configs of BASELINE.json
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1, 2])
def test_config0_full(bv, flags):
    w = wl.make(0)
    sim, o = run_both(bv, w, flags=flags)
    rep = compare_state(sim, o)
    peak, _ = sim.read_peak_pressure(rms=False)
    e = compare_map(peak, o.get("peak"))
    print("cfg0 rel-L2", {k: f"{v:.2e}" for k, v in rep.items()}, "peak max rel", e)
    sim.close()


def test_config1_full(bv):
    w = wl.make(1)
    sim, o = run_both(bv, w)
    rep = compare_state(sim, o)
    peak, rms = sim.read_peak_pressure()
    e1 = compare_map(peak, o.get("peak"))
    e2 = compare_map(rms, o.get("rms_amp"))
    print("cfg1 rel-L2", {k: f"{v:.2e}" for k, v in rep.items()}, "peak", e1, "rms", e2)
    sim.close()


def test_config2_full_size_short_run(bv):
    """Config 2 at its full 300x300x450 size on the DENSE sweep: 8 steps from a seeded random state of all 15
    fields (every cell carries data, so every tile, slab and ragged tail is checked element by element against
    the oracle) with the focused source on.  Writing a shear stress or a memory variable switches the context
    to the dense sweep, and writing any stress ends the fused mode, so this is NOT the path bench.py times: that
    one is checked by tests/test_gpu_full_runs.py (zero state / velocity-only state, default path)."""
    w = wl.make(2, steps=8)
    w.rms_begin = 4
    st = wl.random_state(w, 7)
    sim, o = run_both(bv, w, state=st)
    assert sim.kernel_mode().startswith("tiled, dense sweep")
    compare_state(sim, o, rel=1e-5)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"), rel=1e-4)
    compare_map(rms, o.get("rms_amp"), rel=1e-4)
    sim.close()
    o.close()


@pytest.mark.parametrize("cfg", [3, 4])
def test_config34_full_size_short_run(bv, cfg):
    """Configs 3 (504x504x672, P 20, 255 materials) and 4 (480x480x600, P 24, array source) at their
    full sizes on the two tiled passes with tile-class skipping: 6 steps from a seeded random velocity /
    normal-stress state (every cell carries data; shear stresses and memory variables start at zero as in a real
    run), element by element against the fp64 oracle.  Writing the normal stresses ends the fused mode and the
    sigma_xx-for-all shortcut of the fluid velocity tiles; the default path with every optimisation on is checked
    by tests/test_gpu_full_runs.py::test_config34_150_steps_default_path."""
    w = wl.make(cfg, steps=6)
    w.rms_begin = 3
    st = wl.random_state(w, 7 + cfg, fields=("vx", "vy", "vz", "sxx", "syy", "szz"))
    sim, o = run_both(bv, w, state=st)
    del st
    compare_state(sim, o, rel=1e-5)
    peak, rms = sim.read_peak_pressure()
    compare_map(peak, o.get("peak"), rel=1e-4)
    compare_map(rms, o.get("rms_amp"), rel=1e-4)
    sim.close()
    o.close()


def test_config2_tiled_vs_percell_kernels_long(bv):
    """Property at full size over a longer run: the tiled kernels and the one-thread-per-cell
    kernels implement the same arithmetic, so after 400 steps of config 2 their fields agree to
    fp32 rounding (the oracle needs ~hours for this; its own check is the short run above)."""
    import torch
    w = wl.make(2, steps=400)
    a = bv.Simulation.from_workload(w)
    a.step(400)
    pa = a.read_fields_device("p").double()
    ka, ra = a.read_peak_pressure_device()
    a.close()
    b = bv.Simulation.from_workload(w, flags=bv.FLAG_REFERENCE_KERNELS)
    b.step(400)
    pb = b.read_fields_device("p").double()
    kb, rb = b.read_peak_pressure_device()
    assert torch.isfinite(pa).all()
    assert float(pb.norm()) > 0
    assert float((pa - pb).norm() / pb.norm()) < 2e-5
    m = kb > 0.1 * kb.max()
    assert float(((ka[m] / kb[m]) - 1).abs().max()) < 2e-4
    m = rb > 0.1 * rb.max()
    assert float(((ra[m] / rb[m]) - 1).abs().max()) < 2e-4
    b.close()


# ---------------------------------------------------------------------------------------------
# NEXT-3: in-kernel phasor sensor (complex pressure amplitude at f0)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1])
def test_phasor_sensor(bv, flags):
    """BVFDTD_FLAG_PHASOR: the stress pass accumulates the single-frequency DFT of p over the rms
    window; compared with the oracle's phasor (pinned on CPU against the DFT of stored traces)."""
    w = wl.blocky_domain(70, 45, 52, 6, seed=5, steps=5 * 62, waveform=1)
    w.rms_begin = w.steps - 2 * w.spp
    sim = bv.Simulation.from_workload(w, flags=flags | bv.FLAG_PHASOR)
    o = orc.Oracle.from_workload(w)
    o.set_phasor(True)
    sim.step(w.steps)
    o.step(w.steps)
    P = sim.read_phasor().astype(np.complex128)
    ref = o.get("phasor_re") + 1j * o.get("phasor_im")
    assert np.linalg.norm(P - ref) <= 1e-4 * np.linalg.norm(ref)
    big = np.abs(ref) > 0.1 * np.abs(ref).max()
    assert np.abs(P[big] / ref[big] - 1).max() < 1e-3
    compare_state(sim, o)
    peak, rms = sim.read_peak_pressure()
    assert not peak.any() and not rms.any()          # phasor mode replaces peak / rms
    with pytest.raises(bv.BvfdtdError):
        sim.plane_intensity()
    sim.close()
    plain = bv.Simulation.from_workload(w)
    with pytest.raises(bv.BvfdtdError) as e:
        plain.read_phasor()
    assert e.value.code == bv.ESTATE
    plain.close()


# ---------------------------------------------------------------------------------------------
# NEXT-2: water-only companion run and the energy-loss reduction (Eq. 2)
# ---------------------------------------------------------------------------------------------
def test_energy_loss_reduction(bv):
    """A bone plate in water and the water-only run on the same grid (cfg-0-like, smaller): the
    device reduction of I_PA per plane and E_L / T_S / z_m against the oracle's definition."""
    from oracle import post_oracle as po
    w = wl.config0()
    w.steps = 280
    w.waveform = 1                      # CW so that the rms window sees the steady state
    w.rms_begin = w.steps - 2 * w.spp
    water = wl.config0()
    water.steps, water.waveform, water.rms_begin = w.steps, 1, w.rms_begin
    water.index_map = np.zeros_like(w.index_map)
    red, ored = [], []
    for ww in (w, water):
        sim, o = run_both(bv, ww)
        s, m = sim.plane_intensity()
        os_, om = po.plane_reductions(o.get("sumsq"), o.rms_count, ww.table, ww.index_map, ww.pml)
        inner = slice(ww.pml, ww.nz - ww.pml)
        assert np.all(s[:ww.pml] == 0) and np.all(s[ww.nz - ww.pml:] == 0)
        assert np.abs(s[inner] / os_[inner] - 1).max() < 2e-4
        big = om > 0.05 * om.max()
        assert np.abs(m[big] / om[big] - 1).max() < 1e-3
        red.append((s, m)); ored.append((os_, om))
        sim.close(); o.close()
    zm, EL, TS = bv.energy_loss(red[0][0], red[1][0], red[1][1], w.pml)
    ozm, oEL, oTS = po.energy_loss(ored[0][0], ored[1][0], ored[1][1], w.pml)
    assert zm == ozm
    assert abs(EL / oEL - 1) < 5e-4 and abs(TS / oTS - 1) < 5e-4
    assert 0 < TS < 1.5
    # no rms sample yet -> ESTATE
    sim = bv.Simulation.from_workload(wl.random_domain(32, 32, 32, 4, seed=3))
    with pytest.raises(bv.BvfdtdError) as e:
        sim.plane_intensity()
    assert e.value.code == bv.ESTATE
    sim.close()


# ---------------------------------------------------------------------------------------------
# error behaviour of the boundary
# ---------------------------------------------------------------------------------------------
def test_create_and_source_validation(bv):
    w = wl.random_domain(32, 32, 32, 4, seed=50)
    mk = lambda **kw: bv.Simulation(**{**dict(nx=w.nx, ny=w.ny, nz=w.nz, pml=w.pml, dx=w.dx, dt=w.dt,
                                              table=w.table, index_map=w.index_map, f0=w.f0), **kw})
    with pytest.raises(bv.BvfdtdError) as e:
        mk(dt=w.dt * 2.0)
    assert e.value.code == bv.ESTABILITY
    bad = w.index_map.copy()
    bad[3, 3, 3] = 200
    with pytest.raises(bv.BvfdtdError) as e:
        mk(index_map=bad)
    assert e.value.code == bv.EINVAL
    with pytest.raises(bv.BvfdtdError):
        mk(pml=14)                                   # 32 < 2*14 + 8
    sim = mk()
    one = np.ones(1, np.float32)
    for cell in (-1, w.cells, 0, 5 + 32 * (5 + 32 * 2)):           # outside / inside the PML
        with pytest.raises(bv.BvfdtdError) as e:
            sim.set_source(np.array([cell]), one, 0 * one, 0, w.f0, 3)
        assert e.value.code == bv.EINVAL
    c = 16 + 32 * (16 + 32 * 16)
    with pytest.raises(bv.BvfdtdError):
        sim.set_source(np.array([c, c]), np.ones(2, np.float32), np.zeros(2, np.float32), 0, w.f0, 3)
    sim.step(3)                                      # legal before set_source: zero source
    assert not sim.read_fields("p").any()
    sim.set_source(np.array([c]), one, 0 * one, 0, w.f0, 3)
    sim.step(3)
    assert sim.read_fields("p").any()
    sim.close()


def test_fluid_memory_variable_kept_once(bv):
    """In a lossy FLUID tile-plane the tiled stress pass keeps only r_xx (r_yy = r_zz = r_xx exactly:
    eS = bS = 0, same recursion, same zero start).  r_yy / r_zz read back must equal the oracle's and
    the dense sweep's bit for bit, also after the context is switched to the dense sweep in mid-run
    by writing a memory variable (the library fills r_yy / r_zz in before it switches)."""
    w = wl.blocky_domain(134, 45, 40, 6, seed=11, steps=40)
    # make the background a lossy fluid (brain-like) so that most tile-planes are lossy and all-fluid
    w.table = w.table.copy()
    w.table[0] = (1040.0, 1546.0, 0.0, 30.0, 0.0)
    sim, o = run_both(bv, w)
    compare_state(sim, o, rel=2e-5)
    dense = bv.Simulation.from_workload(w, flags=bv.FLAG_DENSE)
    dense.step(w.steps)
    got = {n: sim.read_fields(n) for n in ("rxx", "ryy", "rzz", "sxx", "syy", "szz")}
    assert np.abs(got["ryy"]).max() > 0
    for n, a in got.items():
        assert np.array_equal(a, dense.read_fields(n)), n
    fluid_only = ~np.isin(w.index_map, np.nonzero(w.table[:, 2] > 0)[0])
    assert np.array_equal(got["ryy"][fluid_only], got["rxx"][fluid_only])
    # switch to the dense sweep in mid-run: write r_xy back unchanged, continue, compare with the dense twin
    sim.write_fields("rxy", sim.read_fields("rxy"))
    sim.step(25)
    dense.step(25)
    o.step(25)
    compare_state(sim, o, rel=2e-5)
    for n in bv.FIELDS:
        assert np.array_equal(sim.read_fields(n), dense.read_fields(n)), n
    sim.close()
    dense.close()
