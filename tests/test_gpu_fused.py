"""GPU parity of the fused single sweep (kernels_fused.cuh): all-fluid 64 x 8 tile columns do the velocity and
the stress update in one z-march, the other tile columns run the two passes from work lists, all against
ping-ponged copies of v and the normal stresses.  The fused path must (a) match the fp64 oracle within
north_star's bars and (b) be BIT-IDENTICAL to the two-pass path (BVFDTD_TUNE_NO_FUSED): same operations in the
same order on the same operands."""
import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2301_12727_b200 import build as bv_build
from paper_2301_12727_b200 import workloads as wl

from test_gpu_parity import compare_map, compare_state

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bv():
    bv_build.build()
    from paper_2301_12727_b200 import binding
    return binding


def _same(a, b, bv):
    for n in bv.FIELDS + ("p",):
        x, y = a.read_fields(n), b.read_fields(n)
        assert np.array_equal(x, y), (n, int((x != y).sum()), np.argwhere(x != y)[:4].tolist())
    pa, ra = a.read_peak_pressure()
    pb, rb = b.read_peak_pressure()
    assert np.array_equal(pa, pb) and np.array_equal(ra, rb)


CASES = [  # dims, P, seed, waveform, steps, velocity start
    ((150, 60, 70), 8, 1, 1, 60, False),
    ((131, 45, 66), 6, 2, 0, 50, True),      # ragged x and y tails
    ((203, 57, 96), 10, 3, 1, 70, True),     # x slab inside the last (ragged) tile, several z chunks
    ((64, 40, 52), 0, 4, 1, 40, True),       # rigid box, no PML
    ((300, 72, 80), 16, 5, 1, 40, False),    # config 2's x layout (5 tiles, slabs in the outer two)
]


@pytest.mark.parametrize("dims,P,seed,wave,steps,vstart", CASES)
def test_fused_matches_oracle_and_two_pass(bv, dims, P, seed, wave, steps, vstart):
    w = wl.fluid_domain(*dims, P, seed=seed, steps=steps, waveform=wave)
    st = wl.random_state(w, 70 + seed, fields=("vx", "vy", "vz")) if vstart else {}
    f = bv.Simulation.from_workload(w, tuning=bv.TUNE_FUSED)        # (small grid: the library would not fuse by itself)
    assert f.mode_bits() & bv.MODE_FUSED, "the fused sweep should take this domain"
    assert f.fused_coverage() > 0.2
    two = bv.Simulation.from_workload(w, tuning=bv.TUNE_NO_FUSED)
    assert not two.mode_bits() & bv.MODE_FUSED
    o = orc.Oracle.from_workload(w)
    for n, a in st.items():
        f.write_fields(n, a)
        two.write_fields(n, a)
        b = a.astype(np.float64).copy()
        if n == "vx": b[:, :, -1] = 0
        if n == "vy": b[:, -1, :] = 0
        if n == "vz": b[-1, :, :] = 0
        o.set(n, b)
    assert f.mode_bits() & bv.MODE_FUSED            # writing a velocity keeps the fused mode
    # odd and even step counts, graph replay and single steps
    f.step(steps - 7); f.step(1); f.step(6)
    two.step(steps)
    o.step(steps)
    compare_state(f, o, rel=2e-5 if vstart else 1e-4)
    peak, rms = f.read_peak_pressure()
    compare_map(peak, o.get("peak"))
    compare_map(rms, o.get("rms_amp"))
    _same(f, two, bv)
    assert f.padding_nonzeros() == 0 and two.padding_nonzeros() == 0      # nothing wrote into the zero ghost cells
    # leaving the fused mode in the middle of a run (a caller writes a stress): sigma_yy / sigma_zz are filled in
    # and the run continues on the two passes, bit-identical to the context that never fused
    sxx = f.read_fields("sxx")
    f.write_fields("sxx", sxx)
    two.write_fields("sxx", sxx)
    assert not f.mode_bits() & bv.MODE_FUSED
    f.step(9); two.step(9)
    _same(f, two, bv)
    f.close(); two.close()


def test_fused_step_phase_leaves_the_fused_mode(bv):
    w = wl.fluid_domain(150, 60, 70, 8, seed=6, steps=30)
    f = bv.Simulation.from_workload(w, tuning=bv.TUNE_FUSED)
    two = bv.Simulation.from_workload(w, tuning=bv.TUNE_NO_FUSED)
    f.step(11); two.step(11)
    assert f.mode_bits() & bv.MODE_FUSED
    for s in (f, two):
        for ph in range(3):
            s.step_phase(ph)
    assert not f.mode_bits() & bv.MODE_FUSED
    f.step(5); two.step(5)
    _same(f, two, bv)
    f.close(); two.close()


def test_fused_on_config2_layout_short(bv):
    """config 2 at full size, 40 steps from a random velocity field: fused vs two-pass bit for bit (the oracle
    comparison of the full-size default path lives in test_gpu_full_runs.py)"""
    w = wl.make(2, steps=40)
    w.rms_begin = 20
    st = wl.random_state(w, 9, fields=("vx", "vy", "vz"))
    f = bv.Simulation.from_workload(w)
    assert f.mode_bits() & bv.MODE_FUSED and f.fused_coverage() > 0.5, f.fused_coverage()
    two = bv.Simulation.from_workload(w, tuning=bv.TUNE_NO_FUSED)
    for n, a in st.items():
        f.write_fields(n, a); two.write_fields(n, a)
    f.step(40); two.step(40)
    for n in ("vx", "vy", "vz", "sxx", "syy", "szz", "sxy", "rxx", "ryy", "p"):
        assert np.array_equal(f.read_fields(n), two.read_fields(n)), n
    pa, ra = f.read_peak_pressure()
    pb, rb = two.read_peak_pressure()
    assert np.array_equal(pa, pb) and np.array_equal(ra, rb)
    f.close(); two.close()


def _check_lists(sim, nx, ny, nz, P):
    """lists 0 + 1 and 0 + 2 cover every tile-plane exactly once; no boundary of a fused item lies inside, or within
    two planes of, a z slab (the chunk would recompute vz there without the psi it does not own)"""
    cover = {}
    for which in (0, 1, 2):
        it, rows = sim.work_items(which)
        cnt = np.zeros(((ny + rows - 1) // rows, (nx + 63) // 64, nz), np.int32)
        for bx, by, a, b in it:
            assert 0 <= a < b <= nz
            cnt[by, bx, a:b] += 1
            if which == 0 and P > 0:
                for e in (a, b):
                    assert e in (0, nz) or P + 2 <= e <= nz - P - 1, (bx, by, a, b)
        cover[which] = (cnt, rows)
    f, v, st = cover[0][0], cover[1][0], cover[2][0]
    assert ((f + v) == 1).all()
    g = cover[2][1] // 8
    assert ((f[::g] + st) == 1).all()
    if g > 1 and f.shape[0] % g == 0:
        assert (f[::g] == f[1::g]).all()          # a 64 x 16 stress tile is fused as a whole


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_work_lists_partition_the_grid(bv, cfg):
    w = wl.make(cfg, steps=2)
    sim = bv.Simulation.from_workload(w)
    assert sim.mode_bits() & bv.MODE_FUSED
    _check_lists(sim, w.nx, w.ny, w.nz, w.pml)
    sim.close()


def test_fused_run_that_would_start_inside_the_top_slab(bv):
    """a solid box just below the top z slab leaves an all-fluid run that starts INSIDE the slab (config 3 has such
    tile columns): it must stay with the two passes"""
    nx, ny, nz, P = 150, 80, 110, 24
    w = wl.fluid_domain(nx, ny, nz, P, seed=7, steps=24, solid_boxes=0)
    w.index_map[76:86, 30:50, 30:100] = 4            # no fused plane in 73..88: the run above would start at 89 > nz-P-1 = 85
    w.index_map[16:22, 28:52, 90:140] = 5            # ... and here the run below would end at 13 < P+2 = 26
    st = wl.random_state(w, 77, fields=("vx", "vy", "vz"))
    f = bv.Simulation.from_workload(w, tuning=bv.TUNE_FUSED)
    two = bv.Simulation.from_workload(w, tuning=bv.TUNE_NO_FUSED)
    assert f.mode_bits() & bv.MODE_FUSED
    _check_lists(f, nx, ny, nz, P)
    for n, a in st.items():
        f.write_fields(n, a); two.write_fields(n, a)
    f.step(24); two.step(24)
    _same(f, two, bv)
    f.close(); two.close()
