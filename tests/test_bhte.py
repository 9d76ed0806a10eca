"""NEXT-4: thermal step.

CPU part: pins of the fp64 oracle ``oracle/bhte_oracle.py`` against closed forms of the
discretised model and textbook special cases, chosen so that a plausible mistake (a dropped term, a
wrong sign, a wrong face mean, a non-conservative stencil, a wrong dose base) fails one of them.
GPU part (``-m gpu``): the CUDA path behind ``bvfdtd_bhte_*`` against the oracle, element by element.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

from oracle import bhte_oracle as bo
from paper_2301_12727_b200 import workloads as wl


def _mode(nz, ny, nx, mz=1, my=1, mx=1):
    """Discrete Dirichlet eigenmode of the 7-point Laplacian on the cell grid, and its eigenvalue
    factor sum_a 4 sin^2(pi m_a / (2 (N_a - 1)))  (times k / dx^2)."""
    z = np.sin(np.pi * mz * np.arange(nz) / (nz - 1))
    y = np.sin(np.pi * my * np.arange(ny) / (ny - 1))
    x = np.sin(np.pi * mx * np.arange(nx) / (nx - 1))
    lam = sum(4.0 * math.sin(math.pi * m / (2.0 * (n - 1))) ** 2 for m, n in ((mz, nz), (my, ny), (mx, nx)))
    return z[:, None, None] * y[None, :, None] * x[None, None, :], lam


def test_eigenmode_decay_with_perfusion():
    """Homogeneous medium, no source: a discrete eigenmode decays by exactly
    g = 1 - dt (k lam / dx^2 + w) / (rho C) per step (amplification factor of forward Euler)."""
    nz, ny, nx = 9, 11, 13
    k, rc, w, dx = 0.5, 3.6e6, 4.0e4, 1e-3
    dt = 0.5 * bo.max_stable_dt([[k, rc, w]], dx)
    o = bo.BhteOracle([[k, rc, w]], np.zeros((nz, ny, nx), np.uint8), dx, dt)
    mode, lam = _mode(nz, ny, nx, 2, 1, 3)
    o.set_temperature(37.0 + 2.0 * mode)
    o.step(25, 1.0)
    g = 1.0 - dt * (k * lam / dx ** 2 + w) / rc
    np.testing.assert_allclose(o.T - 37.0, 2.0 * mode * g ** 25, rtol=0, atol=1e-12)
    # the same mode without perfusion decays more slowly: the perfusion term has the right sign
    assert 0.0 < g < 1.0 - dt * k * lam / dx ** 2 / rc


def test_eigenmode_heating_geometric_sum():
    """A source shaped like an eigenmode drives that mode only: a_{n+1} = g a_n + s dt q0 / (rho C)."""
    nz, ny, nx = 8, 8, 10
    k, rc, w, dx, q0, s = 0.6, 4.0e6, 1.0e3, 5e-4, 3.0e5, 0.3
    dt = 0.4 * bo.max_stable_dt([[k, rc, w]], dx)
    o = bo.BhteOracle([[k, rc, w]], np.zeros((nz, ny, nx), np.uint8), dx, dt)
    mode, lam = _mode(nz, ny, nx)
    o.set_heat(q0 * mode)
    o.step(40, s)
    g = 1.0 - dt * (k * lam / dx ** 2 + w) / rc
    a = s * dt * q0 / rc * (1.0 - g ** 40) / (1.0 - g)
    np.testing.assert_allclose(o.T - 37.0, a * mode, rtol=0, atol=1e-12 * a + 1e-15)
    # ultrasound off: the source is not applied
    o2 = bo.BhteOracle([[k, rc, w]], np.zeros((nz, ny, nx), np.uint8), dx, dt)
    o2.set_heat(q0 * mode)
    o2.step(5, 0.0)
    assert np.all(o2.T == 37.0)


def test_energy_conservation_heterogeneous():
    """Conservative stencil: with no perfusion, and while the heat has not reached the border (the
    explicit stencil moves it one cell per step), sum rho C (T - T_b) = n dt sum Q exactly, whatever
    the conductivities are.  A stencil that uses the cell's own k on its faces fails this."""
    rng = np.random.default_rng(5)
    n = 21
    table = [[0.6, 4.18e6, 0.0], [0.3, 2.5e6, 0.0], [1.2, 3.0e6, 0.0]]
    idx = rng.integers(0, 3, (n, n, n)).astype(np.uint8)
    dx = 1e-3
    dt = 0.9 * bo.max_stable_dt(table, dx)
    o = bo.BhteOracle(table, idx, dx, dt)
    Q = np.zeros((n, n, n))
    Q[9:12, 9:12, 9:12] = rng.random((3, 3, 3)) * 1e6
    o.set_heat(Q)
    steps = 7                       # heat front at most 7 cells from the 3-cube: stays off the border
    o.step(steps, 1.0)
    rc = np.asarray(table)[:, 1][idx]
    assert np.isclose((rc * (o.T - 37.0)).sum(), steps * dt * Q.sum(), rtol=1e-12)
    assert (o.T - 37.0)[10, 10, 10] > 0 and np.all(o.T >= 37.0)


def test_face_conductivity_is_the_composite_wall():
    """One hot cell next to a cell of another material: after one step the neighbour has gained
    dt / (rho C dx^2) * DT / (1/(2 ka) + 1/(2 kb)) -- two half cells in series (composite wall)."""
    table = [[0.6, 4.0e6, 0.0], [0.2, 2.0e6, 0.0]]
    idx = np.zeros((7, 7, 7), np.uint8)
    idx[3, 3, 4] = 1
    dx, dt = 1e-3, 0.05
    for axis_cell in ((3, 3, 4),):
        o = bo.BhteOracle(table, idx, dx, dt)
        T0 = np.full((7, 7, 7), 37.0)
        T0[3, 3, 3] = 38.0                      # material 0, its +x neighbour is material 1
        o.set_temperature(T0)
        o.step(1, 1.0)
        series = 1.0 / (1.0 / (2 * 0.6) + 1.0 / (2 * 0.2))
        assert np.isclose(o.T[axis_cell] - 37.0, dt / (2.0e6 * dx ** 2) * series * 1.0, rtol=1e-13)
        # the -x neighbour (same material): plain k
        assert np.isclose(o.T[3, 3, 2] - 37.0, dt / (4.0e6 * dx ** 2) * 0.6, rtol=1e-13)
        # the hot cell lost what its six neighbours gained (in energy)
        gained = 5 * dt / dx ** 2 * 0.6 + dt / dx ** 2 * series
        assert np.isclose(38.0 - o.T[3, 3, 3], gained / 4.0e6, rtol=1e-12)


def test_insulating_layer_blocks_heat():
    """A layer of vanishing conductivity: nothing crosses it (series mean -> 0; an arithmetic mean
    would let half of the neighbour's conductivity through)."""
    table = [[0.6, 4.0e6, 0.0], [1e-12, 4.0e6, 0.0]]
    idx = np.zeros((12, 9, 9), np.uint8)
    idx[6, :, :] = 1
    dx = 1e-3
    dt = 0.9 * bo.max_stable_dt(table, dx)
    o = bo.BhteOracle(table, idx, dx, dt)
    Q = np.zeros(idx.shape)
    Q[3, 4, 4] = 1e7
    o.set_heat(Q)
    o.step(60, 1.0)
    assert o.T[5, 4, 4] - 37.0 > 1e-3
    assert np.abs(o.T[7:] - 37.0).max() < 1e-9


def test_borders_held_and_dose_closed_form():
    """Borders stay at T_b (L99); at a constant temperature CEM43 = t/60 * R^(43 - T), R = 0.25 below
    43 C and 0.5 from 43 C up [48]."""
    idx = np.zeros((6, 6, 6), np.uint8)
    for T_b, rate in ((37.0, 0.25 ** 6.0), (45.0, 0.5 ** -2.0), (43.0, 1.0)):
        o = bo.BhteOracle([[0.5, 3.6e6, 1e4]], idx, 1e-3, 0.1, T_b=T_b)
        o.step(30, 1.0)
        np.testing.assert_allclose(o.dose, 30 * 0.1 / 60.0 * rate, rtol=1e-13)
        assert np.all(o.T == T_b) and np.all(o.tmax == T_b)
    o = bo.BhteOracle([[0.5, 3.6e6, 0.0]], idx, 1e-3, 0.1)
    o.set_heat(np.full(idx.shape, 1e6))
    o.set_temperature(np.full(idx.shape, 39.0))
    o.step(3, 1.0)
    for face in (o.T[0], o.T[-1], o.T[:, 0], o.T[:, -1], o.T[:, :, 0], o.T[:, :, -1]):
        assert np.all(face == 37.0)
    assert np.all(o.T[1:-1, 1:-1, 1:-1] > 37.0)
    assert np.all(o.tmax[1:-1, 1:-1, 1:-1] >= 39.0)      # the running maximum saw the initial state


def test_heat_source_plane_wave_value():
    """Hand-computed: p = 1e5 Pa in (rho 1000, c 1500, alpha 10 Np/m): I = 1e10 / 3e6 = 3333.33 W/m^2,
    Q = 2 alpha I = 66666.7 W/m^3; bone keeps 0.16 of it (L99)."""
    table = [[1000.0, 1500.0, 0.0, 10.0, 0.0], [2000.0, 3000.0, 1500.0, 100.0, 200.0]]
    idx = np.array([[[0, 1]]], np.uint8)
    Q = bo.heat_source(np.full((1, 1, 2), 1e5), table, [1.0, 0.16], idx)
    assert np.isclose(Q[0, 0, 0], 66666.66666666667, rtol=1e-14)
    assert np.isclose(Q[0, 0, 1], 0.16 * 2 * 100.0 * 1e10 / (2 * 6e6), rtol=1e-14)
    assert np.isclose(bo.heat_source(np.full((1, 1, 2), 1e5), table, [1.0, 0.16], idx, scale=0.5)[0, 0, 0], 33333.333333333336)


def test_stability_bound_is_sharp_enough():
    """At the bound every update coefficient is non-negative (maximum principle: no undershoot below
    T_b from a non-negative source); well above it the checkerboard mode grows."""
    table = [[0.6, 4.0e6, 2e4], [0.3, 2.0e6, 0.0]]
    rng = np.random.default_rng(2)
    idx = rng.integers(0, 2, (9, 9, 9)).astype(np.uint8)
    dx = 1e-3
    dt = bo.max_stable_dt(table, dx)
    o = bo.BhteOracle(table, idx, dx, dt)
    Q = np.zeros(idx.shape); Q[4, 4, 4] = 1e7
    o.set_heat(Q)
    o.step(50, 1.0)
    assert o.T.min() >= 37.0 and np.isfinite(o.T).all()
    o = bo.BhteOracle([[0.6, 4.0e6, 0.0]], np.zeros((9, 9, 9), np.uint8), dx, 2.5 * bo.max_stable_dt([[0.6, 4.0e6, 0.0]], dx))
    cb = (np.indices((9, 9, 9)).sum(0) % 2) * 2.0 - 1.0
    o.set_temperature(37.0 + 1e-3 * cb)
    with np.errstate(over="ignore"):
        o.step(30, 0.0)
    assert np.abs(o.T - 37.0).max() > 1.0


# ------------------------------------------------------------------------------------------
# GPU parity (through the C ABI)
# ------------------------------------------------------------------------------------------

def _thermal_case(nx, ny, nz, seed, n_mat=5):
    w = wl.thermal_domain(nx, ny, nz, seed, n_mat=n_mat)
    return w


def _run_pair(w, schedule, track_max=True, T0=None):
    from paper_2301_12727_b200 import binding as bv
    sim = bv.Bhte(w["nx"], w["ny"], w["nz"], w["dx"], w["dt"], w["table"], w["index_map"], T_b=w["T_b"], track_max=track_max)
    o = bo.BhteOracle(w["table"], w["index_map"], w["dx"], w["dt"], T_b=w["T_b"])
    sim.set_heat(w["Q"].astype(np.float32))
    o.set_heat(w["Q"].astype(np.float32))
    if T0 is not None:
        sim.set_temperature(T0.astype(np.float32))
        o.set_temperature(T0.astype(np.float32))
    for n, s in schedule:
        sim.step(n, s)
        o.step(n, s)
    return sim, o


def _check(sim, o, w, track_max=True):
    """Tolerances: the rise T - T_b is the fp32 state: relative L2 1e-5, max
    error 2e-5 of the largest rise; the temperature itself adds half an ulp of fp32 at 37-64 C (4e-6)."""
    ref = o.T - w["T_b"]
    rise = sim.read("rise").astype(np.float64)
    assert np.linalg.norm(rise - ref) <= 1e-5 * np.linalg.norm(ref), np.linalg.norm(rise - ref) / np.linalg.norm(ref)
    assert np.abs(rise - ref).max() <= 2e-5 * np.abs(ref).max()
    T = sim.read("T").astype(np.float64)
    assert np.abs(T - o.T).max() <= 2e-5 * np.abs(ref).max() + 4e-6
    dose = sim.read("dose").astype(np.float64)
    np.testing.assert_allclose(dose, o.dose, rtol=2e-4)
    if track_max:
        tm = sim.read("tmax").astype(np.float64)
        assert np.abs(tm - o.tmax).max() <= 2e-5 * np.abs(ref).max() + 4e-6
    for face in (T[0], T[-1], T[:, 0], T[:, -1], T[:, :, 0], T[:, :, -1]):
        assert np.all(face == np.float32(w["T_b"]))


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [(70, 37, 29), (64, 16, 12), (131, 50, 41), (9, 9, 9)])
def test_gpu_bhte_parity(shape):
    """Heterogeneous 5-material domain, on (duty 0.3) / off schedule, sizes spanning several tiles,
    ragged tails in x and y and several z chunks."""
    nx, ny, nz = shape
    w = _thermal_case(nx, ny, nz, seed=11 + nx)
    sim, o = _run_pair(w, [(40, 0.3), (25, 0.0), (10, 1.0)])
    _check(sim, o, w)
    assert o.T.max() - w["T_b"] > 1.0          # the case really heats
    sim.close()


@pytest.mark.gpu
def test_gpu_bhte_initial_state_no_max_and_dose_branch():
    """Initial temperature above 43 C in part of the domain (both dose branches), no running maximum."""
    w = _thermal_case(48, 33, 21, seed=3)
    rng = np.random.default_rng(4)
    T0 = w["T_b"] + 9.0 * rng.random((21, 33, 48))
    sim, o = _run_pair(w, [(30, 1.0)], track_max=False, T0=T0)
    _check(sim, o, w, track_max=False)
    assert (o.T > 43.0).any() and (o.T[1:-1, 1:-1, 1:-1] < 43.0).any()
    with pytest.raises(Exception):
        sim.read("tmax")
    sim.close()


@pytest.mark.gpu
def test_gpu_bhte_validation():
    from paper_2301_12727_b200 import binding as bv
    w = _thermal_case(24, 20, 16, seed=1)
    with pytest.raises(bv.BvfdtdError):       # unstable time step
        bv.Bhte(24, 20, 16, w["dx"], 50 * w["dt"], w["table"], w["index_map"])
    bad = w["table"].copy(); bad[1, 0] = 0.0
    with pytest.raises(bv.BvfdtdError):       # k must be positive
        bv.Bhte(24, 20, 16, w["dx"], w["dt"], bad, w["index_map"])
    idx = w["index_map"].copy(); idx[3, 3, 3] = 200
    with pytest.raises(bv.BvfdtdError):       # index outside the table
        bv.Bhte(24, 20, 16, w["dx"], w["dt"], w["table"], idx)


@pytest.mark.gpu
def test_gpu_heat_source_from_acoustic_run():
    """bvfdtd_heat_source on the rms window of an acoustic run = the oracle's Q from the oracle's
    rms amplitude (both sides from their own run), and it feeds the thermal context on the device."""
    from oracle import fdtd_oracle as orc
    from paper_2301_12727_b200 import binding as bv
    w = wl.random_domain(40, 36, 44, 6, seed=21, steps=120, waveform=1)
    w.rms_begin = 120 - w.spp
    sim = bv.Simulation.from_workload(w, device="cuda:0")
    sim.step(w.steps)
    o = orc.Oracle.from_workload(w)
    o.step(w.steps)
    frac = np.where(w.table[:, 2] > 0, 0.16, 1.0)
    Qd = sim.heat_source(frac, scale=2.5)                      # device tensor, dense nx*ny*nz
    Qref = bo.heat_source(o.get("rms_amp"), w.table, frac, w.index_map, scale=2.5)
    Q = Qd.cpu().numpy().reshape(Qref.shape).astype(np.float64)
    m = Qref > 0.01 * Qref.max()
    assert m.any()
    assert np.abs(Q[m] / Qref[m] - 1).max() <= 2e-3           # (amplitude tolerance 1e-3)^2
    assert np.all(Q[Qref == 0] == 0)
    tw = wl.thermal_table_for(w.table)
    th = bv.Bhte(w.nx, w.ny, w.nz, w.dx, 0.01, tw, w.index_map)
    th.set_heat(Qd)
    th.step(5, 1.0)
    ob = bo.BhteOracle(tw, w.index_map, w.dx, 0.01)
    ob.set_heat(Q)
    ob.step(5, 1.0)
    rise = th.read("T").astype(np.float64) - 37.0
    assert np.linalg.norm(rise - (ob.T - 37.0)) <= 1e-5 * np.linalg.norm(ob.T - 37.0) + 1e-7 * rise.size ** 0.5
    th.close(); sim.close()


@pytest.mark.gpu
def test_gpu_bhte_full_size_config2_cropped_oracle():
    """Config 2's grid (300 x 300 x 450, 128 materials) in the launch configuration the bench times.
    The explicit stencil moves information one cell per step, so after n steps the cells of a
    sub-box that lie at least n cells inside it depend on the sub-box only: the oracle runs on two
    cropped sub-boxes (around the focus inside the skull cap, and across the skull) and is compared
    there cell by cell; outside, properties that hold at any size (borders at T_b, no cooling below
    T_b, untouched far field)."""
    from paper_2301_12727_b200 import binding as bv
    w = wl.thermal_config2()
    n = 6
    sim = bv.Bhte(w["nx"], w["ny"], w["nz"], w["dx"], w["dt"], w["table"], w["index_map"], T_b=w["T_b"], track_max=True)
    sim.set_heat(w["Q"])
    sim.step(n, 1.0)
    rise = sim.read("rise").astype(np.float64)
    dose = sim.read("dose").astype(np.float64)
    nz, ny, nx = rise.shape
    kf = int(np.unravel_index(np.argmax(w["Q"]), w["Q"].shape)[0])
    for (z0, y0, x0) in ((kf - 24, ny // 2 - 24, nx // 2 - 24), (60, 100, 120), (nz - 48, ny - 48, nx - 48), (0, 0, 0)):
        sl = (slice(z0, z0 + 48), slice(y0, y0 + 48), slice(x0, x0 + 48))
        o = bo.BhteOracle(w["table"], w["index_map"][sl], w["dx"], w["dt"], T_b=w["T_b"])
        o.set_heat(w["Q"][sl])
        o.step(n, 1.0)
        # the crop's own faces are held at T_b by the oracle: valid cells are n inside, except where
        # a crop face is a face of the full box (there the border condition is the real one)
        lo = [0 if a == 0 else n for a in (z0, y0, x0)]
        hi = [48 if a + 48 == full else 48 - n for a, full in ((z0, nz), (y0, ny), (x0, nx))]
        inner = tuple(slice(l, h) for l, h in zip(lo, hi))
        ref = (o.T - w["T_b"])[inner]
        got = rise[sl][inner]
        assert np.abs(got - ref).max() <= 2e-5 * max(np.abs(ref).max(), 1e-30) + 1e-12
        np.testing.assert_allclose(dose[sl][inner], o.dose[inner], rtol=2e-4)
    assert rise.min() >= 0.0 and rise.max() > 0.0
    for face in (rise[0], rise[-1], rise[:, 0], rise[:, -1], rise[:, :, 0], rise[:, :, -1]):
        assert np.all(face == 0.0)
    sim.close()


@pytest.mark.gpu
def test_gpu_bhte_uniform_regions_and_interfaces():
    """Large single-material regions (the warp-uniform path of the kernel) separated by a slab and a
    box of other materials (the general path), including interfaces that cut a warp's cells."""
    w = _thermal_case(150, 40, 45, seed=8)
    idx = np.ones((45, 40, 150), np.uint8)
    idx[10:14] = 2
    idx[20:30, 8:20, 30:71] = 3
    idx[:, :, 129:] = 0
    idx[31:, 33:, :] = 4
    w["index_map"] = idx
    sim, o = _run_pair(w, [(50, 0.5), (20, 0.0)])
    _check(sim, o, w)
    assert o.T.max() - w["T_b"] > 1.0
    sim.close()
