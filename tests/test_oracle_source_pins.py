"""Pins of the oracle's SOURCE (reading P7) and of its staggered material averaging (reading P2),
CPU only.  Round-1's pins used zero delays and amplitude-cancelling ratios, so `orc_inject` and
`waveform()` (sign, delay, burst gate, ramp) and the 4-cell shear-node means were held by nothing.

  S1  sign, amplitude, delay: orc_inject alone on a zero state gives p = -tr(sigma)/3 = +amp w(t_n - delay)
      at the source cells (positive amp -> positive pressure, "stress source"), touches
      nothing else, and never the memory variables
  S2  time translation: delaying every source cell by m dt delays every probe trace by exactly m steps
  S3  burst gate: no injection for t < 0 and for t >= n_cycles / f
  S4  CW ramp: raised cosine of length n_cycles / f (value 1/4 at a third, 3/4 at two thirds, 1 after),
      steady state independent of n_cycles
  A1  laminate pins of reading P2: on a period-2 laminate (A, B, A, B ... along one axis) every shear
      node of the two kinds that straddle the laminate sees two cells of A and two of B, and every
      velocity node across it one of each, so a shear mode polarised ALONG the laminate axis is an exact
      eigen-mode of the heterogeneous discrete system with rho = arithmetic mean, mu = harmonic mean,
      tau_s = arithmetic mean -> the closed-form dispersion relation T1 with those constants (1e-9).
      An arithmetic mu mean, a harmonic tau_s mean or a harmonic rho mean each fail it.
  A2  the C-PML of a solid at oblique incidence on an x face (all nine psi terms of that face are live:
      D+x sxx, D-x sxy, D-x sxz, D-x vx, D+x vy, D+x vz): reflection bound against a larger box.

The expected values are closed forms written here from DESIGN.md section 2, not taken from the oracle.
"""
import cmath
import math

import numpy as np
import pytest

from oracle import fdtd_oracle as fo

from test_oracle_pins import (BONE, DX, F0, TAU_SIGMA, WATER, K_of, _along, sls_constants, solve_omega)

AX = "xyz"


def _water_box(n=12, pml=0, spp=60):
    dt = 1.0 / (F0 * spp)
    o = fo.Oracle(n, n, n, pml, DX, dt, np.array([WATER, (1040.0, 1546.0, 0.0, 30.0, 0.0)]),
                  np.ones((n, n, n), np.uint8), F0)      # lossy fluid: memory variables are live
    return o, dt


def _cell(n, i, j, k):
    return i + n * (j + n * k)


# --------------------------------------------------------------------------------------
# S1  sign, amplitude, delay of one injection
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("step", [13, 23, 95])
def test_S1_inject_sign_amplitude_delay(step):
    n = 12
    o, dt = _water_box(n)
    cells = np.array([_cell(n, 3, 4, 5), _cell(n, 6, 6, 6), _cell(n, 8, 2, 9), _cell(n, 1, 1, 1)])
    amp = np.array([1.0, -0.5, 2.25, 3.0])
    delay = np.array([0.0, 3.3 * dt, 11.0 * dt, 200.0 * dt])      # the last one has not started yet
    ncyc = 3
    o.set_source(cells, amp, delay, 0, F0, ncyc)
    o.step_index = step
    o.inject()
    t = step * dt - delay
    w = np.where((t >= 0) & (t < ncyc / F0), np.sin(2 * np.pi * F0 * t), 0.0)
    expect = amp * w                                              # +amp w: positive amp -> positive pressure
    assert np.abs(expect[:3]).min() > 1e-3                        # the test is not vacuous
    got = o.probe("p", cells)
    assert np.allclose(got, expect, rtol=0, atol=1e-15)
    assert got[3] == 0.0
    sxx = o.probe("sxx", cells)
    assert np.allclose(sxx, -expect, rtol=0, atol=1e-15)
    for name in ("syy", "szz"):                                   # isotropic: the three normal stresses are one number
        assert np.array_equal(o.probe(name, cells), sxx)
    # nothing else is touched: no other cell, no shear stress, no velocity, no memory variable
    for name in fo.FIELDS:
        a = o.get(name)
        if name in ("sxx", "syy", "szz"):
            a.ravel()[cells] = 0.0
        assert not a.any(), name
    o.close()


# --------------------------------------------------------------------------------------
# S2  time translation
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("waveform", [0, 1])
def test_S2_delay_is_a_time_shift(waveform):
    n, m, steps = 14, 9, 130
    src = np.array([_cell(n, 4, 5, 3), _cell(n, 5, 5, 3), _cell(n, 9, 8, 4)])
    amp = np.array([1.0, 0.7, -1.3])
    base = np.array([0.0, 2.5, 6.0])
    rec = [_cell(n, 7, 7, 10), _cell(n, 3, 9, 8)]
    traces = []
    for shift in (0, m):
        o, dt = _water_box(n)
        o.set_source(src, amp, (base + shift) * dt, waveform, F0, 2)
        tr = np.zeros((steps, len(rec)))
        for s in range(steps):
            o.step(1)
            tr[s] = o.probe("p", rec)
        traces.append(tr)
        o.close()
    scale = np.abs(traces[0]).max()
    assert scale > 0
    assert not traces[1][:m].any()                                # nothing before the delayed start
    assert np.abs(traces[1][m:] - traces[0][:-m]).max() <= 1e-12 * scale
    # and the shift is towards LATER times (t - delay, not t + delay)
    assert np.abs(traces[1][:-m] - traces[0][m:]).max() > 1e-2 * scale


# --------------------------------------------------------------------------------------
# S3  burst gate
# --------------------------------------------------------------------------------------
def test_S3_burst_gate():
    n, spp, ncyc = 12, 60, 3
    o, dt = _water_box(n, spp=spp)
    c = [_cell(n, 6, 6, 6)]
    d = 4.5 * dt
    o.set_source(c, [1.0], [d], 0, F0, ncyc)
    inc = []
    for step in range(0, ncyc * spp + 12):
        o.set("sxx", np.zeros((n, n, n)))
        o.step_index = step
        o.inject()
        inc.append(-o.probe("sxx", c)[0])
    inc = np.array(inc)
    steps = np.arange(inc.size)
    t = steps * dt - d
    on = (t >= 0) & (t < ncyc / F0)
    assert not inc[~on].any()                                     # gated off before the delay and after n_cycles / f
    assert (steps[on][0], steps[on][-1]) == (5, 4 + ncyc * spp)
    assert np.allclose(inc[on], np.sin(2 * np.pi * F0 * t[on]), atol=1e-14)
    o.close()


# --------------------------------------------------------------------------------------
# S4  CW ramp
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("ncyc", [1, 2, 4])
def test_S4_cw_ramp(ncyc):
    n, spp = 12, 60
    o, dt = _water_box(n, spp=spp)
    c = [_cell(n, 5, 6, 7)]
    o.set_source(c, [1.0], [0.0], 1, F0, ncyc)

    def w_at(step):
        o.set("szz", np.zeros((n, n, n)))
        o.step_index = step
        o.inject()
        return -o.probe("szz", c)[0]

    T = ncyc * spp                                                # ramp length in steps
    # envelope 1/4 at T/3, 3/4 at 2T/3 (raised cosine 1/2 (1 - cos(pi t / T))), 1 from T on
    for num, env in ((1, 0.25), (2, 0.75)):
        s = num * T // 3
        assert s * 3 == num * T
        carrier = math.sin(2 * math.pi * s / spp)
        assert abs(carrier) > 0.5
        assert abs(w_at(s) - env * carrier) < 1e-14
    for s in (T + 7, T + 15, 5 * T + 11):
        assert abs(w_at(s) - math.sin(2 * math.pi * s / spp)) < 1e-13
    # monotone envelope on the ramp: sampled at the carrier's maxima (quarter periods)
    env = [w_at(q * spp + spp // 4) for q in range(ncyc)]
    assert all(0 < e <= 1 + 1e-15 for e in env) and env == sorted(env)
    assert w_at(0) == 0.0
    o.close()


def test_S4_steady_state_independent_of_ramp_length():
    """after both ramps have ended the two sources inject the same values, so a probe's steady-state
    amplitude is the same (the run is long enough for the ramp transient to leave through the PML)"""
    n, spp, steps = 36, 60, 11 * 60
    amps = []
    for ncyc in (1, 3):
        dt = 1.0 / (F0 * spp)
        o = fo.Oracle(8, 8, n, 8, DX, dt, np.array([WATER]), np.zeros((n, 8, 8), np.uint8), F0, periodic=(1, 1, 0),
                      rms_begin=steps - 2 * spp)
        cells = [i + 8 * (j + 8 * 12) for j in range(8) for i in range(8)]      # plane source: a plane wave
        o.set_source(cells, np.ones(64), np.zeros(64), 1, F0, ncyc)
        o.step(steps)
        amps.append(o.get("rms_amp")[22, 3, 3])
        o.close()
    assert amps[0] > 0 and abs(amps[1] / amps[0] - 1) < 2e-3


# --------------------------------------------------------------------------------------
# A1  laminate pins of the staggered averages (reading P2)
# --------------------------------------------------------------------------------------
MAT_A = (1900.0, 2800.0, 1500.0, 150.0, 260.0)
MAT_B = (1300.0, 2100.0, 1000.0, 60.0, 90.0)


@pytest.mark.parametrize("lam,axis,pol", [(0, 1, 0), (0, 2, 0), (1, 2, 1), (1, 0, 1), (2, 0, 2), (2, 1, 2)])
def test_A1_laminate_shear_mode(lam, axis, pol):
    """laminate along `lam` (= the polarisation), shear mode travelling along `axis`: the fields are
    (v_pol, s_{axis,pol}, r_{axis,pol}), uniform along the laminate"""
    assert lam == pol and axis != pol
    N, nsteps, m_wave = 64, 500, 5
    n = [4, 4, 4]
    n[axis] = N
    dt = 1.0 / (F0 * 56)
    shape = (n[2], n[1], n[0])
    idx = _along(lam, (np.arange(n[lam]) % 2).astype(np.float64), shape).astype(np.uint8)
    o = fo.Oracle(n[0], n[1], n[2], 0, DX, dt, np.array([MAT_A, MAT_B]), idx, F0, periodic=(1, 1, 1))
    tA, muA = sls_constants(MAT_A[0], MAT_A[2], MAT_A[4])
    tB, muB = sls_constants(MAT_B[0], MAT_B[2], MAT_B[4])
    rho = 0.5 * (MAT_A[0] + MAT_B[0])            # 2-cell arithmetic mean at the velocity node
    MR = 2.0 / (1.0 / muA + 1.0 / muB)           # 4-cell harmonic mean (two cells of each)
    tau = 0.5 * (tA + tB)                        # 4-cell arithmetic mean of tau_s
    k = 2.0 * math.pi * m_wave / (N * DX)
    w = solve_omega(rho, MR, tau, k, DX, dt)
    W = 2.0 / dt * cmath.sin(w * dt / 2.0)
    K = K_of(k, DX).real
    v_hat = -K / (W * rho)
    r_hat = -(MR * tau) * (-1j * K * v_hat) / (cmath.cos(w * dt / 2.0) + 1j * W * TAU_SIGMA)
    xi, xh = np.arange(N) * DX, (np.arange(N) + 0.5) * DX
    ab = "".join(sorted(AX[axis] + AX[pol]))

    def snap(nn):
        tS, tV = cmath.exp(1j * w * nn * dt), cmath.exp(1j * w * (nn - 0.5) * dt)
        return {"s" + ab: (tS * np.exp(-1j * k * xh)).real, "r" + ab: (r_hat * tS * np.exp(-1j * k * xh)).real,
                "v" + AX[pol]: (v_hat * tV * np.exp(-1j * k * xi)).real}

    init, expect = snap(0), snap(nsteps)
    for name, prof in init.items():
        o.set(name, _along(axis, prof, shape))
    o.step(nsteps)
    assert abs(cmath.exp(1j * w * nsteps * dt)) < 0.3             # the mode really decays
    for name in fo.FIELDS:
        got = o.get(name)
        if name in expect:
            scale = np.abs(init[name]).max()
            assert np.abs(got - _along(axis, expect[name], shape)).max() <= 1e-9 * scale, name
        else:
            # (exactly zero up to the rounding of the node coefficients, whose four cells are summed in
            # the order A B A B at one node and B A B A at the next)
            kind_scale = np.abs(init[{"v": "v" + AX[pol], "s": "s" + ab, "r": "r" + ab}[name[0]]]).max()
            assert np.abs(got).max() <= 1e-12 * kind_scale, name
    o.close()
    # the pin discriminates: the closed form with an arithmetic mu mean or a harmonic tau mean is far off
    for MR2, tau2, rho2 in ((0.5 * (muA + muB), tau, rho), (MR, 2.0 / (1.0 / tA + 1.0 / tB), rho),
                            (MR, tau, 2.0 / (1.0 / MAT_A[0] + 1.0 / MAT_B[0]))):
        w2 = solve_omega(rho2, MR2, tau2, k, DX, dt)
        assert abs(cmath.exp(1j * (w2 - w) * nsteps * dt) - 1.0) > 1e-3


def test_A1_fluid_cell_zeroes_the_shear_node():
    """reading P2: a shear node with ANY fluid cell among its four has mu_h = 0 -- on a solid / fluid
    laminate every straddling shear node stays exactly zero whatever the velocities are"""
    n = 8
    rng = np.random.Generator(np.random.PCG64(5))
    idx = _along(0, (np.arange(n) % 2).astype(np.float64), (n, n, n)).astype(np.uint8)
    o = fo.Oracle(n, n, n, 0, DX, 1.0 / (F0 * 56), np.array([WATER, BONE]), idx, F0, periodic=(1, 1, 1))
    for name in ("vx", "vy", "vz"):
        o.set(name, rng.standard_normal((n, n, n)))
    o.step(3)
    for name in ("sxy", "sxz", "rxy", "rxz"):                     # nodes that straddle x: one fluid cell at least
        assert not o.get(name).any(), name
    syz = o.get("syz")                                            # cells (i, j..j+1, k..k+1): all bone at odd i
    assert not syz[:, :, 0::2].any() and syz[:, :, 1::2].any()
    o.close()


# --------------------------------------------------------------------------------------
# A2  C-PML of a solid, oblique incidence on an x face
# --------------------------------------------------------------------------------------
def _solid_traces(nx, off, P, steps):
    ny = nz = 30
    solid = (1900.0, 2800.0, 1500.0, 0.0, 0.0)
    dt = 1.0 / (F0 * 56)
    # only the x faces absorb; y and z are periodic so that the small and the big box differ in x only
    o = fo.Oracle(nx, ny, nz, P, DX, dt, np.array([solid]), np.zeros((nz, ny, nx), np.uint8), F0, periodic=(0, 1, 1))
    # a smooth blob of v_y: radiates P and S waves that reach the x faces at every angle and polarisation
    z, y, x = np.mgrid[0:nz, 0:ny, 0:nx]
    o.set("vy", np.exp(-((x - (off + 10)) ** 2 + (y - 15) ** 2 + (z - 15) ** 2) / 6.0))
    rec = [(off + 6) + nx * (9 + ny * 20), (off + 14) + nx * (22 + ny * 11), (off + 4) + nx * (15 + ny * 15),
           (off + 2) + nx * (5 + ny * 8)]
    out = {q: np.zeros((steps, len(rec))) for q in ("sxx", "sxy", "sxz", "vx", "vy", "vz")}
    for s in range(steps):
        o.step(1)
        for q in out:
            out[q][s] = o.probe(q, rec)
    o.close()
    return out


def test_A2_pml_solid_oblique_incidence_x_face():
    """Reflection from the x slabs of a solid (P = 10) against a box whose walls are 130 cells further out
    (no echo within 400 steps: the P wave covers 0.3 cells per step).  With the profile taken where each
    derivative lands (reading P5) the residuals are 0.3-1.0 % of the incident traces; bounds = 1.5 x those.
    Measured with mutated copies of the oracle: dropping the psi of D+x v_y or of D-x s_xy gives 3.5-9 %,
    swapping the half- for the integer-node profile in D+x v_y 1.1-1.7 % on s_xy, s_xz, v_z -- each fails."""
    P, steps, pad = 10, 400, 130
    small = _solid_traces(2 * P + 24, P, P, steps)
    big = _solid_traces(2 * P + 24 + 2 * pad, P + pad, 0, steps)
    bound = {"sxx": 0.0083, "sxy": 0.0044, "sxz": 0.0045, "vx": 0.0063, "vy": 0.0146, "vz": 0.0104}
    for q in small:
        inc = np.abs(big[q]).max()
        assert inc > 0
        res = np.abs(small[q] - big[q]).max() / inc
        assert res <= bound[q], (q, res)
