"""NEXT-3, second half: corrected phase programming of a phased array
from a point source at the target.

CPU: pins of ``oracle/refocus_oracle.py`` (time reversal of a point source's field focuses exactly;
delay convention; element sums by brute force).  GPU: ``bvfdtd_refocus_weights`` against the oracle,
and the whole chain (point-source FDTD run with the phasor sensor -> Rayleigh back to the elements ->
conjugated weights -> Rayleigh forward -> FDTD run) against the same chain through the oracles, plus
the physical property that refocusing through an aberrating plate restores pressure at the target.
"""
from __future__ import annotations

import numpy as np
import pytest

from oracle import refocus_oracle as ro
from oracle import rs_oracle
from paper_2301_12727_b200 import workloads as wl


def _array(n_elem=8, pts=5, seed=0):
    """A small irregular array: n_elem elements of `pts` surface points each (positions in metres)."""
    rng = np.random.default_rng(seed)
    centres = np.stack([rng.uniform(-8e-3, 8e-3, n_elem), rng.uniform(-8e-3, 8e-3, n_elem), rng.uniform(-2e-3, 0, n_elem)], 1)
    xyz = (centres[:, None, :] + rng.uniform(-4e-4, 4e-4, (n_elem, pts, 3)) * [1, 1, 0]).reshape(-1, 3)
    element = np.repeat(np.arange(n_elem), pts)
    area = rng.uniform(0.5, 1.5, xyz.shape[0]) * 1e-7
    return xyz, element, area


def test_time_reversal_of_a_point_source_focuses_exactly():
    """Field of a point source at r_t on single-point elements: P_m = e^{-jkR_m}/R_m.  The conjugated
    unit weights make every contribution arrive in phase at r_t: |sum_m W_m e^{-jkR_m}/R_m| =
    sum_m 1/R_m exactly, and no other phase set does better (triangle inequality)."""
    f, c0 = 500e3, 1500.0
    k = 2 * np.pi * f / c0
    xyz, _, _ = _array(12, 1, seed=1)
    target = np.array([1e-3, -2e-3, 30e-3])
    R = np.linalg.norm(xyz - target, axis=1)
    P = np.exp(-1j * k * R) / R
    E = ro.element_sums(P, np.arange(12), 12)
    W, delay = ro.phase_programming(E, f)
    focus = (W * np.exp(-1j * k * R) / R).sum()
    assert np.isclose(abs(focus), (1.0 / R).sum(), rtol=1e-12)
    assert np.allclose(np.abs(W), 1.0)
    # delay convention: element m emits cos(w (t - tau_m)); with arg E_m = -k R_m, tau_m = -R_m / c (mod T):
    # the farther element fires earlier, all arrivals coincide
    T = 1.0 / f
    arrival = (delay + R / c0) / T
    assert np.allclose(arrival - np.round(arrival), (arrival - np.round(arrival))[0], atol=1e-9)
    assert np.all((delay >= 0) & (delay < T))
    # emission Re{W e^{jwt}} equals cos(w (t - tau))
    t = 0.37 * T
    assert np.allclose((W * np.exp(1j * 2 * np.pi * f * t)).real, np.cos(2 * np.pi * f * (t - delay)), atol=1e-12)


def test_element_sums_and_point_weights_brute_force():
    rng = np.random.default_rng(3)
    xyz, element, area = _array(6, 7, seed=2)
    P = rng.standard_normal(element.size) + 1j * rng.standard_normal(element.size)
    E = ro.element_sums(P, element, 6)
    for m in range(6):
        acc = 0j
        for q in range(element.size):
            if element[q] == m:
                acc += P[q]
        assert np.isclose(E[m], acc, rtol=1e-14)
    Wp = ro.point_weights(E, element, area, u0=0.02)
    for q in range(element.size):
        assert np.isclose(Wp[q], 0.02 * area[q] * np.conj(E[element[q]]) / abs(E[element[q]]), rtol=1e-14)


def test_refocusing_through_rs_oracle_in_water_recovers_geometric_focusing():
    """Whole back-propagation in water with the Rayleigh oracle only: point source -> plane ->
    elements.  The corrected delays equal the geometric ones (d_max - d_m)/c up to a common shift,
    within the discretisation of the plane (a few degrees)."""
    f, c0 = 500e3, 1500.0
    lam = c0 / f
    xyz, element, area = _array(10, 1, seed=4)
    xyz[:, 2] = -10e-3                                           # a flat array 10 mm behind the plane z = 0
    target = np.array([0.0, 0.0, 25e-3])
    h = lam / 4
    g = (np.arange(-80, 81) * h)
    X, Y = np.meshgrid(g, g)
    plane = np.stack([X.ravel(), Y.ravel(), np.zeros(X.size)], 1)
    P_plane = rs_oracle.rayleigh(target[None, :], np.array([1.0 + 0j]), plane, f)      # point source at the target
    P_el = rs_oracle.rayleigh(plane, P_plane, xyz, f)                                   # plane radiates back
    _, delay = ro.phase_programming(ro.element_sums(P_el, element, 10), f)
    d = np.linalg.norm(xyz - target, axis=1)
    geo = (d.max() - d) / c0
    diff = (delay - geo) * f
    diff = diff - diff[0]
    diff = diff - np.round(diff)
    assert np.abs(diff).max() < 0.03, diff                       # < 11 degrees of phase


# ------------------------------------------------------------------------------------------
# GPU
# ------------------------------------------------------------------------------------------

@pytest.mark.gpu
def test_gpu_refocus_weights_match_oracle():
    from paper_2301_12727_b200 import refocus
    rng = np.random.default_rng(7)
    xyz, element, area = _array(37, 11, seed=5)
    P = (rng.standard_normal(element.size) + 1j * rng.standard_normal(element.size)) * 1e3
    perm = rng.permutation(element.size)                       # points of an element need not be contiguous
    P, element, area = P[perm], element[perm], area[perm]
    f = 250e3
    w_pts, delay, E = refocus.refocus_weights(P.astype(np.complex64), element, area, 37, f, u0=0.5)
    Er = ro.element_sums(P.astype(np.complex64), element, 37)
    unit, dr = ro.phase_programming(Er, f)
    assert np.abs(E - Er).max() <= 1e-5 * np.abs(Er).max()
    dd = (delay - dr) * f
    dd -= np.round(dd)
    assert np.abs(dd).max() <= 1e-5                              # fraction of a period
    Wr = ro.point_weights(Er, element, area.astype(np.float32), u0=0.5)
    assert np.abs(w_pts - Wr).max() <= 2e-5 * np.abs(Wr).max()


def _refocus_case():
    """Water box with a bone plate whose thickness steps from 4 to 12 voxels half way across the
    aperture (a 0.8 pi phase jump at 500 kHz) between a 12-element array and the target."""
    w = wl.random_domain(56, 56, 72, 6, seed=77, steps=1, waveform=1, n_mat=2, solid_fraction=0.0, lossy=False)
    idx = np.zeros((w.nz, w.ny, w.nx), np.uint8)
    idx[22:26] = 1
    idx[26:34, :, 28:] = 1
    table = np.array([wl.WATER, (1900.0, 2800.0, 0.0, 0.0, 0.0)])
    return w, idx, table


@pytest.mark.gpu
def test_gpu_refocusing_chain_matches_oracle_chain_and_restores_the_focus():
    from oracle import fdtd_oracle as orc
    from paper_2301_12727_b200 import refocus
    w, idx, table = _refocus_case()
    f0, dx = w.f0, w.dx
    dt, spp = wl.snapped_dt(dx, f0, 2800.0)
    k_s = w.pml + 3
    target_cell = (28, 27, 56)                                   # (i, j, k)
    steps = 12 * spp
    rng = np.random.default_rng(1)
    n_elem, pts = 12, 4
    cx, cy = rng.uniform(3, 15, n_elem) * 1e-3, rng.uniform(3, 15, n_elem) * 1e-3
    off = rng.uniform(-3e-4, 3e-4, (n_elem, pts, 2))
    el_xyz = np.stack([(cx[:, None] + off[..., 0]).ravel(), (cy[:, None] + off[..., 1]).ravel(), np.full(n_elem * pts, -6e-3)], 1)
    element = np.repeat(np.arange(n_elem), pts)
    area = np.full(n_elem * pts, (0.75e-3) ** 2)
    geom = dict(nx=w.nx, ny=w.ny, nz=w.nz, pml=w.pml, dx=dx, dt=dt, f0=f0, table=table, index_map=idx, k_s=k_s,
                target_cell=target_cell, steps=steps, window=3 * spp)

    res = refocus.back_propagate(geom, el_xyz, element, area, n_elem, u0=1.0, device="cuda:0")

    # ---- the same chain through the oracles --------------------------------------------------
    plane_ij = res["plane_ij"]
    cells = plane_ij[:, 0] + w.nx * (plane_ij[:, 1] + w.ny * k_s)
    tc = target_cell[0] + w.nx * (target_cell[1] + w.ny * target_cell[2])
    o = orc.Oracle(w.nx, w.ny, w.nz, w.pml, dx, dt, table, idx, f0, rms_begin=steps - 3 * spp)
    o.set_phasor(True)
    o.set_source(np.array([tc], np.int64), np.ones(1, np.float32), np.zeros(1, np.float32), 1, f0, 3)
    o.step(steps)
    Pfull = o.get("phasor_re") + 1j * o.get("phasor_im")
    P_plane = Pfull.reshape(-1)[cells]
    plane_xyz = np.stack([plane_ij[:, 0] * dx, plane_ij[:, 1] * dx, np.zeros(len(cells))], 1)
    P_el = rs_oracle.rayleigh(plane_xyz, P_plane, el_xyz, f0)
    E = ro.element_sums(P_el, element, n_elem)
    _, delay_ref = ro.phase_programming(E, f0)
    assert np.abs(res["E"] - E).max() <= 5e-4 * np.abs(E).max()
    dd = (res["delay"] - delay_ref) * f0
    dd -= np.round(dd)
    assert np.abs(dd).max() <= 5e-4, dd                          # 0.18 degrees of phase
    Wref = ro.point_weights(E, element, area)
    assert np.abs(res["w_pts"] - Wref).max() <= 3e-3 * np.abs(Wref).max()

    # ---- physics: corrected phases beat the geometric (water) phases at the target -------------
    tpos = np.array([target_cell[0] * dx, target_cell[1] * dx, (target_cell[2] - k_s) * dx])
    d = np.linalg.norm(el_xyz - tpos, axis=1)
    w_geo = area * np.exp(1j * 2 * np.pi * f0 / 1500.0 * d)      # in water these arrive in phase at the target
    ti, tj, tk = target_cell
    amp_ref = refocus.forward(geom, el_xyz, res["w_pts"])[tk, tj, ti]
    amp_geo = refocus.forward(geom, el_xyz, w_geo)[tk, tj, ti]
    print(f"refocus: max delay error {np.abs(dd).max():.2e} periods, target amplitude refocused {amp_ref:.4g} vs geometric {amp_geo:.4g}")
    assert amp_ref > 1.2 * amp_geo, (amp_ref, amp_geo)
