"""NEXT-1: Rayleigh-Sommerfeld field of a surface-decomposed transducer.

CPU part: the fp64 oracle (oracle/rs_oracle.py) against closed forms.  GPU part (-m gpu): the CUDA
kernel behind ``bvfdtd_rayleigh`` against the oracle, element by element."""
import math

import numpy as np
import pytest

from oracle import rs_oracle as rs
from paper_2301_12727_b200 import workloads as wl

F, C0, RHO = 500e3, 1500.0, 1000.0
LAM = C0 / F
K = 2 * math.pi / LAM


def test_element_areas_add_up():
    pos, area = wl.disc_elements(10e-3, LAM / 4)
    assert abs(area.sum() / (math.pi * 10e-3 ** 2) - 1) < 1e-12
    assert abs(area.mean() / (LAM ** 2 / 16) - 1) < 0.1           # elements of lambda^2/16
    pos, area = wl.bowl_elements(64e-3, 64e-3, LAM / 4)
    cap = 2 * math.pi * 64e-3 ** 2 * (1 - math.cos(math.asin(0.5)))
    assert abs(area.sum() / cap - 1) < 1e-12
    assert np.abs(np.linalg.norm(pos - np.array([0, 0, 64e-3]), axis=1) - 64e-3).max() < 1e-12


def test_oracle_on_axis_field_of_a_piston():
    """Textbook closed form: on the axis of a baffled circular piston of radius a and uniform
    velocity u, |P(z)| = 2 rho c u |sin(k/2 (sqrt(z^2 + a^2) - z))|, and the phase follows
    P = rho c u (e^{-jkz} - e^{-jk sqrt(z^2+a^2)})."""
    a, u = 10e-3, 0.02
    z = np.linspace(5e-3, 80e-3, 31)
    rcv = np.stack([np.zeros_like(z), np.zeros_like(z), z], axis=1)
    ref = RHO * C0 * u * (np.exp(-1j * K * z) - np.exp(-1j * K * np.sqrt(z * z + a * a)))
    err = []
    for h in (LAM / 8, LAM / 16):                                # the midpoint rule converges as h^2
        pos, area = wl.disc_elements(a, h)
        p = rs.rayleigh(pos, u * area, rcv, F, C0, RHO)
        err.append(np.abs(p - ref).max() / np.abs(ref).max())
    assert err[1] < 4e-3 and 3.0 < err[0] / err[1] < 5.0
    assert np.abs(np.abs(ref) - 2 * RHO * C0 * u * np.abs(np.sin(0.5 * K * (np.sqrt(z * z + a * a) - z)))).max() < 1e-9


def test_oracle_far_field_of_a_point_source_and_linearity():
    src = np.array([[0.0, 0.0, 0.0]])
    rcv = np.array([[0.03, 0.04, 0.12]])
    W = 1e-6 * (0.3 - 0.4j)
    R = 0.13
    p = rs.rayleigh(src, [W], rcv, F, C0, RHO)[0]
    assert abs(p - 1j * RHO * C0 * K / (2 * math.pi) * W * np.exp(-1j * K * R) / R) < 1e-12 * abs(p)
    rng = np.random.Generator(np.random.PCG64(3))
    s2 = rng.random((7, 3)) * 1e-2
    w2 = rng.standard_normal(7) + 1j * rng.standard_normal(7)
    both = rs.rayleigh(s2, w2, rcv, F)[0]
    parts = sum(rs.rayleigh(s2[i:i + 1], w2[i:i + 1], rcv, F)[0] for i in range(7))
    assert abs(both - parts) < 1e-12 * abs(both)


def test_oracle_bowl_focuses_at_the_centre_of_curvature():
    """Every element of a spherical cap is at distance R0 from the centre of curvature, so there
    P = (j rho c k / 2 pi) u A_cap e^{-j k R0} / R0 exactly, and the on-axis maximum lies near it."""
    R0, u = 64e-3, 0.01
    pos, area = wl.bowl_elements(64e-3, R0, LAM / 4)
    z = np.linspace(40e-3, 80e-3, 81)
    rcv = np.stack([np.zeros_like(z), np.zeros_like(z), z], axis=1)
    p = rs.rayleigh(pos, u * area, rcv, F, C0, RHO)
    foc = rs.rayleigh(pos, u * area, np.array([[0, 0, R0]]), F, C0, RHO)[0]
    ref = 1j * RHO * C0 * K / (2 * math.pi) * u * area.sum() * np.exp(-1j * K * R0) / R0
    assert abs(foc - ref) < 1e-10 * abs(ref)
    assert abs(z[np.argmax(np.abs(p))] - R0) < 4e-3


def test_cw_source_convention():
    p = np.array([2.0 * np.exp(1j * 0.7), -1.5j, 3.0])
    amp, d = rs.cw_source(p, F)
    t = np.linspace(0, 3 / F, 50)
    for n in range(3):
        assert np.abs(np.real(p[n] * np.exp(2j * math.pi * F * t)) - amp[n] * np.sin(2 * math.pi * F * (t - d[n]))).max() < 1e-9
        assert 0 <= d[n] < 1 / F


@pytest.mark.gpu
def test_gpu_rayleigh_matches_oracle():
    """The focused bowl of config 2 (aperture 64 mm, F# 1) decomposed at lambda/4 with seeded complex
    element weights, evaluated on a 41 x 37 patch of an entry plane 15 mm from the apex (several
    CTAs, a ragged tail and several source tiles)."""
    from paper_2301_12727_b200 import build as bv_build
    bv_build.build()
    from paper_2301_12727_b200 import binding as bv
    pos, area = wl.bowl_elements(64e-3, 64e-3, LAM / 4)
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 77))
    wgt = area * 0.01 * np.exp(2j * math.pi * rng.random(area.size)) * (0.5 + rng.random(area.size))
    xs = (np.arange(41) - 20) * (LAM / 9)
    ys = (np.arange(37) - 18) * (LAM / 9) + 1e-4
    X, Y = np.meshgrid(xs, ys)
    rcv = np.stack([X.ravel(), Y.ravel(), np.full(X.size, 15e-3)], axis=1)
    p, amp, delay = bv.rayleigh(pos, wgt, rcv, F, C0, RHO)
    ref = rs.rayleigh(pos.astype(np.float32), wgt.astype(np.complex64), rcv.astype(np.float32), F, C0, RHO)
    assert np.linalg.norm(p - ref) <= 1e-4 * np.linalg.norm(ref)
    ramp, rdelay = rs.cw_source(ref, F)
    big = ramp > 0.1 * ramp.max()
    assert np.abs(amp[big] / ramp[big] - 1).max() < 1e-3
    dd = np.abs(delay[big] - rdelay[big])
    dd = np.minimum(dd, 1 / F - dd)                              # delays are equal modulo one period
    assert dd.max() * F < 2e-4
    # uniform weights: the focus value is the closed form of the cap
    p2 = bv.rayleigh(pos, 0.01 * area, np.array([[0.0, 0.0, 64e-3]]), F, C0, RHO, want_source=False)
    ref2 = 1j * RHO * C0 * K / (2 * math.pi) * 0.01 * area.sum() * np.exp(-1j * K * 64e-3) / 64e-3
    assert abs(p2[0] - ref2) < 2e-4 * abs(ref2)


def test_oracle_receiver_on_a_source_point_takes_the_other_sources():
    """reading: a pair with R = 0 is left out; the field there is the plain sum of the rest"""
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 78))
    pos = rng.random((7, 3)) * 1e-2
    wgt = rng.random(7) + 1j * rng.random(7)
    got = rs.rayleigh(pos, wgt, pos[[3]], F, C0, RHO)[0]
    rest = np.delete(np.arange(7), 3)
    want = rs.rayleigh(pos[rest], wgt[rest], pos[[3]], F, C0, RHO)[0]
    assert np.isfinite(got) and abs(got - want) <= 1e-14 * abs(want)


@pytest.mark.gpu
def test_gpu_rayleigh_receiver_on_a_source_point_and_mufu_probe():
    from paper_2301_12727_b200 import build as bv_build
    bv_build.build()
    from paper_2301_12727_b200 import binding as bv
    pos, area = wl.disc_elements(5e-3, LAM / 4)
    rcv = np.concatenate([pos[[0, 17]], [[0.0, 0.0, 4e-3]]], axis=0)      # two receivers ON source points
    p, amp, delay = bv.rayleigh(pos, 0.01 * area, rcv, F, C0, RHO)
    ref = rs.rayleigh(pos.astype(np.float32), (0.01 * area).astype(np.complex64), rcv.astype(np.float32), F, C0, RHO)
    assert np.isfinite(p).all() and np.isfinite(amp).all() and np.isfinite(delay).all()
    assert np.abs(p - ref).max() <= 2e-4 * np.abs(ref).max()
    # the measured MUFU rate that k_rayleigh's roofline uses: at least one lane per scheduler, at most 32 per SM
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    rate = bv.probe_mufu()
    assert 4 * sms * 1e9 < rate < 32 * sms * 2.2e9, rate
