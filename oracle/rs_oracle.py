"""fp64 CPU ORACLE for the Rayleigh-Sommerfeld source-plane field.

TEST INFRASTRUCTURE, NOT THE PRODUCT (only ``tests/`` and the oracle legs of bench/smoke import it; no
code shared with ``paper_2301_12727_b200``).

PAPER.md:L95: the transducer is decomposed into surface elements of area lambda^2/16 and "the acoustic
field is first calculated with a GPU-accelerated implementation of the Rayleigh-Sommerfeld equation
[45] over the incident interface of the simulation domain, with the coupling medium modeled as water".
The paper prints no formula; reading: first Rayleigh integral of a baffled
source, e^{+j w t} convention,

    P(r) = (j rho0 c0 k / 2 pi) sum_s W_s exp(-j k R_s) / R_s,   R_s = |r - r_s|,  k = 2 pi f / c0,

with W_s = u_s A_s.  The function below is that double sum written out (one receiver at a time, numpy
over the sources, fp64), nothing else.  A receiver that coincides with a source point (R_s = 0) takes the sum
over the OTHER source points: the point-element term has no finite value there (reading).
"""
from __future__ import annotations

import numpy as np


def rayleigh(src_xyz, src_weight, rcv_xyz, f, c0=1500.0, rho0=1000.0):
    s = np.asarray(src_xyz, dtype=np.float64)
    w = np.asarray(src_weight, dtype=np.complex128)
    r = np.asarray(rcv_xyz, dtype=np.float64)
    k = 2.0 * np.pi * f / c0
    out = np.zeros(r.shape[0], dtype=np.complex128)
    for n in range(r.shape[0]):
        R = np.sqrt(((r[n] - s) ** 2).sum(axis=1))
        ok = R > 0.0
        out[n] = (w[ok] * np.exp(-1j * k * R[ok]) / R[ok]).sum()
    return 1j * rho0 * c0 * k / (2.0 * np.pi) * out


def cw_source(p, f):
    """(amp, delay) with p(t) = Re{P e^{j w t}} = amp sin(w (t - delay)), delay in [0, 1/f)."""
    w = 2.0 * np.pi * f
    a = -(np.angle(p) + 0.5 * np.pi)
    a = a - 2.0 * np.pi * np.floor(a / (2.0 * np.pi))
    return np.abs(p), a / w
