"""fp64 CPU ORACLE for the corrected phase programming of a phased array (SURVEY.md 8(f) NEXT-3,
second half: "point-source back-propagation for phased-array refocusing").

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/`` may import this module; it shares no code with
``paper_2301_12727_b200``.

PAPER.md:L95: "if refocusing is requested, a punctual source is placed at the intended target,
back-propagated to the domain interface, and then propagated back with Rayleigh-Sommerfeld to the
transducer elements to calculate the corrected phase programming of the transducer elements.
Finally, the forward propagated field is calculated."

The paper gives no formula; readings:
  * the FDTD run from the point source yields the phasor P (p(t) = Re{P e^{jwt}}) on the entry
    plane; that plane radiates back to the transducer as a baffled source whose weight is
    proportional to P (u = P / (rho0 c0) times the cell area: a common positive factor, which the
    normalisation below removes), through the Rayleigh sum of ``rs_oracle.rayleigh``;
  * E_m = sum of that field over the surface points of element m;
  * time reversal: element m emits Re{conj(E_m)/|E_m| e^{jwt}}: unit amplitude, phase -arg E_m, i.e.
    cos(w (t - tau_m)) with tau_m = arg(E_m) / w taken in [0, 1/f);
  * every surface point of element m carries the weight u0 * area * conj(E_m)/|E_m|.
The functions below are these definitions written out with numpy in fp64.
"""
from __future__ import annotations

import numpy as np


def element_sums(P, element, n_elem):
    """E_m = sum of P over the points whose element index is m (plain loop over the elements)."""
    P = np.asarray(P, dtype=np.complex128)
    element = np.asarray(element)
    return np.array([P[element == m].sum() for m in range(n_elem)], dtype=np.complex128)


def phase_programming(E, f):
    """(unit weights conj(E)/|E|, delays arg(E)/w in [0, 1/f))."""
    E = np.asarray(E, dtype=np.complex128)
    w = 2.0 * np.pi * f
    phi = np.angle(E)
    phi = phi - 2.0 * np.pi * np.floor(phi / (2.0 * np.pi))
    return np.conj(E) / np.abs(E), phi / w


def point_weights(E, element, area, u0=1.0):
    """Complex weight u0 * area * conj(E_m)/|E_m| of every surface point."""
    unit, _ = phase_programming(E, 1.0)
    return u0 * np.asarray(area, dtype=np.float64) * unit[np.asarray(element)]
