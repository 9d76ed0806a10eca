"""fp64 CPU ORACLE for the thermal step.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/`` (and the bench/smoke oracle legs) may import
this module; it shares no code with ``paper_2301_12727_b200``.

PAPER.md:L99: "The thermal simulation step solves the Bio Heat Transfer Equation (BHTE) with a
finite-difference time-difference solver in Cartesian coordinates [46].  Boundary conditions are
assumed conservatively with a temperature of 37 C at the domain's borders.  The user specifies the
sonication regime ... duration of ultrasound, time off after ultrasound, and duty cycle ...  The
fraction of attenuation in skull bone transformed into heat was set to 0.16 ...  Safety metrics
... maximal temperature, and thermal dose [48]".

The paper prints neither the equation nor its discretisation, so everything below is a READING
("parity unpinned vs paper"; the oracle itself is pinned by closed forms of
the discretised model in tests/test_bhte.py):

  Pennes:   rho C dT/dt = div(k grad T) - w (T - T_b) + s(t) Q
  * per-material constants: k (W/m/K), rho C (J/m^3/K), w = perfusion coefficient
    w_b rho_b C_b (W/m^3/K); arterial temperature T_b = border temperature (37 C, L99);
  * forward Euler in time, conservative 7-point stencil on the cell grid of the acoustic run;
    the conductivity of the face between two cells is the series (harmonic) mean
    k_f = 2 k_a k_b / (k_a + k_b) (two half cells in series: the composite-wall resistance);
  * cells on the six borders of the box are held at T_b (Dirichlet, L99);
  * s(t) = `heat_scale` of the step: the duty cycle while the ultrasound is on, 0 while off
    (L99 "duration of ultrasound, time off after ultrasound, and duty cycle");
  * thermal dose [48] (Sapareto-Dewey cumulative equivalent minutes at 43 C), accumulated with the
    temperature reached at the end of each step:  CEM43 += (dt / 60) R^(43 - T),
    R = 0.5 for T >= 43, 0.25 below;  running maximum temperature likewise;
  * heat deposition of a harmonic field of pressure amplitude p_amp in a medium (rho, c_L, alpha):
    plane-wave intensity I = p_amp^2 / (2 rho c_L), absorbed power density Q = 2 a alpha I with
    a = the absorbed fraction of the attenuation (0.16 in bone, L99; 1 in soft tissue).

Everything is the definition written out with numpy slices in fp64, no blocking or reordering.
Arrays are shaped (nz, ny, nx).
"""
from __future__ import annotations

import numpy as np


def face_conductivity(ka, kb):
    """Series mean of the two half cells either side of a face."""
    return 2.0 * ka * kb / (ka + kb)


class BhteOracle:
    """table: rows (k, rho_C, perf); index_map: uint8 (nz, ny, nx)."""

    def __init__(self, table, index_map, dx, dt, T_b=37.0):
        t = np.asarray(table, dtype=np.float64)
        idx = np.asarray(index_map)
        self.k = t[:, 0][idx]
        self.rho_c = t[:, 1][idx]
        self.perf = t[:, 2][idx]
        self.dx, self.dt, self.T_b = float(dx), float(dt), float(T_b)
        self.T = np.full(idx.shape, self.T_b)
        self.dose = np.zeros(idx.shape)
        self.tmax = np.full(idx.shape, self.T_b)
        self.Q = np.zeros(idx.shape)

    def set_heat(self, Q):
        self.Q = np.asarray(Q, dtype=np.float64).copy()

    def set_temperature(self, T):
        """Initial condition; the border cells are held at T_b whatever is passed."""
        self.T = np.asarray(T, dtype=np.float64).copy()
        self._hold_border(self.T)
        self.tmax = np.maximum(self.tmax, self.T)

    def _hold_border(self, T):
        T[0, :, :] = T[-1, :, :] = self.T_b
        T[:, 0, :] = T[:, -1, :] = self.T_b
        T[:, :, 0] = T[:, :, -1] = self.T_b

    def step(self, n, heat_scale):
        k, T_b, dx, dt = self.k, self.T_b, self.dx, self.dt
        c = (slice(1, -1),) * 3                      # the interior cells
        for _ in range(int(n)):
            T = self.T
            div = np.zeros_like(T)
            for axis in range(3):
                lo = [slice(1, -1)] * 3
                hi = [slice(1, -1)] * 3
                lo[axis] = slice(0, -2)
                hi[axis] = slice(2, None)
                lo, hi = tuple(lo), tuple(hi)
                div[c] += face_conductivity(k[c], k[hi]) * (T[hi] - T[c]) / dx ** 2
                div[c] += face_conductivity(k[c], k[lo]) * (T[lo] - T[c]) / dx ** 2
            Tn = T.copy()
            Tn[c] = T[c] + dt / self.rho_c[c] * (div[c] - self.perf[c] * (T[c] - T_b) + heat_scale * self.Q[c])
            self._hold_border(Tn)
            R = np.where(Tn >= 43.0, 0.5, 0.25)
            self.dose += dt / 60.0 * R ** (43.0 - Tn)
            self.tmax = np.maximum(self.tmax, Tn)
            self.T = Tn


def heat_source(p_amp, table_acoustic, absorbed_fraction, index_map, scale=1.0):
    """Q = scale * a * 2 alpha_L * p_amp^2 / (2 rho c_L) per cell (W/m^3); table rows are the acoustic
    material rows (rho, cL, cS, alphaL, alphaS), absorbed_fraction one value per material."""
    t = np.asarray(table_acoustic, dtype=np.float64)
    idx = np.asarray(index_map)
    rho, cL, aL = t[:, 0][idx], t[:, 1][idx], t[:, 3][idx]
    a = np.asarray(absorbed_fraction, dtype=np.float64)[idx]
    I = np.asarray(p_amp, dtype=np.float64) ** 2 / (2.0 * rho * cL)
    return scale * a * 2.0 * aL * I


def max_stable_dt(table, dx):
    """Forward-Euler bound of the 7-point stencil with perfusion: dt (6 k / dx^2 + w) / (rho C) <= 1
    for every material (a face mean never exceeds the larger of its two cells' k)."""
    t = np.asarray(table, dtype=np.float64)
    kmax = t[:, 0].max()
    return float(np.min(t[:, 1] / (6.0 * kmax / dx ** 2 + t[:, 2])))
