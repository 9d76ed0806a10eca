"""fp64 CPU ORACLE for the reductions that follow the FDTD run.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/`` (and the bench/smoke oracle legs) may import
this module; it shares no code with ``paper_2301_12727_b200``.

PAPER.md:L107-L110 (Eq. 2): after the tissue run and a water-only run on the same grid (L95),

    E_L = sum_xy I_PA-brain(x, y, z_m) / sum_xy I_PA-water(x, y, z_m),

"where I_PA is the intensity peak average.  E_L is calculated over the plane at a distance z_m where
water conditions show the maximal intensity"; L164: "A pressure transmission coefficient T_S was
calculated with T_S = sqrt(E_L)".

Readings (the paper does not define I_PA for a cell):
  * I_PA(cell) = p_amp^2 / (2 rho c_L), the plane-wave pulse-average intensity of a harmonic field of
    pressure amplitude p_amp = rms_amp = sqrt(2 sumsq / count) (reading P8), with rho, c_L the table
    values of the cell's own material: I_PA = sumsq / (count rho c_L).
  * sums and the maximum run over the cells outside the PML mask; z_m = the interior plane holding
    the largest water-run I_PA (first such plane on ties).
Everything below is the definition written out with numpy in fp64, no blocking or reordering.
"""
from __future__ import annotations

import numpy as np


def intensity_map(sumsq, count, table, index_map):
    """I_PA per cell (W/m^2), arrays shaped (nz, ny, nx)."""
    t = np.asarray(table, dtype=np.float64)
    z = t[:, 0] * t[:, 1]                                  # rho * c_L per material
    if count <= 0:
        return np.zeros(np.shape(sumsq))
    return np.asarray(sumsq, dtype=np.float64) / (float(count) * z[np.asarray(index_map)])


def plane_reductions(sumsq, count, table, index_map, pml):
    """(plane_sum, plane_max) over the interior cells of every z plane; PML planes give 0."""
    I = intensity_map(sumsq, count, table, index_map)
    nz, ny, nx = I.shape
    s = np.zeros(nz)
    m = np.zeros(nz)
    P = int(pml)
    for k in range(P, nz - P):
        inner = I[k, P:ny - P, P:nx - P]
        s[k] = inner.sum()
        m[k] = inner.max()
    return s, m


def energy_loss(sum_tissue, sum_water, max_water, pml):
    """z_m, E_L (Eq. 2) and T_S = sqrt(E_L) (L164) from the plane reductions of the two runs."""
    P = int(pml)
    nz = len(sum_water)
    k = P + int(np.argmax(np.asarray(max_water)[P:nz - P]))
    EL = float(sum_tissue[k]) / float(sum_water[k])
    return k, EL, float(np.sqrt(EL))
