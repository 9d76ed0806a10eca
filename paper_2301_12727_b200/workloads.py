"""Seeded synthetic workloads for the viscoelastic FDTD step (numpy only).

This module is the ONLY code shared by the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2301_12727_b200/csrc``).  It holds none of the method's arithmetic: it builds
inputs only -- the uint8 material index map, the material table (rho, cL, cS, alphaL,
alphaS), the source cell list (cell, amplitude, delay), the time step and the sensor
windows -- for the five configurations of ``BASELINE.json:configs`` as made concrete in
SURVEY.md section 8(d) and restated in DESIGN.md ("Input recipe").

The paper's own workloads are patient CT/MRI datasets that are not available
(PAPER.md:L128); these synthetic domains take their shapes, sizes and value ranges
(three-layer skull 10/80/10; Table 1 property ranges, PAPER.md:L65-L73;
6-9 PPW grids, L57/L148; focused apertures at F# ~ 1, L35/L146) and stand in for them.

Conventions: node (i, j, k) sits at (x, y, z) = (i, j, k) * dx, the linear cell index is
``i + nx * (j + ny * k)`` (x fastest, z = acoustic axis); numpy arrays are
shaped (nz, ny, nx).  RNG: ``numpy.random.Generator(PCG64(230112727 + cfg))``; random
fields are drawn plane by plane along z (identical stream to one (nz, ny, nx) draw).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

WATER = (1000.0, 1500.0, 0.0, 0.0, 0.0)
SEED_BASE = 230112727
CFL = 0.3


@dataclass
class Workload:
    """Everything ``bvfdtd_create`` / ``bvfdtd_set_source`` (and the oracle) need."""

    name: str
    nx: int
    ny: int
    nz: int
    pml: int
    dx: float
    dt: float
    f0: float
    spp: int                       # time steps per source period (integer by construction)
    steps: int
    table: np.ndarray              # (n_mat, 5) float64: rho, cL, cS, alphaL, alphaS (Np/m at f0)
    index_map: np.ndarray          # (nz, ny, nx) uint8
    src_cell: np.ndarray           # (n_src,) int64 linear cell indices
    src_amp: np.ndarray            # (n_src,) float32
    src_delay: np.ndarray          # (n_src,) float32 seconds
    waveform: int                  # 0 = burst, 1 = ramped CW
    f_src: float
    n_cycles: int
    peak_begin: int = 0
    rms_begin: int = -1            # < 0: no rms window (set to `steps`, i.e. empty)
    sensor_end: int = -1           # < 0: unbounded
    pml_R: float = 1e-4
    notes: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    def mean_mask_bits(self) -> float:
        p = self.pml
        return 2.0 * p / self.nx + 2.0 * p / self.ny + 2.0 * p / self.nz

    def bytes_per_cell_step(self, rms_on: bool = False) -> float:
        """Algorithmic bytes per cell-step, B_dense of SURVEY.md 8(d): 49 (S2) + 109 (S3)
        + 8 (peak) + 8 (sumsq, when on) + 48 per PML mask bit set."""
        return 49.0 + 109.0 + 8.0 + (8.0 if rms_on else 0.0) + 48.0 * self.mean_mask_bits()


def _min_bytes(self, rms_frac: float = 0.0) -> float:
    """Class-aware minimum B_min of SURVEY.md 8(d) per cell-step: a fluid cell moves no shear stress
    and no shear memory variable (-60 B), a lossless cell no memory variable at all (-48 B in
    total), and in a lossy FLUID cell the three normal memory variables are one and the same number
    (eS = bS = 0: one recursion from the same zero start), so only one of them must move (-16 B):
    and its three normal stresses are one number too (the pressure), so the velocity pass needs to
    read only one of them (-8 B; the stress pass still updates all three):
    fluid-lossless 74 B, fluid-lossy 82 B (SURVEY.md prints 82 / 114 with three of each),
    solid-lossless 118 B, solid-lossy 166 B, plus
    48 B per PML mask bit and 8 B per cell while the rms window is open.  Accounting only."""
    t = self.table
    solid = t[:, 2] > 0
    lossy = (t[:, 3] > 0) | ((t[:, 4] > 0) & solid)
    per_mat = np.where(solid, np.where(lossy, 166.0, 118.0), np.where(lossy, 82.0, 74.0))
    counts = np.bincount(self.index_map.ravel(), minlength=t.shape[0]).astype(np.float64)
    base = float((per_mat * counts).sum() / counts.sum())
    return base + 48.0 * self.mean_mask_bits() + 8.0 * rms_frac


Workload.min_bytes_per_cell_step = _min_bytes


def snapped_dt(dx: float, f0: float, c_max: float, cfl: float = CFL):
    """Reading P6: dt0 = CFL dx / c_max, snapped so that one period is a whole number of
    steps.  Returns (dt, steps_per_period)."""
    dt0 = cfl * dx / c_max
    spp = int(math.ceil(1.0 / (f0 * dt0) - 1e-9))
    return 1.0 / (f0 * spp), spp


def bone_shear_speed(cL):
    """cS = 0.55 cL where cL >= 1800 m/s, else 0 (chosen)."""
    cL = np.asarray(cL, dtype=np.float64)
    return np.where(cL >= 1800.0, 0.55 * cL, 0.0)


def _disc_cells(nx, ny, k_s, radius_cells, xc, yc):
    j, i = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    m = (i - xc) ** 2 + (j - yc) ** 2 <= radius_cells ** 2
    return (i[m] + nx * (j[m] + ny * k_s)).astype(np.int64), i[m], j[m]


# ----------------------------------------------------------------------------------------
# config 0: water + flat cortical plate, piston burst
# ----------------------------------------------------------------------------------------
def config0() -> Workload:
    nx = ny = nz = 64
    P = 8
    dx = 1e-3 / 3.0
    f0 = 500e3
    table = np.array([WATER, (1900.0, 2800.0, 1500.0, 200.0, 200.0)], dtype=np.float64)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    idx = np.zeros((nz, ny, nx), dtype=np.uint8)
    idx[29:35] = 1
    cells, _, _ = _disc_cells(nx, ny, 12, 10.0, 31.5, 31.5)
    n = cells.size
    return Workload("cfg0_plate64", nx, ny, nz, P, dx, dt, f0, spp, 300, table, idx,
                    cells, np.ones(n, np.float32), np.zeros(n, np.float32),
                    waveform=0, f_src=f0, n_cycles=3, peak_begin=0, rms_begin=-1)


# ----------------------------------------------------------------------------------------
# config 1: spherical shell with 64 HU-like materials, CW piston
# ----------------------------------------------------------------------------------------
def config1(steps: int = 800) -> Workload:
    nx = ny = nz = 128
    P = 12
    dx = 1e-3 / 3.0
    f0 = 500e3
    fm = f0 / 1e6
    t = np.arange(64) / 63.0
    cL = 1500.0 + 1600.0 * t
    rows = [WATER] + [
        (1000.0 + 1100.0 * t[e], cL[e], float(bone_shear_speed(cL[e])), 163.0 * fm * t[e],
         (329.0 * fm * t[e]) if cL[e] >= 1800.0 else 0.0)
        for e in range(64)
    ]
    table = np.array(rows, dtype=np.float64)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1))
    idx = np.zeros((nz, ny, nx), dtype=np.uint8)
    jj, ii = np.meshgrid(np.arange(ny) - 63.5, np.arange(nx) - 63.5, indexing="ij")
    for k in range(nz):
        g = rng.standard_normal((ny, nx))
        hu = np.clip(1200.0 + 300.0 * g, 200.0, 2200.0)
        e = np.minimum(63, np.floor((hu - 200.0) * 64.0 / 2000.0)).astype(np.int64)
        r = np.sqrt(ii ** 2 + jj ** 2 + (k - 63.5) ** 2)
        shell = (r > 19.0) & (r <= 40.0)
        idx[k] = np.where(shell, 1 + e, 0).astype(np.uint8)
    cells, _, _ = _disc_cells(nx, ny, 16, 20.0, 63.5, 63.5)
    n = cells.size
    return Workload("cfg1_shell128", nx, ny, nz, P, dx, dt, f0, spp, steps, table, idx,
                    cells, np.ones(n, np.float32), np.zeros(n, np.float32),
                    waveform=1, f_src=f0, n_cycles=3, peak_begin=0,
                    rms_begin=max(0, steps - 3 * spp))


# ----------------------------------------------------------------------------------------
# configs 2-4: layered ellipsoidal skull + brain
# ----------------------------------------------------------------------------------------
def _skull_table(n_rows: int, f0: float) -> np.ndarray:
    """water; brain; nb = n_rows - 2 bone entries indexed by porosity (0 .. 0.5)."""
    fm = f0 / 1e6
    nb = n_rows - 2
    phi = 0.5 * np.arange(nb) / (nb - 1)
    rho = 1000.0 * phi + 2100.0 * (1.0 - phi)
    cL = 1500.0 * phi + 3100.0 * (1.0 - phi)
    cS = bone_shear_speed(cL)
    rows = [WATER, (1040.0, 1546.0, 0.0, 60.0 * fm, 0.0)]
    rows += [(rho[e], cL[e], cS[e], 163.0 * fm, 329.0 * fm if cS[e] > 0 else 0.0)
             for e in range(nb)]
    return np.array(rows, dtype=np.float64)


def _layered_skull_map(nx, ny, nz, dx, zc_mm, outer_mm, thick_mm, nb, rng, thick_sd_mm=0.0):
    """Material ids: 0 water, 1 brain, 2 + e bone entry e (porosity phi = 0.5 e / (nb-1)).

    Ellipsoid centred (x_c, y_c, zc); outer semi-axes `outer_mm`, inner = outer - T with
    T = thick_mm (+ clip(G, -3, 3) * thick_sd_mm per voxel when thick_sd_mm > 0, config 4).
    Depth fraction u = (1 - s_out) / ((1 - s_out) + (s_in - 1)); cortical if u < 0.1 or
    u >= 0.9 else trabecular (10/80/10).  Porosity: 0.1 U (cortical),
    0.1 + 0.4 U (trabecular), U = random().  Draw order per z-plane: all G planes first
    (config 4 only), then all U planes, each as one pass over z.
    """
    idx = np.zeros((nz, ny, nx), dtype=np.uint8)
    xmm = (np.arange(nx) - (nx - 1) / 2.0) * dx * 1e3
    ymm = (np.arange(ny) - (ny - 1) / 2.0) * dx * 1e3
    Y, X = np.meshgrid(ymm, xmm, indexing="ij")
    ax, ay, az = outer_mm
    gs = None
    if thick_sd_mm > 0.0:
        gs = np.empty((nz, ny, nx), dtype=np.float32)  # kept as the float32 cast of the draw
        for k in range(nz):
            gs[k] = rng.standard_normal((ny, nx)).astype(np.float32)
    for k in range(nz):
        zmm = k * dx * 1e3 - zc_mm
        U = rng.random((ny, nx))
        s_out = np.sqrt((X / ax) ** 2 + (Y / ay) ** 2 + (zmm / az) ** 2)
        if gs is None:
            T = thick_mm
        else:
            T = thick_mm + np.clip(gs[k].astype(np.float64), -3.0, 3.0) * thick_sd_mm
        s_in = np.sqrt((X / (ax - T)) ** 2 + (Y / (ay - T)) ** 2 + (zmm / (az - T)) ** 2)
        water = s_out > 1.0
        brain = s_in <= 1.0
        skull = ~(water | brain)
        with np.errstate(divide="ignore", invalid="ignore"):
            u = (1.0 - s_out) / ((1.0 - s_out) + (s_in - 1.0))
        cortical = (u < 0.1) | (u >= 0.9)
        phi = np.where(cortical, 0.1 * U, 0.1 + 0.4 * U)
        e = np.rint(phi / 0.5 * (nb - 1)).astype(np.int64)
        plane = np.where(brain, 1, 0)
        plane = np.where(skull, 2 + e, plane)
        idx[k] = plane.astype(np.uint8)
    return idx


def _focused_aperture(nx, ny, k_s, dx, radius_mm, focal_mm):
    """Focused bowl projected on plane k_s (stand-in for the Rayleigh-Sommerfeld step,
    PAPER.md:L95): amp = F / d, delay = (d_max - d) / 1500 with d the distance to the focus."""
    xc, yc = (nx - 1) / 2.0, (ny - 1) / 2.0
    cells, i, j = _disc_cells(nx, ny, k_s, radius_mm * 1e-3 / dx, xc, yc)
    rho_mm = np.sqrt((i - xc) ** 2 + (j - yc) ** 2) * dx * 1e3
    d = np.sqrt(rho_mm ** 2 + focal_mm ** 2)
    d_max = math.sqrt(radius_mm ** 2 + focal_mm ** 2)
    amp = (focal_mm / d).astype(np.float32)
    delay = ((d_max - d) * 1e-3 / 1500.0).astype(np.float32)
    return cells, amp, delay


def config2(steps: int = 3000) -> Workload:
    nx, ny, nz, P = 300, 300, 450, 16
    dx = 1e-3 / 3.0
    f0 = 500e3
    table = _skull_table(128, f0)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    k_s = P + 4
    zc_mm = k_s * dx * 1e3 + 10.0 + 95.0
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 2))
    idx = _layered_skull_map(nx, ny, nz, dx, zc_mm, (85.0, 70.0, 95.0), 7.0, 126, rng)
    cells, amp, delay = _focused_aperture(nx, ny, k_s, dx, 32.0, 60.0)
    return Workload("cfg2_skull300x300x450", nx, ny, nz, P, dx, dt, f0, spp, steps, table, idx,
                    cells, amp, delay, waveform=1, f_src=f0, n_cycles=3, peak_begin=0,
                    rms_begin=max(0, steps - 3 * spp))


def config3(steps: int = 5000) -> Workload:
    nx, ny, nz, P = 504, 504, 672, 20
    f0 = 700e3
    dx = 1500.0 / (f0 * 9.0)
    table = _skull_table(255, f0)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    k_s = P + 4
    zc_mm = k_s * dx * 1e3 + 10.0 + 95.0
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 3))
    idx = _layered_skull_map(nx, ny, nz, dx, zc_mm, (85.0, 70.0, 95.0), 7.0, 253, rng)
    cells, amp, delay = _focused_aperture(nx, ny, k_s, dx, 32.0, 60.0)
    return Workload("cfg3_skull504x504x672", nx, ny, nz, P, dx, dt, f0, spp, steps, table, idx,
                    cells, amp, delay, waveform=1, f_src=f0, n_cycles=3, peak_begin=0,
                    rms_begin=max(0, steps - 3 * spp))


def config4(steps: int = 6000) -> Workload:
    nx, ny, nz, P = 480, 480, 600, 24
    dx = 0.25e-3
    f0 = 250e3
    table = _skull_table(128, f0)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    k_s = P + 4
    z_cap_mm = k_s * dx * 1e3
    zc_mm = z_cap_mm + 30.0 + 95.0
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 4))
    idx = _layered_skull_map(nx, ny, nz, dx, zc_mm, (85.0, 70.0, 95.0), 7.0, 126, rng,
                             thick_sd_mm=1.0)
    # 128-element array on a spherical cap (radius of curvature 80 mm, aperture 100 mm),
    # apex (x_c, y_c, z_cap), concave toward +z; sunflower lattice of element centres.
    u0 = rng.random()
    n_el = 128
    Rc = 80.0
    th_max = math.asin(50.0 / Rc)
    m = np.arange(n_el)
    th = np.arccos(1.0 - (m + 0.5) / n_el * (1.0 - math.cos(th_max)))
    ph = m * math.pi * (3.0 - math.sqrt(5.0)) + 2.0 * math.pi * u0
    xc_mm = (nx - 1) / 2.0 * dx * 1e3
    yc_mm = (ny - 1) / 2.0 * dx * 1e3
    centre = np.array([xc_mm, yc_mm, z_cap_mm + Rc])          # centre of curvature
    el = np.stack([centre[0] + Rc * np.sin(th) * np.cos(ph),
                   centre[1] + Rc * np.sin(th) * np.sin(ph),
                   centre[2] - Rc * np.cos(th)], axis=1)     # (128, 3) mm
    target = np.array([xc_mm + 10.0, yc_mm, centre[2]])       # geometric focus + 10 mm in x
    d_el = np.linalg.norm(el - target, axis=1)
    jitter = rng.standard_normal(n_el) * (1.0 / f0) / 50.0
    delay_el = (d_el.max() - d_el) * 1e-3 / 1500.0 + jitter
    delay_el -= delay_el.min()
    # voxels of the cap: |dist to centre of curvature - Rc| <= dx/2 and within 3.5 mm of
    # the nearest element centre.  Only planes the cap can reach are scanned.
    sag_mm = Rc - math.sqrt(Rc ** 2 - 50.0 ** 2)
    k_hi = int(math.ceil((z_cap_mm + sag_mm + 4.0) / (dx * 1e3)))
    xs = np.arange(nx) * dx * 1e3
    ys = np.arange(ny) * dx * 1e3
    Y, X = np.meshgrid(ys, xs, indexing="ij")
    cells_l, delay_l = [], []
    for k in range(max(P, k_s - 2), min(nz - P, k_hi + 1)):
        z = k * dx * 1e3
        dist = np.sqrt((X - centre[0]) ** 2 + (Y - centre[1]) ** 2 + (z - centre[2]) ** 2)
        on = np.abs(dist - Rc) <= dx * 1e3 / 2.0
        on &= (np.arange(ny)[:, None] >= P) & (np.arange(ny)[:, None] < ny - P)
        on &= (np.arange(nx)[None, :] >= P) & (np.arange(nx)[None, :] < nx - P)
        if not on.any():
            continue
        jj, ii = np.nonzero(on)
        pts = np.stack([xs[ii], ys[jj], np.full(ii.size, z)], axis=1)
        d2 = ((pts[:, None, :] - el[None, :, :]) ** 2).sum(axis=2)
        near = d2.argmin(axis=1)
        ok = d2[np.arange(ii.size), near] <= 3.5 ** 2
        cells_l.append((ii[ok] + nx * (jj[ok] + ny * k)).astype(np.int64))
        delay_l.append(delay_el[near[ok]])
    cells = np.concatenate(cells_l)
    delay = np.concatenate(delay_l).astype(np.float32)
    order = np.argsort(cells, kind="stable")
    cells, delay = cells[order], delay[order]
    return Workload("cfg4_array480x480x600", nx, ny, nz, P, dx, dt, f0, spp, steps, table, idx,
                    cells, np.ones(cells.size, np.float32), delay, waveform=1, f_src=f0,
                    n_cycles=3, peak_begin=0, rms_begin=-1)


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def make(cfg: int, **kw) -> Workload:
    return CONFIGS[cfg](**kw)


# ----------------------------------------------------------------------------------------
# small seeded domains for unit / edge-case parity tests
# ----------------------------------------------------------------------------------------
def random_domain(nx, ny, nz, pml, seed, n_mat=6, solid_fraction=0.5, lossy=True,
                  f0=500e3, dx=1e-3 / 3.0, steps=20, waveform=0) -> Workload:
    """A small heterogeneous fluid + solid block map for kernel-level parity tests.

    Blocks of 3x3x3 voxels get a random material so that every averaging case (fluid-fluid,
    fluid-solid, solid-solid, lossy/lossless) appears next to every kind of node."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1000 + seed))
    rows = [WATER]
    for m in range(1, n_mat):
        solid = rng.random() < solid_fraction
        rho = 1000.0 + 1100.0 * rng.random()
        cL = 1500.0 + 1600.0 * rng.random()
        cS = (0.45 + 0.1 * rng.random()) * cL if solid else 0.0
        aL = 200.0 * rng.random() if lossy else 0.0
        aS = 300.0 * rng.random() if (lossy and solid) else 0.0
        rows.append((rho, cL, cS, aL, aS))
    table = np.array(rows, dtype=np.float64)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    bz, by, bx = (nz + 2) // 3, (ny + 2) // 3, (nx + 2) // 3
    blocks = rng.integers(0, n_mat, size=(bz, by, bx), dtype=np.int64)
    idx = np.repeat(np.repeat(np.repeat(blocks, 3, 0), 3, 1), 3, 2)[:nz, :ny, :nx]
    idx = np.ascontiguousarray(idx).astype(np.uint8)
    # sources: a few cells in the interior (outside the PML mask)
    lo = pml
    ci = rng.integers(lo, nx - lo, size=5)
    cj = rng.integers(lo, ny - lo, size=5)
    ck = rng.integers(lo, nz - lo, size=5)
    cells = np.unique((ci + nx * (cj + ny * ck)).astype(np.int64))
    amp = (0.5 + rng.random(cells.size)).astype(np.float32)
    delay = (rng.random(cells.size) * 2.0 / f0 * 0.25).astype(np.float32)
    return Workload(f"rand_{nx}x{ny}x{nz}_p{pml}_s{seed}", nx, ny, nz, pml, dx, dt, f0, spp,
                    steps, table, idx, cells, amp, delay, waveform=waveform, f_src=f0,
                    n_cycles=3, peak_begin=0, rms_begin=max(0, steps // 2))


def blocky_domain(nx, ny, nz, pml, seed, steps=20, waveform=1, f0=500e3, dx=1e-3 / 3.0) -> Workload:
    """Mostly lossless water with a few box-shaped inclusions (lossy solids, one lossy fluid, one
    lossless solid) whose faces are not aligned with the 64 x 8 tiles and of which one runs into
    the PML slabs: the layout that exercises the tile-class skipping of the tiled kernels
    (all-fluid tile-planes next to partly solid ones, lossless next to lossy)."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 3000 + seed))
    table = np.array([WATER,
                      (1900.0, 2800.0, 1500.0, 200.0, 200.0),     # lossy solid
                      (1040.0, 1546.0, 0.0, 30.0, 0.0),           # lossy fluid
                      (1700.0, 2500.0, 1300.0, 0.0, 0.0),         # lossless solid
                      (2100.0, 3100.0, 1700.0, 80.0, 160.0)], dtype=np.float64)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    idx = np.zeros((nz, ny, nx), dtype=np.uint8)
    dims = np.array([nz, ny, nx])
    for b in range(6):
        lo = np.array([rng.integers(0, max(1, d - 4)) for d in dims])
        ext = np.array([rng.integers(2, max(3, d // 2)) for d in dims])
        hi = np.minimum(dims, lo + ext)
        idx[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = 1 + b % 4
    idx[:, :3, :] = np.where(idx[:, :3, :] == 0, 4, idx[:, :3, :]) if seed % 2 else idx[:, :3, :]
    lo = pml
    ci = rng.integers(lo, nx - lo, size=6)
    cj = rng.integers(lo, ny - lo, size=6)
    ck = rng.integers(lo, nz - lo, size=6)
    cells = np.unique((ci + nx * (cj + ny * ck)).astype(np.int64))
    amp = (0.5 + rng.random(cells.size)).astype(np.float32)
    delay = (rng.random(cells.size) * 0.5 / f0).astype(np.float32)
    return Workload(f"blocky_{nx}x{ny}x{nz}_p{pml}_s{seed}", nx, ny, nz, pml, dx, dt, f0, spp,
                    steps, table, idx, cells, amp, delay, waveform=waveform, f_src=f0,
                    n_cycles=3, peak_begin=0, rms_begin=max(0, steps // 2))


def fluid_domain(nx, ny, nz, pml, seed, steps=40, waveform=1, f0=500e3, dx=1e-3 / 3.0, solid_boxes=2) -> Workload:
    """Mostly fluid: lossless water with blobs of three other fluids (two lossy, different densities and speeds)
    and a few solid boxes well inside the grid.  Most 64 x 8 tile columns have no solid cell within reach of
    their stencils over long z runs -- the layout on which the fused single sweep (kernels_fused.cuh) takes
    over from the two passes -- next to tile columns, and z ranges, that keep the two passes."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 5000 + seed))
    table = np.array([WATER,
                      (1040.0, 1546.0, 0.0, 30.0, 0.0),           # lossy fluid (brain-like)
                      (920.0, 1450.0, 0.0, 0.0, 0.0),             # lossless light fluid
                      (1100.0, 1600.0, 0.0, 60.0, 0.0),           # lossy heavy fluid
                      (1900.0, 2800.0, 1500.0, 200.0, 200.0),     # lossy solid
                      (1700.0, 2500.0, 1300.0, 0.0, 0.0)], dtype=np.float64)
    dt, spp = snapped_dt(dx, f0, table[:, 1].max())
    idx = np.zeros((nz, ny, nx), dtype=np.uint8)
    dims = np.array([nz, ny, nx])
    for b in range(8):
        lo = np.array([rng.integers(0, max(1, d - 4)) for d in dims])
        ext = np.array([rng.integers(3, max(4, d // 2)) for d in dims])
        hi = np.minimum(dims, lo + ext)
        idx[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = 1 + b % 3
    for b in range(solid_boxes):
        lo = np.array([rng.integers(d // 4, max(d // 4 + 1, d // 2)) for d in dims])
        ext = np.array([rng.integers(3, max(4, d // 5)) for d in dims])
        hi = np.minimum(dims, lo + ext)
        idx[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = 4 + b % 2
    lo = pml
    n = 10
    ci = rng.integers(lo, nx - lo, size=n)
    cj = rng.integers(lo, ny - lo, size=n)
    ck = rng.integers(lo, nz - lo, size=n)
    cells = np.unique((ci + nx * (cj + ny * ck)).astype(np.int64))
    amp = (0.5 + rng.random(cells.size)).astype(np.float32)
    delay = (rng.random(cells.size) * 0.5 / f0).astype(np.float32)
    return Workload(f"fluid_{nx}x{ny}x{nz}_p{pml}_s{seed}", nx, ny, nz, pml, dx, dt, f0, spp,
                    steps, table, idx, cells, amp, delay, waveform=waveform, f_src=f0,
                    n_cycles=3, peak_begin=0, rms_begin=max(0, steps // 2))


# ----------------------------------------------------------------------------------------
# transducer surface decompositions (inputs of the Rayleigh-Sommerfeld step)
# ----------------------------------------------------------------------------------------
def disc_elements(radius: float, h: float, z: float = 0.0):
    """A flat circular piston of the given radius in the plane z, cut into polar-ring elements of
    side ~h (the paper uses areas of lambda^2/16, i.e. h = lambda/4): positions (n,3) and areas (n,).
    The areas add up to pi radius^2 exactly."""
    n_r = max(1, int(round(radius / h)))
    dr = radius / n_r
    pos, area = [], []
    for i in range(n_r):
        r = (i + 0.5) * dr
        n_t = max(1, int(round(2.0 * math.pi * r / dr)))
        t = (np.arange(n_t) + 0.5) * (2.0 * math.pi / n_t)
        pos.append(np.stack([r * np.cos(t), r * np.sin(t), np.full(n_t, z)], axis=1))
        area.append(np.full(n_t, math.pi * ((r + 0.5 * dr) ** 2 - (r - 0.5 * dr) ** 2) / n_t))
    return np.concatenate(pos), np.concatenate(area)


def bowl_elements(aperture: float, focal: float, h: float):
    """A spherical-cap (focused bowl) radiator with its apex at the origin, axis +z and centre of
    curvature at (0, 0, focal), cut into rings of elements of side ~h: positions and areas (the
    areas add up to the cap area 2 pi focal^2 (1 - cos theta_max))."""
    th_max = math.asin(0.5 * aperture / focal)
    n_r = max(1, int(round(focal * th_max / h)))
    dth = th_max / n_r
    pos, area = [], []
    for i in range(n_r):
        th = (i + 0.5) * dth
        ring_r = focal * math.sin(th)
        n_t = max(1, int(round(2.0 * math.pi * ring_r / (focal * dth))))
        t = (np.arange(n_t) + 0.5) * (2.0 * math.pi / n_t)
        pos.append(np.stack([ring_r * np.cos(t), ring_r * np.sin(t), np.full(n_t, focal * (1.0 - math.cos(th)))], axis=1))
        a_ring = 2.0 * math.pi * focal ** 2 * (math.cos(th - 0.5 * dth) - math.cos(th + 0.5 * dth))
        area.append(np.full(n_t, a_ring / n_t))
    return np.concatenate(pos), np.concatenate(area)


def random_state(w: Workload, seed: int, scale_v: float = 1e-6, fields=None) -> dict:
    """Seeded random state for single-pass parity tests: 3 v, 6 sigma, 6 r as float32 arrays
    shaped (nz, ny, nx) (values exactly representable in fp32 so both sides start equal).
    ``fields``: draw only these (the others are left out of the result)."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 2000 + seed))
    out = {}
    shape = (w.nz, w.ny, w.nx)
    for names, scale in ((("vx", "vy", "vz"), scale_v), (("sxx", "syy", "szz", "sxy", "sxz", "syz"), 1.0),
                         (("rxx", "ryy", "rzz", "rxy", "rxz", "ryz"), 1e5)):
        for name in names:
            if fields is not None and name not in fields:
                continue
            a = rng.standard_normal(shape, dtype=np.float32)
            if scale != 1.0:
                a *= np.float32(scale)
            out[name] = a
    return out


# ----------------------------------------------------------------------------------------
# thermal step: inputs only
# ----------------------------------------------------------------------------------------
# PAPER.md lists no thermal tissue constants ("must be supplied by the
# user"); these are typical literature values (chosen): k W/m/K, specific heat J/kg/K, perfusion
# coefficient w_b rho_b C_b W/m^3/K.
THERMAL_WATER = (0.60, 4180.0, 0.0)
THERMAL_SOFT = (0.51, 3630.0, 4.0e4)
THERMAL_BONE = (0.32, 1313.0, 7.0e2)
BONE_ABSORBED_FRACTION = 0.16


def thermal_table_for(table) -> np.ndarray:
    """(k, rho C, w) rows for an acoustic table: solids are bone, lossy fluids soft tissue, the rest water."""
    rows = []
    for rho, cL, cS, aL, aS in np.asarray(table, dtype=np.float64):
        k, c, w = THERMAL_BONE if cS > 0 else (THERMAL_SOFT if aL > 0 else THERMAL_WATER)
        rows.append((k, rho * c, w))
    return np.array(rows, dtype=np.float64)


def absorbed_fraction_for(table) -> np.ndarray:
    """Fraction of the attenuation turned into heat: 0.16 in bone, 1 elsewhere."""
    t = np.asarray(table, dtype=np.float64)
    return np.where(t[:, 2] > 0, BONE_ABSORBED_FRACTION, 1.0)


def thermal_dt(table_thermal, dx: float, fraction: float = 0.4) -> float:
    """A time step (an input): `fraction` of dx^2 min(rho C) / (6 max k), two significant digits."""
    t = np.asarray(table_thermal, dtype=np.float64)
    dt = fraction * dx * dx * t[:, 1].min() / (6.0 * t[:, 0].max())
    e = 10.0 ** (math.floor(math.log10(dt)) - 1)
    return math.floor(dt / e) * e


def focal_heat(nx, ny, nz, dx, centre_mm, fwhm_mm=(3.0, 3.0, 12.0), q_max=2.0e6) -> np.ndarray:
    """A Gaussian focal spot of heat deposition (W/m^3), float32 (nz, ny, nx): the shape of the
    pressure-squared focus of an F# ~ 1 transducer at 500 kHz (about 3 x 3 x 12 mm)."""
    ax = [np.arange(n, dtype=np.float64) * dx * 1e3 for n in (nx, ny, nz)]
    g = [np.exp(-4.0 * math.log(2.0) * ((a - c) / f) ** 2) for a, c, f in zip(ax, centre_mm, fwhm_mm)]
    return (q_max * g[2][:, None, None] * g[1][None, :, None] * g[0][None, None, :]).astype(np.float32)


def thermal_domain(nx, ny, nz, seed, n_mat=5, dx=1e-3 / 3.0, T_b=37.0) -> dict:
    """A small heterogeneous block map with random thermal rows and a focal heat source plus
    scattered hot cells, for kernel-level parity tests of the thermal step."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 3000 + seed))
    rows = [(THERMAL_WATER[0], 1000.0 * THERMAL_WATER[1], 0.0)]
    for m in range(1, n_mat):
        rows.append((0.2 + rng.random(), 2.0e6 + 2.2e6 * rng.random(), 5.0e4 * rng.random() * (m % 2)))
    table = np.array(rows, dtype=np.float64)
    bz, by, bx = (nz + 2) // 3, (ny + 2) // 3, (nx + 2) // 3
    blocks = rng.integers(0, n_mat, size=(bz, by, bx), dtype=np.int64)
    idx = np.repeat(np.repeat(np.repeat(blocks, 3, 0), 3, 1), 3, 2)[:nz, :ny, :nx]
    idx = np.ascontiguousarray(idx).astype(np.uint8)
    dt = thermal_dt(table, dx)
    c_mm = [0.5 * n * dx * 1e3 for n in (nx, ny, nz)]
    # strong enough to heat by a few kelvin within ~50 steps of this small dt
    Q = focal_heat(nx, ny, nz, dx, c_mm, fwhm_mm=(2.0, 1.5, 3.0), q_max=0.2 * 3.0e6 / dt)
    Q = Q + (rng.random((nz, ny, nx)) < 0.02).astype(np.float32) * np.float32(0.05 * 3.0e6 / dt)
    return dict(nx=nx, ny=ny, nz=nz, dx=dx, dt=dt, T_b=T_b, table=table, index_map=idx, Q=Q)


def thermal_config2() -> dict:
    """Thermal run on config 2's domain (300 x 300 x 450, 128 materials): tissue rows by
    `thermal_table_for`, a focal spot 60 mm beyond the source plane (the bowl's focus), 40 s on at
    30 % duty + 20 s off in steps of dt."""
    w = config2(steps=1)
    table = thermal_table_for(w.table)
    dt = thermal_dt(table, w.dx)
    k_s = w.pml + 4
    c_mm = [(w.nx - 1) / 2 * w.dx * 1e3, (w.ny - 1) / 2 * w.dx * 1e3, k_s * w.dx * 1e3 + 60.0]
    Q = focal_heat(w.nx, w.ny, w.nz, w.dx, c_mm, q_max=2.0e6)
    return dict(nx=w.nx, ny=w.ny, nz=w.nz, dx=w.dx, dt=dt, T_b=37.0, table=table, index_map=w.index_map, Q=Q,
                duty=0.3, steps_on=int(round(40.0 / dt)), steps_off=int(round(20.0 / dt)))
