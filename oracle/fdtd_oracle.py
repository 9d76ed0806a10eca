"""ctypes front end of the fp64 CPU oracle (``fdtd_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this module.  It
shares no code with ``paper_2301_12727_b200`` and does not import it.

The arithmetic is all in ``fdtd_oracle.c`` (which cites PAPER.md passage by passage); this
file only marshals numpy arrays.  numpy arrays are shaped (nz, ny, nx), i.e. the dense
x-fastest layout ``i + nx*(j + ny*k)``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fdtd_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

FIELDS = ("vx", "vy", "vz", "sxx", "syy", "szz", "sxy", "sxz", "syz",
          "rxx", "ryy", "rzz", "rxy", "rxz", "ryz")
FIELD_ID = {n: i for i, n in enumerate(FIELDS)}
FIELD_ID.update(p=15, peak=16, rms_amp=17, sumsq=18, phasor_re=19, phasor_im=20)
DERIVED = ("rho", "pi_R", "mu_R", "tau_p", "tau_s", "pi_U", "mu_U", "c_U")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (no fast-math, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.orc_new.restype = C.c_void_p
        L.orc_new.argtypes = [C.c_int] * 4 + [C.c_double] * 2 + [C.c_int, dp, C.c_void_p,
                                                                 C.c_double, C.c_double,
                                                                 C.c_int64, C.c_int64, C.c_int64,
                                                                 C.POINTER(C.c_int)]
        L.orc_free.argtypes = [C.c_void_p]
        L.orc_set_source.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, dp, dp, C.c_int,
                                     C.c_double, C.c_int]
        L.orc_step.argtypes = [C.c_void_p, C.c_int64]
        L.orc_save_state.argtypes = [C.c_void_p, C.c_char_p]
        L.orc_load_state.argtypes = [C.c_void_p, C.c_char_p]
        for fn in ("orc_inject", "orc_velocity_pass", "orc_stress_pass", "orc_sensor"):
            getattr(L, fn).argtypes = [C.c_void_p]
        L.orc_step_index.restype = C.c_int64
        L.orc_step_index.argtypes = [C.c_void_p]
        L.orc_set_step_index.argtypes = [C.c_void_p, C.c_int64]
        L.orc_set_phasor.argtypes = [C.c_void_p, C.c_int]
        L.orc_rms_count.restype = C.c_int64
        L.orc_rms_count.argtypes = [C.c_void_p]
        L.orc_get_field.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_set_field.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_probe.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_void_p, dp]
        L.orc_get_derived.argtypes = [C.c_void_p, dp]
        L.orc_get_profile.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_derive_materials.argtypes = [C.c_int, dp, C.c_double, dp]
        L.orc_pml_profiles.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                       C.c_double, C.c_double, dp, dp, dp, dp]
        L.orc_pml_mask.argtypes = [C.c_int] * 4 + [C.c_void_p]
        L.orc_max_courant.restype = C.c_double
        L.orc_max_courant.argtypes = [C.c_int, dp, C.c_double, C.c_double]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def derive_materials(table, f0):
    """(n,5) rows (rho, cL, cS, alphaL, alphaS) -> (n,8) rho, pi_R, mu_R, tau_p, tau_s,
    pi_U, mu_U, c_U.  Raises ValueError on an invalid row."""
    t = np.ascontiguousarray(table, dtype=np.float64)
    out = np.zeros((t.shape[0], 8))
    if lib().orc_derive_materials(t.shape[0], _dp(t), float(f0), _dp(out)):
        raise ValueError("invalid material table")
    return out


def pml_profiles(n, P, dx, dt, f0, R, c_ref):
    """Returns (a_int, b_int, a_half, b_half), each of length n (fp64)."""
    arrs = [np.zeros(n) for _ in range(4)]
    lib().orc_pml_profiles(n, P, dx, dt, f0, R, c_ref, *[_dp(a) for a in arrs])
    return arrs


def pml_mask(nx, ny, nz, P):
    m = np.zeros((nz, ny, nx), dtype=np.uint8)
    lib().orc_pml_mask(nx, ny, nz, P, m.ctypes.data)
    return m


def max_courant(derived, dt, dx):
    d = np.ascontiguousarray(derived, dtype=np.float64)
    return lib().orc_max_courant(d.shape[0], _dp(d), dt, dx)


class Oracle:
    """One simulation context.  ``periodic`` is a test-only option (closed-form pins)."""

    def __init__(self, nx, ny, nz, pml, dx, dt, table, index_map, f0, pml_R=1e-4,
                 peak_begin=0, rms_begin=None, sensor_end=-1, periodic=(0, 0, 0)):
        self.nx, self.ny, self.nz, self.pml = nx, ny, nz, pml
        self.dx, self.dt, self.f0 = dx, dt, f0
        t = np.ascontiguousarray(table, dtype=np.float64)
        idx = np.ascontiguousarray(index_map, dtype=np.uint8)
        assert idx.size == nx * ny * nz
        if rms_begin is None or rms_begin < 0:
            rms_begin = np.iinfo(np.int64).max
        per = (C.c_int * 3)(*[int(p) for p in periodic])
        self._h = lib().orc_new(nx, ny, nz, pml, dx, dt, t.shape[0], _dp(t), idx.ctypes.data,
                                f0, pml_R, int(peak_begin), int(rms_begin), int(sensor_end), per)
        if not self._h:
            raise ValueError("oracle rejected the inputs (invalid table or index map)")
        self.shape = (nz, ny, nx)

    @classmethod
    def from_workload(cls, w, **kw):
        o = cls(w.nx, w.ny, w.nz, w.pml, w.dx, w.dt, w.table, w.index_map, w.f0, w.pml_R,
                w.peak_begin, w.rms_begin, w.sensor_end, **kw)
        o.set_source(w.src_cell, w.src_amp, w.src_delay, w.waveform, w.f_src, w.n_cycles)
        return o

    def close(self):
        if getattr(self, "_h", None):
            lib().orc_free(self._h)
            self._h = None

    __del__ = close

    def set_source(self, cell, amp, delay, waveform, f_src, n_cycles):
        cell = np.ascontiguousarray(cell, dtype=np.int64)
        amp = np.ascontiguousarray(amp, dtype=np.float64)
        delay = np.ascontiguousarray(delay, dtype=np.float64)
        if lib().orc_set_source(self._h, cell.size, cell.ctypes.data, _dp(amp), _dp(delay),
                                int(waveform), float(f_src), int(n_cycles)):
            raise ValueError("source cell outside the grid")

    def step(self, n=1):
        lib().orc_step(self._h, int(n))

    def save_state(self, path):
        """checkpoint of the time-dependent state (fields, psi, sensor maps, counters); no arithmetic"""
        if lib().orc_save_state(self._h, os.fsencode(path)):
            raise OSError(f"could not write {path}")

    def load_state(self, path):
        """resume from a checkpoint written by an oracle created with the same arguments"""
        if lib().orc_load_state(self._h, os.fsencode(path)):
            raise OSError(f"could not read {path} (or it belongs to another grid)")

    def inject(self):
        lib().orc_inject(self._h)

    def velocity_pass(self):
        lib().orc_velocity_pass(self._h)

    def stress_pass(self):
        lib().orc_stress_pass(self._h)

    def sensor(self):
        lib().orc_sensor(self._h)

    @property
    def step_index(self):
        return lib().orc_step_index(self._h)

    @step_index.setter
    def step_index(self, n):
        lib().orc_set_step_index(self._h, int(n))

    @property
    def rms_count(self):
        return lib().orc_rms_count(self._h)

    def set_phasor(self, on=True):
        """NEXT-3: the rms window accumulates the single-frequency phasor at f0 instead of peak / rms."""
        if lib().orc_set_phasor(self._h, 1 if on else 0):
            raise MemoryError("phasor accumulators")

    def get(self, name):
        out = np.zeros(self.shape)
        if lib().orc_get_field(self._h, FIELD_ID[name], _dp(out)):
            raise KeyError(name)
        return out

    def set(self, name, arr):
        a = np.ascontiguousarray(arr, dtype=np.float64)
        assert a.shape == self.shape
        if lib().orc_set_field(self._h, FIELD_ID[name], _dp(a)):
            raise KeyError(name)

    def probe(self, name, cells):
        cells = np.ascontiguousarray(cells, dtype=np.int64)
        out = np.zeros(cells.size)
        if lib().orc_probe(self._h, FIELD_ID[name], cells.size, cells.ctypes.data, _dp(out)):
            raise KeyError(name)
        return out

    def derived(self, n_mat):
        out = np.zeros((n_mat, 8))
        lib().orc_get_derived(self._h, _dp(out))
        return out

    def profile(self, axis, which):
        out = np.zeros((self.nx, self.ny, self.nz)[axis])
        lib().orc_get_profile(self._h, axis, which, _dp(out))
        return out
