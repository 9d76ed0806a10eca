"""Thin ctypes binding of ``include/bvfdtd.h`` -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; this module never computes
fields.  PyTorch is used for device memory (the caller-owned workspace) and the CUDA stream only.
There is no CPU fallback: if ``libbvfdtd.so`` is missing or no CUDA device is present, the calls
raise.  Names mirror the C entry points (``bvfdtd_create`` -> ``Simulation.__init__``,
``bvfdtd_set_source`` -> ``set_source``, ``bvfdtd_step`` -> ``step``, ``bvfdtd_read_fields`` ->
``read_fields``, ``bvfdtd_read_peak_pressure`` -> ``read_peak_pressure``).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbvfdtd.so")

FIELDS = ("vx", "vy", "vz", "sxx", "syy", "szz", "sxy", "sxz", "syz",
          "rxx", "ryy", "rzz", "rxy", "rxz", "ryz")
FIELD_ID = {n: i for i, n in enumerate(FIELDS)}
FIELD_ID.update(p=15, material=16, pml_mask=17, derived=18, pml_profiles=19, sumsq=20)
FLAG_REFERENCE_KERNELS = 1
FLAG_DENSE = 2
FLAG_PHASOR = 4
FLAG_ZLO_OPEN = 8
FLAG_ZHI_OPEN = 16
# bvfdtd_opts.tuning: launch-plan requests for tests and experiments (results never depend on them)
TUNE_VEL_2CTA, TUNE_VEL_3CTA, TUNE_STRESS_8, TUNE_STRESS_16, TUNE_NO_GRAPH, TUNE_NO_FUSED, TUNE_FUSED = 1, 2, 4, 8, 16, 32, 64

OK, EINVAL, ENOMEM, ESTABILITY, ECUDA, ESTATE = 0, -1, -2, -3, -4, -5

# every symbol include/bvfdtd.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "bvfdtd_workspace_bytes", "bvfdtd_create", "bvfdtd_set_source", "bvfdtd_step",
    "bvfdtd_step_index", "bvfdtd_read_fields", "bvfdtd_write_fields",
    "bvfdtd_read_peak_pressure", "bvfdtd_destroy", "bvfdtd_strerror", "bvfdtd_last_cuda_error",
    "bvfdtd_enable_kernel_timing", "bvfdtd_kernel_times", "bvfdtd_derive_materials",
    "bvfdtd_pml_profiles", "bvfdtd_pml_mask", "bvfdtd_max_courant",
    "bvfdtd_plane_intensity", "bvfdtd_energy_loss", "bvfdtd_rayleigh", "bvfdtd_rayleigh_noalloc", "bvfdtd_probe_mufu", "bvfdtd_read_phasor",
    "bvfdtd_bhte_workspace_bytes", "bvfdtd_bhte_create", "bvfdtd_bhte_set_heat",
    "bvfdtd_bhte_set_temperature", "bvfdtd_bhte_step", "bvfdtd_bhte_read", "bvfdtd_bhte_destroy",
    "bvfdtd_heat_source", "bvfdtd_step_phase", "bvfdtd_step_phase_planes", "bvfdtd_plane_span",
    "bvfdtd_refocus_weights", "bvfdtd_rms_count", "bvfdtd_kernel_mode", "bvfdtd_fused_coverage", "bvfdtd_work_items", "bvfdtd_padding_nonzeros", "bvfdtd_fused_lists_host",
)
MODE_REFERENCE, MODE_DENSE, MODE_SIGMA_WRITTEN, MODE_FUSED, MODE_GRAPH = 1, 2, 4, 8, 16
BHTE_TRACK_MAX = 1
BHTE_WHAT = {"T": 0, "dose": 1, "tmax": 2, "rise": 3}


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("pml", C.c_int32)]


class Material(C.Structure):
    _fields_ = [("rho", C.c_double), ("cL", C.c_double), ("cS", C.c_double),
                ("alphaL", C.c_double), ("alphaS", C.c_double)]


class Thermal(C.Structure):
    _fields_ = [("k", C.c_double), ("rho_c", C.c_double), ("perf", C.c_double)]


class Opts(C.Structure):
    _fields_ = [("f0", C.c_double), ("pml_R", C.c_double), ("peak_begin", C.c_int64),
                ("rms_begin", C.c_int64), ("sensor_end", C.c_int64), ("flags", C.c_uint32),
                ("tuning", C.c_uint32)]


class BvfdtdError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().bvfdtd_strerror(code).decode()
        if code == ECUDA or (code == ENOMEM and where == "bvfdtd_rayleigh_noalloc"):
            msg += ": " + lib().bvfdtd_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})")


_lib = None


def lib():
    """Load the C-ABI library (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2301_12727_b200.build`"
                              " (there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u32, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_double
        fp = C.POINTER(C.c_float)
        L.bvfdtd_workspace_bytes.argtypes = [C.POINTER(Grid), C.POINTER(C.c_size_t)]
        L.bvfdtd_create.argtypes = [C.POINTER(vp), C.POINTER(Grid), dbl, dbl, C.POINTER(Material),
                                    i32, vp, C.POINTER(Opts), vp, C.c_size_t, vp]
        L.bvfdtd_set_source.argtypes = [vp, i64, vp, vp, vp, i32, dbl, i32]
        L.bvfdtd_step.argtypes = [vp, i64]
        L.bvfdtd_step_index.argtypes = [vp]
        L.bvfdtd_step_index.restype = i64
        L.bvfdtd_rms_count.argtypes = [vp]
        L.bvfdtd_rms_count.restype = i64
        L.bvfdtd_kernel_mode.argtypes = [vp, C.POINTER(u32)]
        L.bvfdtd_fused_coverage.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
        L.bvfdtd_fused_lists_host.argtypes = [C.POINTER(Grid), vp, i32, i32, i32, vp, i64, C.POINTER(i64), vp]
        L.bvfdtd_padding_nonzeros.argtypes = [vp, C.POINTER(i64)]
        L.bvfdtd_work_items.argtypes = [vp, i32, vp, i64, C.POINTER(i64), C.POINTER(i32)]
        L.bvfdtd_read_fields.argtypes = [vp, u32, vp, C.c_size_t, i32]
        L.bvfdtd_write_fields.argtypes = [vp, u32, vp, C.c_size_t, i32]
        L.bvfdtd_read_peak_pressure.argtypes = [vp, vp, vp, i32]
        L.bvfdtd_destroy.argtypes = [vp]
        L.bvfdtd_strerror.argtypes = [C.c_int]
        L.bvfdtd_strerror.restype = C.c_char_p
        L.bvfdtd_last_cuda_error.restype = C.c_char_p
        L.bvfdtd_enable_kernel_timing.argtypes = [vp, i32]
        L.bvfdtd_kernel_times.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
        L.bvfdtd_derive_materials.argtypes = [C.POINTER(Material), i32, dbl, fp]
        L.bvfdtd_pml_profiles.argtypes = [i32, i32, dbl, dbl, dbl, dbl, dbl, fp, fp, fp, fp]
        L.bvfdtd_pml_mask.argtypes = [C.POINTER(Grid), vp]
        L.bvfdtd_max_courant.argtypes = [C.POINTER(Material), i32, dbl, dbl, dbl]
        L.bvfdtd_plane_intensity.argtypes = [vp, vp, vp]
        L.bvfdtd_read_phasor.argtypes = [vp, vp, vp, i32]
        L.bvfdtd_rayleigh.argtypes = [i64, vp, vp, i64, vp, dbl, dbl, dbl, vp, vp, vp, vp, vp]
        L.bvfdtd_rayleigh_noalloc.argtypes = [i64, vp, vp, i64, vp, dbl, dbl, dbl, vp, vp, vp, vp, vp]
        L.bvfdtd_probe_mufu.argtypes = [C.POINTER(dbl), vp]
        L.bvfdtd_energy_loss.argtypes = [vp, vp, vp, i32, i32, C.POINTER(i32), C.POINTER(dbl), C.POINTER(dbl)]
        L.bvfdtd_max_courant.restype = dbl
        L.bvfdtd_bhte_workspace_bytes.argtypes = [i32, i32, i32, u32, C.POINTER(C.c_size_t)]
        L.bvfdtd_bhte_create.argtypes = [C.POINTER(vp), i32, i32, i32, dbl, dbl, C.POINTER(Thermal), i32, vp, dbl, u32,
                                         vp, C.c_size_t, vp]
        L.bvfdtd_bhte_set_heat.argtypes = [vp, vp, i32]
        L.bvfdtd_bhte_set_temperature.argtypes = [vp, vp, i32]
        L.bvfdtd_bhte_step.argtypes = [vp, i64, dbl]
        L.bvfdtd_bhte_read.argtypes = [vp, u32, vp, C.c_size_t, i32]
        L.bvfdtd_bhte_destroy.argtypes = [vp]
        L.bvfdtd_heat_source.argtypes = [vp, vp, dbl, vp]
        L.bvfdtd_step_phase.argtypes = [vp, i32]
        L.bvfdtd_step_phase_planes.argtypes = [vp, i32, i32, i32]
        L.bvfdtd_refocus_weights.argtypes = [i64, vp, vp, vp, vp, i32, dbl, dbl, vp, vp, vp, vp]
        L.bvfdtd_plane_span.argtypes = [C.POINTER(Grid), u32, i32, i32, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
        _lib = L
    return _lib


def _check(code, where):
    if code != OK:
        raise BvfdtdError(code, where)


def _materials(table):
    t = np.ascontiguousarray(table, dtype=np.float64).reshape(-1, 5)
    arr = (Material * t.shape[0])()
    C.memmove(arr, t.ctypes.data, t.nbytes)
    return arr, t.shape[0]


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


# ---- host-only helpers (no GPU needed) -----------------------------------------------------

def workspace_bytes(nx, ny, nz, pml):
    g = Grid(nx, ny, nz, pml)
    out = C.c_size_t(0)
    _check(lib().bvfdtd_workspace_bytes(C.byref(g), C.byref(out)), "bvfdtd_workspace_bytes")
    return out.value


def derive_materials(table, f0):
    arr, n = _materials(table)
    out = np.zeros((n, 8), dtype=np.float32)
    _check(lib().bvfdtd_derive_materials(arr, n, float(f0), _fp(out)), "bvfdtd_derive_materials")
    return out


def pml_profiles(n, pml, dx, dt, f0, pml_R, c_ref):
    arrs = [np.zeros(n, dtype=np.float32) for _ in range(4)]
    _check(lib().bvfdtd_pml_profiles(n, pml, dx, dt, f0, pml_R, c_ref, *[_fp(a) for a in arrs]),
           "bvfdtd_pml_profiles")
    return arrs


def pml_mask(nx, ny, nz, pml):
    g = Grid(nx, ny, nz, pml)
    m = np.zeros((nz, ny, nx), dtype=np.uint8)
    _check(lib().bvfdtd_pml_mask(C.byref(g), m.ctypes.data), "bvfdtd_pml_mask")
    return m


def fused_lists_host(nx, ny, nz, pml, cls, stress_tile_rows=8, slots=444):
    """host-only: (fused items, velocity items, stress items, flag words (nty, ntx, nz + 4)) for class bytes
    cls[(nty, ntx, nz)] (bit 0 fluid within reach, bit 1 lossy), as bvfdtd_create builds them"""
    g = Grid(nx, ny, nz, pml)
    ntx, nty = (nx + 63) // 64, (ny + 7) // 8
    c = np.ascontiguousarray(cls, dtype=np.uint8).reshape(nty, ntx, nz)
    flags = np.zeros((nty, ntx, nz + 4), dtype=np.uint32)
    out = []
    for which in range(3):
        n = C.c_int64(0)
        _check(lib().bvfdtd_fused_lists_host(C.byref(g), c.ctypes.data, stress_tile_rows, slots, which, None, 0, C.byref(n), None),
               "bvfdtd_fused_lists_host")
        a = np.zeros((max(1, n.value), 4), dtype=np.int32)
        _check(lib().bvfdtd_fused_lists_host(C.byref(g), c.ctypes.data, stress_tile_rows, slots, which, a.ctypes.data, n.value,
                                             C.byref(n), flags.ctypes.data), "bvfdtd_fused_lists_host")
        out.append(a[:n.value])
    return out[0], out[1], out[2], flags


def max_courant(table, f0, dt, dx):
    arr, n = _materials(table)
    v = lib().bvfdtd_max_courant(arr, n, float(f0), float(dt), float(dx))
    if v < 0:
        raise BvfdtdError(int(v), "bvfdtd_max_courant")
    return v


# ---- the simulation -----------------------------------------------------------------------

def energy_loss(sum_tissue, sum_water, max_water, pml):
    """(z_m, E_L, T_S) of PAPER.md Eq. 2 / L164 from the plane reductions of the two runs."""
    a = np.ascontiguousarray(sum_tissue, dtype=np.float64)
    b = np.ascontiguousarray(sum_water, dtype=np.float64)
    c = np.ascontiguousarray(max_water, dtype=np.float64)
    zm, el, ts = C.c_int32(0), C.c_double(0.0), C.c_double(0.0)
    _check(lib().bvfdtd_energy_loss(a.ctypes.data, b.ctypes.data, c.ctypes.data, a.size, int(pml),
                                    C.byref(zm), C.byref(el), C.byref(ts)), "bvfdtd_energy_loss")
    return zm.value, el.value, ts.value


def rayleigh(src_xyz, src_weight, rcv_xyz, f, c0=1500.0, rho0=1000.0, device="cuda:0", want_source=True):
    """Rayleigh-Sommerfeld field (NEXT-1): complex64 pressure at the receivers and, if asked, the
    (amp, delay) arrays for ``Simulation.set_source``.  Inputs are numpy arrays (n,3), (n,) complex."""
    import torch
    dev = torch.device(device)
    s = torch.from_numpy(np.ascontiguousarray(src_xyz, dtype=np.float32)).to(dev)
    wc = np.ascontiguousarray(src_weight, dtype=np.complex64)
    w = torch.from_numpy(wc.view(np.float32).reshape(-1, 2).copy()).to(dev)
    r = torch.from_numpy(np.ascontiguousarray(rcv_xyz, dtype=np.float32)).to(dev)
    n_s, n_r = s.shape[0], r.shape[0]
    out = torch.empty((4, n_r), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    _check(lib().bvfdtd_rayleigh(n_s, s.data_ptr(), w.data_ptr(), n_r, r.data_ptr(), float(f), float(c0), float(rho0),
                                 out[0].data_ptr(), out[1].data_ptr(),
                                 out[2].data_ptr() if want_source else None, out[3].data_ptr() if want_source else None,
                                 stream), "bvfdtd_rayleigh")
    torch.cuda.synchronize(dev)
    o = out.cpu().numpy()
    p = o[0].astype(np.complex64) + 1j * o[1].astype(np.complex64)
    return (p, o[2], o[3]) if want_source else p


RAYLEIGH_NOALLOC_MAX_SRC = 65536


def rayleigh_noalloc(src_xyz, src_weight, rcv_xyz, f, c0=1500.0, rho0=1000.0, device="cuda:0"):
    """``bvfdtd_rayleigh_noalloc``: the field of ``rayleigh`` through the entry point that allocates nothing on the
    device (static scratch of RAYLEIGH_NOALLOC_MAX_SRC sources).  Returns (p complex64, amp, delay).  (The torch
    tensors below are this binding's marshalling of numpy inputs; a caller with device arrays passes its pointers.)"""
    import torch
    dev = torch.device(device)
    s = torch.from_numpy(np.ascontiguousarray(src_xyz, dtype=np.float32)).to(dev)
    wc = np.ascontiguousarray(src_weight, dtype=np.complex64)
    w = torch.from_numpy(wc.view(np.float32).reshape(-1, 2).copy()).to(dev)
    r = torch.from_numpy(np.ascontiguousarray(rcv_xyz, dtype=np.float32)).to(dev)
    out = torch.empty((4, r.shape[0]), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    _check(lib().bvfdtd_rayleigh_noalloc(s.shape[0], s.data_ptr(), w.data_ptr(), r.shape[0], r.data_ptr(), float(f), float(c0),
                                         float(rho0), out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(),
                                         out[3].data_ptr(), stream), "bvfdtd_rayleigh_noalloc")
    torch.cuda.synchronize(dev)
    o = out.cpu().numpy()
    return o[0].astype(np.complex64) + 1j * o[1].astype(np.complex64), o[2], o[3]


def probe_mufu(device="cuda:0"):
    """measured special-function-unit rate of the device (operations per second)"""
    import torch
    v = C.c_double(0.0)
    with torch.cuda.device(torch.device(device)):
        _check(lib().bvfdtd_probe_mufu(C.byref(v), torch.cuda.current_stream().cuda_stream), "bvfdtd_probe_mufu")
    return v.value


class Simulation:
    """``bvfdtd_create`` .. ``bvfdtd_destroy`` around a torch-owned device workspace."""

    def __init__(self, nx, ny, nz, pml, dx, dt, table, index_map, f0, pml_R=1e-4, peak_begin=0,
                 rms_begin=None, sensor_end=-1, flags=0, device="cuda:0", stream=None, tuning=0):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("bvfdtd needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.nx, self.ny, self.nz, self.pml = int(nx), int(ny), int(nz), int(pml)
        self.shape = (self.nz, self.ny, self.nx)
        self.cells = self.nx * self.ny * self.nz
        self.device = torch.device(device)
        idx = np.ascontiguousarray(index_map, dtype=np.uint8)
        if idx.size != self.cells:
            raise ValueError("index_map size does not match the grid")
        if rms_begin is None or rms_begin < 0:
            rms_begin = np.iinfo(np.int64).max
        g = Grid(self.nx, self.ny, self.nz, self.pml)
        nbytes = C.c_size_t(0)
        _check(lib().bvfdtd_workspace_bytes(C.byref(g), C.byref(nbytes)), "bvfdtd_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        arr, n = _materials(table)
        self.n_materials = n
        o = Opts(float(f0), float(pml_R), int(peak_begin), int(rms_begin), int(sensor_end),
                 int(flags), int(tuning))
        h = C.c_void_p(None)
        with torch.cuda.device(self.device):
            rc = lib().bvfdtd_create(C.byref(h), C.byref(g), float(dx), float(dt), arr, n,
                                     idx.ctypes.data, C.byref(o), self.workspace.data_ptr(),
                                     nbytes.value, self._stream.cuda_stream)
        _check(rc, "bvfdtd_create")
        self._h = h

    @classmethod
    def from_workload(cls, w, **kw):
        sim = cls(w.nx, w.ny, w.nz, w.pml, w.dx, w.dt, w.table, w.index_map, w.f0, w.pml_R,
                  w.peak_begin, w.rms_begin, w.sensor_end, **kw)
        sim.set_source(w.src_cell, w.src_amp, w.src_delay, w.waveform, w.f_src, w.n_cycles)
        return sim

    def close(self):
        h = getattr(self, "_h", None)
        if h:
            lib().bvfdtd_destroy(h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_source(self, cell, amp, delay, waveform, f_src, n_cycles):
        cell = np.ascontiguousarray(cell, dtype=np.int64)
        amp = np.ascontiguousarray(amp, dtype=np.float32)
        delay = np.ascontiguousarray(delay, dtype=np.float32)
        if not (cell.size == amp.size == delay.size):
            raise ValueError("source arrays differ in length")
        _check(lib().bvfdtd_set_source(self._h, cell.size, cell.ctypes.data, amp.ctypes.data,
                                       delay.ctypes.data, int(waveform), float(f_src),
                                       int(n_cycles)), "bvfdtd_set_source")

    def step(self, n=1):
        _check(lib().bvfdtd_step(self._h, int(n)), "bvfdtd_step")

    def step_phase(self, phase):
        """NEXT-5: one pass of the current step (0 inject, 1 velocity, 2 stress + sensor), in order."""
        _check(lib().bvfdtd_step_phase(self._h, int(phase)), "bvfdtd_step_phase")

    def step_phase_planes(self, phase, k0, k1):
        """NEXT-5: pass 1 or 2 over the planes [k0, k1) only (the ranges of a pass must add up to all planes)."""
        _check(lib().bvfdtd_step_phase_planes(self._h, int(phase), int(k0), int(k1)), "bvfdtd_step_phase_planes")

    @property
    def step_index(self):
        return lib().bvfdtd_step_index(self._h)

    @property
    def rms_count(self):
        return lib().bvfdtd_rms_count(self._h)

    def mode_bits(self):
        m = C.c_uint32(0)
        _check(lib().bvfdtd_kernel_mode(self._h, C.byref(m)), "bvfdtd_kernel_mode")
        return m.value

    def kernel_mode(self):
        """the path the next step runs, in words (what bench.py prints as config.kernels)"""
        m = self.mode_bits()
        if m & MODE_REFERENCE:
            return "reference (one thread per cell)"
        if m & MODE_DENSE:
            return "tiled, dense sweep"
        s = "tiled, tile-class skipping"
        if m & MODE_FUSED:
            s += ", fused sweep in all-fluid tile columns"
        if m & MODE_SIGMA_WRITTEN:
            s += " (normal stresses written by the caller: fluid shortcuts off)"
        return s

    def fused_coverage(self):
        """fraction of the 64 x 8 tile-planes the fused single sweep takes (0.0 outside the fused mode)"""
        a, b = C.c_int64(0), C.c_int64(0)
        _check(lib().bvfdtd_fused_coverage(self._h, C.byref(a), C.byref(b)), "bvfdtd_fused_coverage")
        return a.value / max(1, b.value)

    def padding_nonzeros(self):
        """non-zero floats in the zero gaps of the private layout (0 unless a kernel wrote out of bounds)"""
        n = C.c_int64(0)
        _check(lib().bvfdtd_padding_nonzeros(self._h, C.byref(n)), "bvfdtd_padding_nonzeros")
        return n.value

    def work_items(self, which):
        """(items (n, 4) int32: tile x, tile y, kz0, kz1; rows per tile) of work list 0 fused / 1 velocity / 2 stress"""
        n, rows = C.c_int64(0), C.c_int32(0)
        _check(lib().bvfdtd_work_items(self._h, which, None, 0, C.byref(n), C.byref(rows)), "bvfdtd_work_items")
        a = np.zeros((max(1, n.value), 4), dtype=np.int32)
        _check(lib().bvfdtd_work_items(self._h, which, a.ctypes.data, n.value, C.byref(n), C.byref(rows)), "bvfdtd_work_items")
        return a[:n.value], rows.value

    def synchronize(self):
        self._stream.synchronize()

    # -- readback -------------------------------------------------------------------------
    def read_fields(self, name, out=None):
        """Host numpy copy of one field, shaped (nz, ny, nx) for grid fields.  ``out`` may be a
        preallocated (pinned) numpy array of the right size."""
        fid = FIELD_ID[name]
        if name == "derived":
            a = np.zeros((self.n_materials, 8), dtype=np.float32)
        elif name == "pml_profiles":
            a = np.zeros(4 * (self.nx + self.ny + self.nz), dtype=np.float32)
        elif name in ("material", "pml_mask"):
            a = np.zeros(self.shape, dtype=np.uint8)
        else:
            a = np.zeros(self.shape, dtype=np.float32) if out is None else out
        _check(lib().bvfdtd_read_fields(self._h, fid, a.ctypes.data, a.nbytes, 0),
               "bvfdtd_read_fields")
        return a

    def read_fields_device(self, name):
        """Dense torch tensor on the device (enqueued on the context's stream)."""
        torch = self._torch
        fid = FIELD_ID[name]
        dt = torch.uint8 if name in ("material", "pml_mask") else torch.float32
        t = torch.empty(self.shape, dtype=dt, device=self.device)
        _check(lib().bvfdtd_read_fields(self._h, fid, t.data_ptr(), t.numel() * t.element_size(),
                                        1), "bvfdtd_read_fields")
        return t

    def write_fields(self, name, arr):
        a = np.ascontiguousarray(arr, dtype=np.float32)
        if a.size != self.cells:
            raise ValueError("field size does not match the grid")
        _check(lib().bvfdtd_write_fields(self._h, FIELD_ID[name], a.ctypes.data, a.nbytes, 0),
               "bvfdtd_write_fields")

    def read_peak_pressure(self, peak=True, rms=True, out_peak=None, out_rms=None):
        """(peak, rms_amp) as host numpy arrays (None for the one not requested)."""
        p = (np.zeros(self.shape, dtype=np.float32) if out_peak is None else out_peak) if peak else None
        r = (np.zeros(self.shape, dtype=np.float32) if out_rms is None else out_rms) if rms else None
        _check(lib().bvfdtd_read_peak_pressure(self._h, p.ctypes.data if peak else None,
                                               r.ctypes.data if rms else None, 0),
               "bvfdtd_read_peak_pressure")
        return p, r

    def read_peak_pressure_device(self):
        torch = self._torch
        p = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        r = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        _check(lib().bvfdtd_read_peak_pressure(self._h, p.data_ptr(), r.data_ptr(), 1),
               "bvfdtd_read_peak_pressure")
        return p, r

    # -- NEXT-3: complex pressure amplitude -------------------------------------------------
    def read_phasor(self):
        """complex64 (nz, ny, nx): P with p(t) = Re{P exp(j 2 pi f0 t)} (needs FLAG_PHASOR)."""
        re = np.empty(self.shape, dtype=np.float32)
        im = np.empty(self.shape, dtype=np.float32)
        _check(lib().bvfdtd_read_phasor(self._h, re.ctypes.data, im.ctypes.data, 0), "bvfdtd_read_phasor")
        return re + 1j * im

    def read_phasor_device(self):
        """(re, im) as dense float32 torch tensors on the device."""
        torch = self._torch
        re = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        im = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        _check(lib().bvfdtd_read_phasor(self._h, re.data_ptr(), im.data_ptr(), 1), "bvfdtd_read_phasor")
        return re, im

    # -- NEXT-2: plane reductions of the pulse-average intensity ---------------------------
    def plane_intensity(self):
        """(plane_sum, plane_max) of I_PA over the interior cells of every z plane (float64, nz)."""
        s = np.zeros(self.nz, dtype=np.float64)
        m = np.zeros(self.nz, dtype=np.float64)
        _check(lib().bvfdtd_plane_intensity(self._h, s.ctypes.data, m.ctypes.data), "bvfdtd_plane_intensity")
        return s, m

    # -- NEXT-4: heat deposition of the harmonic field ---------------------------------------
    def heat_source(self, absorbed_fraction, scale=1.0):
        """Q (W/m^3) as a dense float32 torch tensor (nz, ny, nx) on the device."""
        torch = self._torch
        a = np.ascontiguousarray(absorbed_fraction, dtype=np.float64)
        if a.size != self.n_materials:
            raise ValueError("one absorbed fraction per material")
        q = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        _check(lib().bvfdtd_heat_source(self._h, a.ctypes.data, float(scale), q.data_ptr()), "bvfdtd_heat_source")
        return q

    # -- device-time accounting (bench) ---------------------------------------------------
    def enable_kernel_timing(self, on=True):
        _check(lib().bvfdtd_enable_kernel_timing(self._h, 1 if on else 0),
               "bvfdtd_enable_kernel_timing")

    def kernel_times(self):
        ms = (C.c_double * 4)()
        n = (C.c_int64 * 4)()
        _check(lib().bvfdtd_kernel_times(self._h, ms, n), "bvfdtd_kernel_times")
        names = ("inject", "fused", "velocity", "stress_sensor")
        return {k: {"ms": ms[i], "launches": n[i]} for i, k in enumerate(names)}


class Bhte:
    """``bvfdtd_bhte_create`` .. ``bvfdtd_bhte_destroy`` (NEXT-4, thermal step) around a torch-owned
    device workspace.  ``table`` rows are (k, rho C, perfusion coefficient)."""

    def __init__(self, nx, ny, nz, dx, dt, table, index_map, T_b=37.0, track_max=True, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("bvfdtd needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.cells = self.nx * self.ny * self.nz
        self.device = torch.device(device)
        self.T_b = float(T_b)
        idx = np.ascontiguousarray(index_map, dtype=np.uint8)
        if idx.size != self.cells:
            raise ValueError("index_map size does not match the grid")
        t = np.ascontiguousarray(table, dtype=np.float64).reshape(-1, 3)
        arr = (Thermal * t.shape[0])()
        C.memmove(arr, t.ctypes.data, t.nbytes)
        flags = BHTE_TRACK_MAX if track_max else 0
        nbytes = C.c_size_t(0)
        _check(lib().bvfdtd_bhte_workspace_bytes(self.nx, self.ny, self.nz, flags, C.byref(nbytes)),
               "bvfdtd_bhte_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p(None)
            rc = lib().bvfdtd_bhte_create(C.byref(h), self.nx, self.ny, self.nz, float(dx), float(dt), arr, t.shape[0],
                                          idx.ctypes.data, self.T_b, flags, self.workspace.data_ptr(), nbytes.value,
                                          self._stream.cuda_stream)
        _check(rc, "bvfdtd_bhte_create")
        self._h = h

    def close(self):
        h = getattr(self, "_h", None)
        if h:
            lib().bvfdtd_bhte_destroy(h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _src(self, a):
        """(pointer, is_device, keep-alive) of a dense float32 field given as numpy or a torch device tensor."""
        torch = self._torch
        if isinstance(a, torch.Tensor):
            t = a.to(device=self.device, dtype=torch.float32).contiguous()
            if t.numel() != self.cells:
                raise ValueError("field size does not match the grid")
            return t.data_ptr(), 1, t
        n = np.ascontiguousarray(a, dtype=np.float32)
        if n.size != self.cells:
            raise ValueError("field size does not match the grid")
        return n.ctypes.data, 0, n

    def set_heat(self, Q):
        p, dev, keep = self._src(Q)
        _check(lib().bvfdtd_bhte_set_heat(self._h, p, dev), "bvfdtd_bhte_set_heat")
        if dev:
            self._stream.synchronize()      # `keep` may be a temporary

    def set_temperature(self, T):
        p, dev, keep = self._src(T)
        _check(lib().bvfdtd_bhte_set_temperature(self._h, p, dev), "bvfdtd_bhte_set_temperature")
        if dev:
            self._stream.synchronize()

    def step(self, n, heat_scale):
        _check(lib().bvfdtd_bhte_step(self._h, int(n), float(heat_scale)), "bvfdtd_bhte_step")

    def synchronize(self):
        self._stream.synchronize()

    def read(self, what, out=None):
        """Host float32 (nz, ny, nx): "T", "dose" (CEM43 minutes), "tmax", "rise" (T - T_b)."""
        a = np.empty(self.shape, dtype=np.float32) if out is None else out
        _check(lib().bvfdtd_bhte_read(self._h, BHTE_WHAT[what], a.ctypes.data, a.nbytes, 0), "bvfdtd_bhte_read")
        return a
