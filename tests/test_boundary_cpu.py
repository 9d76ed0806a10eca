"""CPU-only checks of the C-ABI boundary (no compute calls): the library loads, exports every
symbol include/bvfdtd.h declares, and its host-side S0 constructions (per-material constants,
C-PML profiles, PML mask, stability number, workspace sizing) agree with the oracle's.

Construction parity: mask bit-exact; fp32 tables identical up to <= 1 ulp(fp32) for
entries that pass through tan/exp (the two sides are separate implementations of the same fp64
formulas, rounded once)."""
import os
import re

import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2301_12727_b200 import build as bv_build
from paper_2301_12727_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bv():
    bv_build.build()
    from paper_2301_12727_b200 import binding
    binding.lib()
    return binding


def test_header_symbols_exported(bv):
    hdr = open(os.path.join(ROOT, "include", "bvfdtd.h")).read()
    declared = set(re.findall(r"\b(bvfdtd_[a-z_]+)\s*\(", hdr))
    assert declared == set(bv.SYMBOLS), declared ^ set(bv.SYMBOLS)
    L = bv.lib()
    for s in declared:
        assert hasattr(L, s), s


def test_library_does_not_link_the_oracle(bv):
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", bv.LIB_PATH], capture_output=True, text=True).stdout
    assert "orc_" not in out
    srcs = os.listdir(os.path.join(ROOT, "paper_2301_12727_b200", "csrc"))
    for f in srcs:
        text = open(os.path.join(ROOT, "paper_2301_12727_b200", "csrc", f)).read()
        assert "orc_" not in text
        for inc in re.findall(r'#include\s+[<"]([^>"]+)[>"]', text):
            assert "oracle" not in inc
    for f in ("binding.py", "build.py", "__init__.py"):
        text = open(os.path.join(ROOT, "paper_2301_12727_b200", f)).read()
        assert "oracle" not in text


def _ulp_diff(a, b):
    a = np.asarray(a, np.float32).view(np.int32).astype(np.int64)
    b = np.asarray(b, np.float32).view(np.int32).astype(np.int64)
    return np.abs(a - b).max()


@pytest.mark.parametrize("cfg", [0, 1])
def test_derived_constants_match_oracle(bv, cfg):
    w = wl.make(cfg)
    got = bv.derive_materials(w.table, w.f0)
    ref = orc.derive_materials(w.table, w.f0).astype(np.float32)
    assert got.shape == ref.shape
    assert _ulp_diff(got, ref) <= 1
    # columns that involve no transcendental: exact
    assert np.array_equal(got[:, 0], ref[:, 0])


def test_derived_constants_big_tables(bv):
    for f0, n in ((500e3, 128), (700e3, 255), (250e3, 128)):
        t = wl._skull_table(n, f0)
        assert _ulp_diff(bv.derive_materials(t, f0), orc.derive_materials(t, f0).astype(np.float32)) <= 1


@pytest.mark.parametrize("n,P", [(64, 8), (300, 16), (41, 4), (40, 0), (672, 20)])
def test_pml_profiles_match_oracle(bv, n, P):
    dx, f0 = 1e-3 / 3, 500e3
    dt, _ = wl.snapped_dt(dx, f0, 3100.0)
    got = bv.pml_profiles(n, P, dx, dt, f0, 1e-4, 3100.0)
    ref = orc.pml_profiles(n, P, dx, dt, f0, 1e-4, 3100.0)
    for g, r in zip(got, ref):
        assert _ulp_diff(g, r.astype(np.float32)) <= 1
    # a is exactly zero outside the layer and at the low-side half node P-1 (xi = 0 there)
    a_int, _, a_half, _ = got
    assert np.all(a_int[P:n - P] == 0) and np.all(a_half[max(P - 1, 0):n - P] == 0)
    if P:
        assert np.all(a_int[:P] < 0) and np.all(a_int[n - P:] < 0)


@pytest.mark.parametrize("dims,P", [((64, 64, 64), 8), ((37, 29, 41), 4), ((24, 30, 26), 0)])
def test_pml_mask_bit_exact(bv, dims, P):
    nx, ny, nz = dims
    assert np.array_equal(bv.pml_mask(nx, ny, nz, P), orc.pml_mask(nx, ny, nz, P))


def test_max_courant_and_limits(bv):
    w = wl.make(0)
    c = bv.max_courant(w.table, w.f0, w.dt, w.dx)
    ref = orc.max_courant(orc.derive_materials(w.table, w.f0), w.dt, w.dx)
    assert abs(c - ref) <= 1e-12 * ref
    assert 0.3 < c < 0.494          # unrelaxed bone speed > table speed (reading P6)


def test_invalid_rows_rejected(bv):
    bad = [
        (0.0, 1500.0, 0.0, 0.0, 0.0),            # rho <= 0
        (1000.0, 0.0, 0.0, 0.0, 0.0),            # cL <= 0
        (1000.0, 1500.0, -1.0, 0.0, 0.0),        # cS < 0
        (1900.0, 2800.0, 2500.0, 0.0, 0.0),      # cS >= sqrt(3)/2 cL
        (1900.0, 2800.0, 1500.0, -1.0, 0.0),     # alpha < 0
        (1900.0, 2800.0, 1500.0, 500.0, 0.0),    # Q <= 1: 500*2800/(2 pi 5e5) = 0.446 > tan(pi/8)
    ]
    for row in bad:
        with pytest.raises(bv.BvfdtdError) as e:
            bv.derive_materials(np.array([wl.WATER, row]), 500e3)
        assert e.value.code == bv.EINVAL
        with pytest.raises(ValueError):
            orc.derive_materials(np.array([wl.WATER, row]), 500e3)


def test_workspace_bytes(bv):
    # 25 grid arrays (15 state, peak, sumsq, 2 phasor accumulators, the 6 ping-pong copies of the fused sweep)
    # + a dense scratch plane + the index map; padding and PML overhead below 25 % at config 2 size
    nx, ny, nz, P = 300, 300, 450, 16
    n = bv.workspace_bytes(nx, ny, nz, P)
    dense = nx * ny * nz * (26 * 4 + 1)
    assert dense < n < 1.25 * dense
    with pytest.raises(bv.BvfdtdError):
        bv.workspace_bytes(20, 64, 64, 8)        # dim < 2*pml + 8
    with pytest.raises(bv.BvfdtdError):
        bv.workspace_bytes(64, 64, 64, -1)


def test_no_gpu_means_loud_failure(bv):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    w = wl.make(0)
    with pytest.raises(RuntimeError):
        bv.Simulation.from_workload(w)


def test_tuning_bits_validated_before_any_device_call(bv):
    """bvfdtd_opts.tuning: unknown bits and contradictory requests are BVFDTD_EINVAL (checked with the other
    argument rules, before the library touches CUDA)."""
    import ctypes as C
    w = wl.make(0)
    g = bv.Grid(w.nx, w.ny, w.nz, w.pml)
    arr, n = bv._materials(w.table)
    for tuning in (128, 1 << 31, bv.TUNE_VEL_2CTA | bv.TUNE_VEL_3CTA, bv.TUNE_STRESS_8 | bv.TUNE_STRESS_16,
                   bv.TUNE_FUSED | bv.TUNE_NO_FUSED):
        o = bv.Opts(w.f0, 1e-4, 0, 0, -1, 0, tuning)
        h = C.c_void_p(None)
        rc = bv.lib().bvfdtd_create(C.byref(h), C.byref(g), w.dx, w.dt, arr, n, w.index_map.ctypes.data, C.byref(o),
                                    C.c_void_p(4096), 1 << 40, None)
        assert rc == bv.EINVAL and not h.value


def test_library_reads_no_environment_variable():
    """the launch plan of the shipped library must not depend on the caller's environment: every getenv in csrc/
    sits inside an #ifdef BVFDTD_DEV_KNOBS block, and the build does not define that macro"""
    csrc = os.path.join(ROOT, "paper_2301_12727_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        guarded = 0
        for line in open(os.path.join(csrc, f)):
            t = line.strip()
            if t.startswith("#ifdef BVFDTD_DEV_KNOBS"):
                guarded += 1
            elif t.startswith("#endif") and guarded:
                guarded -= 1
            elif t.startswith("#else") and guarded:
                guarded = 0
            if "getenv(" in line:
                assert guarded, (f, line)
    assert "BVFDTD_DEV_KNOBS" not in " ".join(bv_build.NVCC_FLAGS)
