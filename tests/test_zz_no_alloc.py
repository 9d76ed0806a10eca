"""bvfdtd_rayleigh_noalloc: the Rayleigh-Sommerfeld field through the one entry point that allocates nothing on the
device (callers under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Its scratch --
the sources packed as float4 -- is a static device array of BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC entries that all calls
share and that keeps the last call's contents.

GPU test: two calls in a row (the second with FEWER sources and other positions, so stale entries of the first call
sit behind the ones it reads) against the existing path `bvfdtd_rayleigh`, within the tolerance of
tests/test_rayleigh.py (relative L2 1e-4, amplitudes 1e-3, delays 2e-4 of a period); then the first call again.
The file name sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide other tests.
It passes alone in a fresh process and after the other tests (the scratch address is resolved on first use)."""
import math

import numpy as np
import pytest

from paper_2301_12727_b200 import workloads as wl

F, C0, RHO = 500e3, 1500.0, 1000.0
LAM = C0 / F


def test_header_states_the_limit():
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "bvfdtd.h")).read()
    m = re.search(r"BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC\s*=\s*(\d+)", hdr)
    from paper_2301_12727_b200 import build as bv_build
    bv_build.build()
    from paper_2301_12727_b200 import binding as bv
    assert m and int(m.group(1)) == bv.RAYLEIGH_NOALLOC_MAX_SRC == 65536


def _case(seed, aperture, n_x, n_y):
    pos, area = wl.bowl_elements(aperture, 64e-3, LAM / 4)
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + seed))
    wgt = area * 0.01 * np.exp(2j * math.pi * rng.random(area.size)) * (0.5 + rng.random(area.size))
    xs = (np.arange(n_x) - n_x // 2) * (LAM / 9)
    ys = (np.arange(n_y) - n_y // 2) * (LAM / 9) + 1e-4
    X, Y = np.meshgrid(xs, ys)
    rcv = np.stack([X.ravel(), Y.ravel(), np.full(X.size, 15e-3)], axis=1)
    return pos, wgt, rcv


def _agree(got, ref):
    p, amp, delay = got
    p0, amp0, delay0 = ref
    assert np.isfinite(p).all() and np.isfinite(amp).all() and np.isfinite(delay).all()
    assert np.linalg.norm(p - p0) <= 1e-4 * np.linalg.norm(p0)
    big = amp0 > 0.1 * amp0.max()
    assert np.abs(amp[big] / amp0[big] - 1).max() < 1e-3
    dd = np.abs(delay[big] - delay0[big])
    dd = np.minimum(dd, 1 / F - dd)
    assert dd.max() * F < 2e-4


@pytest.mark.gpu
def test_gpu_rayleigh_noalloc_matches_the_existing_path_on_two_calls_in_a_row():
    from paper_2301_12727_b200 import build as bv_build
    bv_build.build()
    from paper_2301_12727_b200 import binding as bv
    first = _case(91, 64e-3, 41, 37)          # ~6000 sources, 1517 receivers: several source tiles, a ragged tail
    second = _case(92, 30e-3, 23, 50)         # fewer sources, other positions and weights
    assert second[0].shape[0] < first[0].shape[0] <= bv.RAYLEIGH_NOALLOC_MAX_SRC
    got1 = bv.rayleigh_noalloc(*first, F, C0, RHO)
    got2 = bv.rayleigh_noalloc(*second, F, C0, RHO)         # shares the scratch with the call before
    _agree(got1, bv.rayleigh(*first, F, C0, RHO))
    _agree(got2, bv.rayleigh(*second, F, C0, RHO))
    got3 = bv.rayleigh_noalloc(*first, F, C0, RHO)
    for a, b in zip(got1, got3):
        assert np.array_equal(a, b)                         # the same call gives the same bits, whatever ran before
    # beyond the static scratch: refused with an error that names the limit, nothing launched
    n = bv.RAYLEIGH_NOALLOC_MAX_SRC + 1
    with pytest.raises(bv.BvfdtdError) as e:
        bv.rayleigh_noalloc(np.zeros((n, 3), np.float32) + 1e-3, np.ones(n, np.complex64), first[2][:4], F, C0, RHO)
    assert e.value.code == bv.ENOMEM and "BVFDTD_RAYLEIGH_NOALLOC_MAX_SRC" in str(e.value)
    # exactly at the limit it runs
    rng = np.random.Generator(np.random.PCG64(wl.SEED_BASE + 93))
    pos = (rng.random((bv.RAYLEIGH_NOALLOC_MAX_SRC, 3)) * 2e-2).astype(np.float32)
    pos[:, 2] = 0.0
    w = np.ones(pos.shape[0], np.complex64) * 1e-9
    rc = np.array([[0.0, 0.0, 3e-2], [5e-3, 1e-3, 2e-2]])
    _agree(bv.rayleigh_noalloc(pos, w, rc, F, C0, RHO), bv.rayleigh(pos, w, rc, F, C0, RHO))
