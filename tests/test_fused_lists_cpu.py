"""CPU tests of the host logic behind the fused mode (`fused_lists`, csrc/kernels_fused.cuh) through the host-only
entry point bvfdtd_fused_lists_host: from per-(tile, plane) class bytes to the three work lists and the flag words.

Invariants (what the kernels rely on):
  * lists fused + velocity, and fused + stress, cover every tile-plane exactly once (in-place arrays -- psi, r, the
    sensor maps -- must be updated once per step);
  * a plane is fused only if planes k-3 .. k+3 of the tile (and of its partner in a 64 x 16 stress tile) are fluid
    within reach; runs have at least 16 planes;
  * no boundary of a fused item lies inside, or within two planes of, a z slab (a chunk recomputes vz at kz0-2,
    kz0-1, kz1 without the psi it does not own) -- config 3 has tile columns whose all-fluid run starts inside the
    top slab;
  * tiles whose halo columns would need the x-psi of a neighbouring tile are never fused;
  * a fused plane carries FF_WYY when a y-neighbour tile runs the two passes there, FF_WZZ when a plane within
    k-2 .. k+1 of the same tile does (the velocity pass of that neighbour reads sigma_yy / sigma_zz there)."""
import numpy as np
import pytest

from paper_2301_12727_b200 import build as bv_build

FLUID4, LOSSY, RUN, WYY, WZZ = 1, 2, 4, 8, 16


@pytest.fixture(scope="module")
def bv():
    bv_build.build()
    from paper_2301_12727_b200 import binding
    binding.lib()
    return binding


def _cover(items, nty, ntx, nz):
    cnt = np.zeros((nty, ntx, nz), np.int32)
    for bx, by, a, b in items:
        assert 0 <= a < b <= nz and 0 <= bx < ntx and 0 <= by < nty
        cnt[by, bx, a:b] += 1
    return cnt


def _check(bv, nx, ny, nz, P, cls, sty):
    ntx, nty = (nx + 63) // 64, (ny + 7) // 8
    f, v, s, flags = bv.fused_lists_host(nx, ny, nz, P, cls, stress_tile_rows=sty, slots=296)
    cf, cv = _cover(f, nty, ntx, nz), _cover(v, nty, ntx, nz)
    g = sty // 8
    cs = _cover(s, (ny + sty - 1) // sty, ntx, nz)
    assert ((cf + cv) == 1).all()
    assert ((cf[::g] + cs) == 1).all()
    run = (flags[:, :, 2:nz + 2] & RUN) != 0
    assert np.array_equal(run, cf == 1)
    assert (flags[:, :, :2] == 0).all() and (flags[:, :, nz + 2:] == 0).all()
    fluid = (cls.reshape(nty, ntx, nz) & FLUID4) != 0
    for by in range(nty):
        for bx in range(ntx):
            r = run[by, bx]
            if not r.any():
                continue
            partner = by ^ 1 if g == 2 and (by ^ 1) < nty else by
            ok = fluid[by, bx] & fluid[partner, bx]
            if g == 2:
                assert np.array_equal(r, run[partner, bx])
            for k in np.nonzero(r)[0]:
                assert ok[max(0, k - 3):k + 4].all(), (bx, by, k)
            # runs: at least 16 planes, ends outside the slabs
            edges = np.flatnonzero(np.diff(np.concatenate([[0], r.astype(np.int8), [0]])))
            for a, b in zip(edges[::2], edges[1::2]):
                assert b - a >= 16
                for e in (a, b):
                    assert P == 0 or e in (0, nz) or P + 2 <= e <= nz - P - 1, (bx, by, a, b)
            # x rule: the two columns left and the one right of the tile are outside the x slabs (or the grid)
            x0 = 64 * bx
            for i in (x0 - 2, x0 - 1, x0 + 64):
                assert not (P > 0 and 0 <= i < nx and (i < P or i >= nx - P)), (bx, i)
    if P > 0:
        for bx, by, a, b in f:
            for e in (a, b):
                assert e in (0, nz) or P + 2 <= e <= nz - P - 1
    # the extra stores
    w = flags[:, :, 2:nz + 2]
    for by in range(nty):
        for bx in range(ntx):
            for k in np.nonzero(run[by, bx])[0]:
                nb = [run[q, bx, k] for q in (by - 1, by + 1) if 0 <= q < nty]
                assert bool(w[by, bx, k] & WYY) == (not all(nb))
                zz = [run[by, bx, q] for q in range(k - 2, k + 2) if 0 <= q < nz]
                assert bool(w[by, bx, k] & WZZ) == (not all(zz))
    assert ((w & LOSSY) != 0).sum() == ((cls & LOSSY) != 0).sum()
    return f, v, s, run


@pytest.mark.parametrize("sty", [8, 16])
@pytest.mark.parametrize("dims,P", [((300, 72, 120), 16), ((150, 60, 96), 6), ((200, 44, 70), 0), ((504, 88, 140), 20)])
def test_lists_from_random_class_maps(bv, dims, P, sty):
    nx, ny, nz = dims
    ntx, nty = (nx + 63) // 64, (ny + 7) // 8
    rng = np.random.default_rng(nx + 7 * ny + sty)
    for trial in range(4):
        cls = np.full((nty, ntx, nz), FLUID4, np.uint8)
        for _ in range(rng.integers(1, 6)):          # blobs of "solid within reach"
            y0, x0, z0 = rng.integers(0, nty), rng.integers(0, ntx), rng.integers(0, nz)
            cls[y0:y0 + rng.integers(1, 4), x0:x0 + rng.integers(1, 3), z0:z0 + rng.integers(1, nz // 2)] = 0
        cls |= (rng.random(cls.shape) < 0.3).astype(np.uint8) * LOSSY
        if P > 0 and ny < 2 * P + 24:
            f, v, s, flags = bv.fused_lists_host(nx, ny, nz, P, cls, stress_tile_rows=sty)
            assert len(f) == 0                       # a tile (or its halo rows) would touch both y slabs: never fused
            continue
        _check(bv, nx, ny, nz, P, cls, sty)


def test_run_inside_the_top_slab_is_not_fused(bv):
    """the case config 3 brought up: solids under the top z slab leave an all-fluid run that starts inside it"""
    nx, ny, nz, P = 504, 88, 140, 20
    ntx, nty = 8, 11
    cls = np.full((nty, ntx, nz), FLUID4, np.uint8)
    cls[4:6, 1, 100:119] = 0                          # fluid again from plane 119 on: 119 + 3 = 122 > nz - P - 1 = 119
    cls[8, 2, 5:9] = 0                                # ... and a run [0, 2) under the low slab
    f, v, s, run = _check(bv, nx, ny, nz, P, cls, 8)
    assert not run[4, 1, 97:].any() and run[4, 1, :97].all()
    assert not run[8, 2, :12].any()
    # lossless all-fluid grid: everything fused, one column per tile, chunk boundaries outside the slabs
    cls[:] = FLUID4
    f, v, s, run = _check(bv, nx, ny, nz, P, cls, 16)
    assert run.all() and len(v) == 0 and len(s) == 0


def test_x_rule_and_small_y(bv):
    # nx = 330, P = 16: the high slab [314, 330) lies in tiles 4 (256..319) and 5; column 320 (right of tile 4) is in
    # the slab and so are 318, 319 (left of tile 5): neither tile is fused
    nx, ny, nz, P = 330, 72, 64, 16
    cls = np.full((9, 6, nz), FLUID4, np.uint8)
    f, v, s, run = _check(bv, nx, ny, nz, P, cls, 8)
    assert not run[:, 4].any() and not run[:, 5].any() and run[:, :4].all()
