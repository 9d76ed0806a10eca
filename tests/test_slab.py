"""NEXT-5: z-slab decomposition.

CPU: the partition, the local workloads, the halo plan (``bvfdtd_plane_span`` is host-only) and the
point-to-point exchange itself on CPU byte tensors under gloo with 2 and 3 ranks.
GPU (one device): all slabs of a run in one process, stepped in lock step, reproduce the undivided
run BIT FOR BIT on every owned plane (state, peak, rms), with the tiled and the per-cell kernels, whole passes
and passes split around the exchange; SlabRank as a two-process torch.distributed job (gloo, staged exchange) on
the one GPU, against the undivided run and the oracle.
"""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

from paper_2301_12727_b200 import binding as bv
from paper_2301_12727_b200 import slab
from paper_2301_12727_b200 import workloads as wl


def test_partition_and_local_workloads_cover_the_domain():
    w = wl.random_domain(40, 36, 91, 6, seed=5, steps=10)
    for world in (1, 2, 3):
        parts = slab.partition(w.nz, world, w.pml)
        assert parts[0][0] == 0 and parts[-1][1] == w.nz
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        assert max(z1 - z0 for z0, z1 in parts) - min(z1 - z0 for z0, z1 in parts) <= 1
        n_src = 0
        for r in range(world):
            lw, meta = slab.local_workload(w, r, world)
            lo, hi = meta["lo"], meta["hi"]
            assert (lo, hi) == ((2 if r > 0 else 0), (2 if r < world - 1 else 0))
            assert lw.nz == meta["z1"] - meta["z0"] + lo + hi
            assert np.array_equal(lw.index_map, w.index_map[meta["z0"] - lo:meta["z1"] + hi])
            # local source cells map back to the global ones, all inside the owned planes
            g = lw.src_cell + (meta["z0"] - lo) * w.nx * w.ny
            assert np.all(np.isin(g, w.src_cell))
            k = g // (w.nx * w.ny)
            assert np.all((k >= meta["z0"]) & (k < meta["z1"]))
            n_src += g.size
        assert n_src == w.src_cell.size
    with pytest.raises(ValueError):
        slab.partition(40, 4, 8)            # slabs thinner than 2 pml + 8


def test_plane_span_is_contiguous_and_inside_the_workspace():
    nx, ny, nz, P = 50, 44, 37, 6
    total = bv.workspace_bytes(nx, ny, nz, P)
    spans = {}
    for f in slab.STRESS + slab.VELOCITY:
        o0, b0 = slab.plane_span(nx, ny, nz, P, f, 0, 1)
        o1, b1 = slab.plane_span(nx, ny, nz, P, f, 1, 1)
        o2, b2 = slab.plane_span(nx, ny, nz, P, f, 0, 2)
        assert b0 == b1 and o1 == o0 + b0 and (o2, b2) == (o0, 2 * b0)   # consecutive planes are adjacent
        assert b0 >= nx * ny * 4 and o0 % 4 == 0
        oe, be = slab.plane_span(nx, ny, nz, P, f, nz - 2, 2)
        assert oe + be <= total
        spans[f] = (o0, oe + be)
    iv = sorted(spans.values())
    assert all(a[1] <= b[0] for a, b in zip(iv, iv[1:]))                  # fields do not overlap
    with pytest.raises(bv.BvfdtdError):
        slab.plane_span(nx, ny, nz, P, "sxx", nz - 1, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _exchange_worker(rank, world, port, nx, ny, nz, pml, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        z0, z1 = slab.partition(nz, world, pml)[rank]
        lo, hi = slab.local_halos(rank, world)
        nzl = z1 - z0 + lo + hi
        ws = torch.zeros(bv.workspace_bytes(nx, ny, nzl, pml), dtype=torch.uint8)
        plan = slab.halo_plan(nx, ny, nzl, pml, lo, hi, slab.STRESS)
        # every owned plane of every field carries (field number, GLOBAL plane number); halos carry 255
        for fi, f in enumerate(slab.STRESS):
            for kl in range(nzl):
                off, nb = slab.plane_span(nx, ny, nzl, pml, f, kl, 1)
                owned = lo <= kl < nzl - hi
                ws[off:off + nb] = (16 * fi + (z0 - lo + kl) % 16) if owned else 255
        before = ws.clone()
        slab.exchange_distributed(ws, plan, rank, world)
        ok = True
        for fi, f in enumerate(slab.STRESS):
            for kl in range(nzl):
                off, nb = slab.plane_span(nx, ny, nzl, pml, f, kl, 1)
                want = 16 * fi + (z0 - lo + kl) % 16      # after the exchange halos hold their owner's values
                ok &= bool((ws[off:off + nb] == want).all())
        # nothing outside the received halo blocks changed
        mask = torch.ones_like(ws, dtype=torch.bool)
        for e in plan:
            for key in ("recv_lo", "recv_hi"):
                if key in e:
                    mask[e[key][0]:e[key][0] + e[key][1]] = False
        ok &= bool((ws[mask] == before[mask]).all())
        q.put((rank, ok))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_gloo(world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_exchange_worker, args=(r, world, port, 24, 20, 75, 4, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(res) == [(r, True) for r in range(world)]


# ------------------------------------------------------------------------------------------
# GPU: the decomposition reproduces the undivided run bit for bit
# ------------------------------------------------------------------------------------------

@pytest.mark.gpu
@pytest.mark.parametrize("n_slabs,flags", [(2, 0), (3, 0), (2, bv.FLAG_REFERENCE_KERNELS), (3, bv.FLAG_DENSE)])
def test_gpu_slabs_match_the_undivided_run_bitwise(n_slabs, flags):
    w = wl.random_domain(70, 45, 96, 6, seed=31, steps=45, waveform=1)
    w.rms_begin = 20
    full = bv.Simulation.from_workload(w, device="cuda:0", flags=flags)
    full.step(w.steps)
    grp = slab.SlabGroup(w, n_slabs, device="cuda:0", flags=flags)
    grp.step(w.steps)
    for name in bv.FIELDS:
        a, b = full.read_fields(name), grp.read_fields(name)
        assert np.abs(a).max() > 0
        assert np.array_equal(a, b), (name, float(np.abs(a - b).max()))
    pk, rm = full.read_peak_pressure()
    pk2, rm2 = grp.read_peak_pressure()
    assert np.array_equal(pk, pk2) and np.array_equal(rm, rm2)
    # the mask of a slab shows no z absorber on its interfaces
    m = grp.slabs[0].sim.read_fields("pml_mask")
    assert (m[-1] & 4).max() == 0 and (m[0] & 4).min() == 4
    full.close(); grp.close()


@pytest.mark.gpu
def test_gpu_step_phase_order_is_enforced():
    w = wl.random_domain(40, 36, 44, 6, seed=2, steps=4)
    a = bv.Simulation.from_workload(w, device="cuda:0")
    b = bv.Simulation.from_workload(w, device="cuda:0")
    a.step(3)
    for _ in range(3):
        b.step_phase(0); b.step_phase(1); b.step_phase(2)
    assert b.step_index == 3
    for name in bv.FIELDS:
        assert np.array_equal(a.read_fields(name), b.read_fields(name))
    with pytest.raises(bv.BvfdtdError):
        b.step_phase(1)                       # velocity before inject
    b.step_phase(0)
    with pytest.raises(bv.BvfdtdError):
        b.step(1)                             # a step is in progress
    with pytest.raises(bv.BvfdtdError):
        b.step_phase(2)
    b.step_phase(1); b.step_phase(2)
    assert b.step_index == 4
    a.close(); b.close()


@pytest.mark.gpu
@pytest.mark.parametrize("n_slabs", [2, 3])
def test_gpu_slabs_split_passes_match_bitwise_and_the_oracle(n_slabs):
    """every pass split the way SlabRank overlaps it with the exchange (planes that read no halo first, the planes
    next to the interfaces after the exchange, bvfdtd_step_phase_planes): bit-identical to the undivided run, and
    the stitched field meets the oracle within north_star's bars"""
    from oracle import fdtd_oracle as orc
    from test_gpu_parity import compare_map
    w = wl.random_domain(70, 45, 96, 6, seed=33, steps=40, waveform=1)
    w.rms_begin = 18
    full = bv.Simulation.from_workload(w, device="cuda:0")
    full.step(w.steps)
    grp = slab.SlabGroup(w, n_slabs, device="cuda:0", split=True)
    grp.step(w.steps)
    o = orc.Oracle.from_workload(w)
    o.step(w.steps)
    for name in bv.FIELDS:
        a, b = full.read_fields(name), grp.read_fields(name)
        assert np.array_equal(a, b), name
        ref = o.get(name)
        nrm = np.linalg.norm(ref)
        if nrm > 0:
            assert np.linalg.norm(b - ref) / nrm <= 1e-4, name
    pk, rm = full.read_peak_pressure()
    pk2, rm2 = grp.read_peak_pressure()
    assert np.array_equal(pk, pk2) and np.array_equal(rm, rm2)
    compare_map(pk2, o.get("peak"))
    compare_map(rm2, o.get("rms_amp"))
    full.close(); grp.close()


@pytest.mark.gpu
def test_gpu_step_phase_planes_rules():
    w = wl.random_domain(40, 36, 60, 6, seed=3, steps=4)
    a = bv.Simulation.from_workload(w, device="cuda:0")
    b = bv.Simulation.from_workload(w, device="cuda:0")
    a.step(2)
    for _ in range(2):
        b.step_phase(0)
        b.step_phase_planes(1, 40, 60); b.step_phase_planes(1, 0, 13); b.step_phase_planes(1, 13, 40)     # any order
        with pytest.raises(bv.BvfdtdError):
            b.step_phase_planes(1, 0, 5)              # the velocity pass is complete
        b.step_phase_planes(2, 0, 31)
        with pytest.raises(bv.BvfdtdError):
            b.step_phase(2)                           # a split pass is in progress
        with pytest.raises(bv.BvfdtdError):
            b.step_phase_planes(2, 20, 60)            # more planes than the grid has: an overlap
        b.step_phase_planes(2, 31, 60)
    assert b.step_index == 2
    for name in bv.FIELDS:
        assert np.array_equal(a.read_fields(name), b.read_fields(name)), name
    with pytest.raises(bv.BvfdtdError):
        b.step_phase_planes(1, 0, 60)                 # velocity before inject
    a.close(); b.close()


def _rank_worker(rank, world, port, q, overlap):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.random_domain(70, 45, 96, 6, seed=35, steps=30, waveform=1)
        w.rms_begin = 12
        r = slab.SlabRank(w, rank, world, "cuda:0", overlap=overlap)
        r.step(w.steps)
        out = {n: r.owned(r.sim.read_fields(n)) for n in ("vx", "vz", "sxx", "sxy", "rzz", "p")}
        pk, rm = r.sim.read_peak_pressure()
        out["peak"], out["rms"] = r.owned(pk), r.owned(rm)
        q.put((rank, out))
        dist.barrier()
        r.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.parametrize("overlap", [True, False])
def test_gpu_slab_ranks_as_two_processes(overlap):
    """SlabRank as a real torch.distributed job: two processes, one rank each, both on this box's one GPU, halo
    blocks staged through pinned host memory because gloo cannot move device memory (NCCL refuses two ranks on one
    device; the kernels of the two ranks never wait on one another, only the hosts do).  The stitched result is
    bit-identical to the undivided run and meets the oracle."""
    import torch.multiprocessing as mp
    from oracle import fdtd_oracle as orc
    w = wl.random_domain(70, 45, 96, 6, seed=35, steps=30, waveform=1)
    w.rms_begin = 12
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_worker, args=(r, 2, port, q, overlap)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    full = bv.Simulation.from_workload(w, device="cuda:0")
    full.step(w.steps)
    o = orc.Oracle.from_workload(w)
    o.step(w.steps)
    for n in ("vx", "vz", "sxx", "sxy", "rzz", "p"):
        got = np.concatenate([res[0][n], res[1][n]], axis=0)
        assert np.array_equal(got, full.read_fields(n)), n
        ref = o.get(n)
        assert np.linalg.norm(got - ref) <= 1e-4 * np.linalg.norm(ref), n
    pk, rm = full.read_peak_pressure()
    assert np.array_equal(np.concatenate([res[0]["peak"], res[1]["peak"]], axis=0), pk)
    assert np.array_equal(np.concatenate([res[0]["rms"], res[1]["rms"]], axis=0), rm)
    full.close()
