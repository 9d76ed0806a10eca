"""z-slab decomposition of one simulation over several GPUs.

Host-side orchestration only: every pass runs in the CUDA kernels behind ``bvfdtd_step_phase``; a
halo exchange is a plain copy of contiguous plane blocks (``bvfdtd_plane_span``) between the
workspaces of two z neighbours -- point-to-point, no collective (the peak / rms maps are cell-local).

* ``partition`` / ``local_box`` / ``local_workload``: who owns which planes, the local index map
  (owned planes + two halo planes on every interface), the local source list.
* ``halo_plan``: the byte ranges sent and received on each interface.
* ``SlabRank``: one rank of a ``torch.distributed`` job (NCCL between GPUs; the exchange itself is
  backend-agnostic and is tested on CPU tensors with gloo).
* ``SlabGroup``: all slabs of a run inside ONE process on one GPU, stepped in lock step with
  device-to-device copies -- the single-GPU check that the decomposition reproduces the undivided
  run bit for bit.  It is a test vehicle, not a way to run faster.

Per step (include/bvfdtd.h): inject -> exchange the six stresses -> velocity pass -> exchange the
three velocities -> stress + sensor pass.  On config 2 a face carries 2 planes x 9 arrays =
6.5 MB per step.
"""
from __future__ import annotations

import ctypes as C
import dataclasses

import numpy as np

from . import binding as bv

HALO = 2                       # the 4th-order staggered differences reach two planes (reading P1)
STRESS = ("sxx", "syy", "szz", "sxy", "sxz", "syz")
VELOCITY = ("vx", "vy", "vz")
FLAG_ZLO_OPEN, FLAG_ZHI_OPEN = 8, 16


def partition(nz: int, world: int, pml: int):
    """Owned z ranges [(z0, z1), ...], as even as possible; every local box (owned + halos) must
    satisfy the library's minimum extent 2 pml + 8."""
    if world < 1:
        raise ValueError("world must be >= 1")
    base, rem = divmod(nz, world)
    out, z = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((z, z + n))
        z += n
    for r, (z0, z1) in enumerate(out):
        lo, hi = local_halos(r, world)
        if (z1 - z0) + lo + hi < 2 * pml + 8 or z1 - z0 < HALO:
            raise ValueError(f"slab {r} of {world} is too thin for nz = {nz}, pml = {pml}")
    return out


def local_halos(rank: int, world: int):
    """(halo planes below, halo planes above) of this rank's box."""
    return (HALO if rank > 0 else 0), (HALO if rank < world - 1 else 0)


def local_flags(rank: int, world: int) -> int:
    return (FLAG_ZLO_OPEN if rank > 0 else 0) | (FLAG_ZHI_OPEN if rank < world - 1 else 0)


def local_workload(w, rank: int, world: int):
    """The rank's box as a Workload: planes [z0 - lo, z1 + hi) of the index map, the sources that
    lie in its OWNED planes (a halo plane's stresses arrive from their owner, already injected)."""
    z0, z1 = partition(w.nz, world, w.pml)[rank]
    lo, hi = local_halos(rank, world)
    zb0, zb1 = z0 - lo, z1 + hi
    plane = w.nx * w.ny
    k = w.src_cell // plane
    keep = (k >= z0) & (k < z1)
    cells = w.src_cell[keep] - zb0 * plane
    lw = dataclasses.replace(w, name=f"{w.name}_slab{rank}of{world}", nz=zb1 - zb0,
                             index_map=np.ascontiguousarray(w.index_map[zb0:zb1]),
                             src_cell=cells.astype(np.int64), src_amp=w.src_amp[keep], src_delay=w.src_delay[keep])
    return lw, dict(z0=z0, z1=z1, lo=lo, hi=hi)


def plane_span(nx, ny, nz, pml, field, k, n_planes):
    g = bv.Grid(nx, ny, nz, pml)
    off, nb = C.c_size_t(0), C.c_size_t(0)
    bv._check(bv.lib().bvfdtd_plane_span(C.byref(g), bv.FIELD_ID[field], int(k), int(n_planes), C.byref(off), C.byref(nb)),
              "bvfdtd_plane_span")
    return off.value, nb.value


def halo_plan(nx, ny, nz_local, pml, lo, hi, fields):
    """Per field the (offset, bytes) blocks of the workspace: what goes to / comes from the lower
    neighbour (send_lo = my two lowest owned planes, recv_lo = my lower halo) and the upper one."""
    plan = []
    for f in fields:
        e = {"field": f}
        if lo:
            e["send_lo"] = plane_span(nx, ny, nz_local, pml, f, lo, HALO)
            e["recv_lo"] = plane_span(nx, ny, nz_local, pml, f, 0, HALO)
        if hi:
            e["send_hi"] = plane_span(nx, ny, nz_local, pml, f, nz_local - hi - HALO, HALO)
            e["recv_hi"] = plane_span(nx, ny, nz_local, pml, f, nz_local - hi, HALO)
        plan.append(e)
    return plan


def _view(ws, span):
    return ws[span[0]:span[0] + span[1]]


def exchange_distributed(ws, plan, rank, world, group=None):
    """One halo exchange of the fields in `plan` with both z neighbours (torch.distributed
    point-to-point, batched; `ws` is the rank's workspace as a flat uint8 tensor).  With a backend
    that cannot move device memory (gloo) the blocks are staged through pinned host buffers."""
    import torch
    import torch.distributed as dist
    staged = ws.is_cuda and dist.get_backend(group) != "nccl"
    ops, back = [], []

    def buf(span, recv):
        v = _view(ws, span)
        if not staged:
            return v
        h = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
        if recv:
            back.append((v, h))
        else:
            h.copy_(v, non_blocking=True)
        return h

    for e in plan:
        if "send_lo" in e:
            ops.append(dist.P2POp(dist.isend, buf(e["send_lo"], False), rank - 1, group))
            ops.append(dist.P2POp(dist.irecv, buf(e["recv_lo"], True), rank - 1, group))
        if "send_hi" in e:
            ops.append(dist.P2POp(dist.isend, buf(e["send_hi"], False), rank + 1, group))
            ops.append(dist.P2POp(dist.irecv, buf(e["recv_hi"], True), rank + 1, group))
    if staged:
        torch.cuda.current_stream(ws.device).synchronize()      # the device-to-host copies of the send blocks
    if ops:
        for r in dist.batch_isend_irecv(ops):
            r.wait()
    for v, h in back:
        v.copy_(h, non_blocking=True)


def exchange_local(workspaces, plans):
    """The same exchange between slabs that live in one process (device-to-device copies)."""
    for r in range(len(workspaces) - 1):
        for e_lo, e_hi in zip(plans[r], plans[r + 1]):
            _view(workspaces[r + 1], e_hi["recv_lo"]).copy_(_view(workspaces[r], e_lo["send_hi"]))
            _view(workspaces[r], e_lo["recv_hi"]).copy_(_view(workspaces[r + 1], e_hi["send_lo"]))


class _Slab:
    def __init__(self, w, rank, world, device, flags=0):
        self.rank, self.world = rank, world
        self.w, self.meta = local_workload(w, rank, world)
        lw = self.w
        self.sim = bv.Simulation.from_workload(lw, device=device, flags=flags | local_flags(rank, world))
        lo, hi = self.meta["lo"], self.meta["hi"]
        self.plan_s = halo_plan(lw.nx, lw.ny, lw.nz, lw.pml, lo, hi, STRESS)
        self.plan_v = halo_plan(lw.nx, lw.ny, lw.nz, lw.pml, lo, hi, VELOCITY)

    def owned(self, a):
        """The owned planes of a local (nz, ny, nx) array."""
        lo = self.meta["lo"]
        return a[lo:lo + (self.meta["z1"] - self.meta["z0"])]


def split_ranges(nz_local, lo, hi):
    """(interior, boundary) plane ranges of a pass: a pass at plane k reads planes k-2 .. k+2 of the exchanged
    arrays, so the planes [lo + 2, nz - hi - 2) read no halo plane and can run while the exchange is in flight;
    the owned planes next to an interface run after it.  The halo planes themselves ([0, lo) and [nz - hi, nz)) are
    in the boundary ranges too: what a pass computes there is overwritten by the next exchange, but every plane must
    be swept for the pass to complete."""
    i0 = lo + HALO if lo else 0
    i1 = nz_local - hi - HALO if hi else nz_local
    if i1 <= i0:                       # a slab too thin to have such planes: everything runs after the exchange
        return (0, 0), [(0, nz_local)]
    boundary = []
    if i0 > 0:
        boundary.append((0, i0))
    if i1 < nz_local:
        boundary.append((i1, nz_local))
    return (i0, i1), boundary


class SlabRank(_Slab):
    """One rank of a torch.distributed z-slab run (one process per GPU).  Per step, with overlap:

        inject -> [ exchange of the six stresses  ||  velocity pass on the planes that read no halo ]
               -> velocity pass on the planes next to the interfaces
               -> [ exchange of the three velocities  ||  stress pass on the planes that read no halo ]
               -> stress pass on the planes next to the interfaces

    The passes run on the simulation's stream, the exchanges on a side stream of the same device; events order
    them (the exchange waits for what it sends, the boundary planes wait for what was received)."""

    def __init__(self, w, rank, world, device, group=None, flags=0, overlap=True):
        import torch
        self._torch = torch
        torch.cuda.set_device(torch.device(device))     # NCCL point-to-point runs on the current device
        super().__init__(w, rank, world, device, flags)
        self.group = group
        self.overlap = overlap
        self.main = self.sim._stream
        self.side = torch.cuda.Stream(device=self.sim.device)
        self.interior, self.boundary = split_ranges(self.w.nz, self.meta["lo"], self.meta["hi"])

    def _exchange(self, plan):
        torch = self._torch
        self.side.wait_stream(self.main)                # what is sent was written on the main stream
        with torch.cuda.stream(self.side):
            exchange_distributed(self.sim.workspace, plan, self.rank, self.world, self.group)

    def _pass(self, phase, plan):
        if not self.overlap or self.world == 1:
            self._exchange(plan)
            self.main.wait_stream(self.side)
            self.sim.step_phase(phase)
            return
        # the interior planes are enqueued first; the exchange then runs beside them
        mark = self._torch.cuda.Event()
        mark.record(self.main)                          # everything the exchange sends is complete here
        i0, i1 = self.interior
        if i1 > i0:
            self.sim.step_phase_planes(phase, i0, i1)
        self.side.wait_event(mark)
        with self._torch.cuda.stream(self.side):
            exchange_distributed(self.sim.workspace, plan, self.rank, self.world, self.group)
        self.main.wait_stream(self.side)
        for k0, k1 in self.boundary:
            self.sim.step_phase_planes(phase, k0, k1)

    def step(self, n=1):
        for _ in range(int(n)):
            self.sim.step_phase(0)
            self._pass(1, self.plan_s)
            self._pass(2, self.plan_v)

    def close(self):
        self.sim.close()


class SlabGroup:
    """All slabs of a run in one process on one device, stepped in lock step (a correctness vehicle)."""

    def __init__(self, w, n_slabs, device="cuda:0", flags=0, split=False):
        self.w = w
        self.slabs = [_Slab(w, r, n_slabs, device, flags) for r in range(n_slabs)]
        self.split = split          # run every pass the way SlabRank overlaps it: interior planes, exchange, boundary planes

    def _pass(self, phase, ws, plans):
        if not self.split:
            exchange_local(ws, plans)
            for s in self.slabs:
                s.sim.step_phase(phase)
            return
        ranges = [split_ranges(s.w.nz, s.meta["lo"], s.meta["hi"]) for s in self.slabs]
        for s, ((i0, i1), _) in zip(self.slabs, ranges):
            if i1 > i0:
                s.sim.step_phase_planes(phase, i0, i1)
        exchange_local(ws, plans)
        for s, (_, boundary) in zip(self.slabs, ranges):
            for k0, k1 in boundary:
                s.sim.step_phase_planes(phase, k0, k1)

    def step(self, n=1):
        ws = [s.sim.workspace for s in self.slabs]
        ps = [s.plan_s for s in self.slabs]
        pv = [s.plan_v for s in self.slabs]
        for _ in range(int(n)):
            for s in self.slabs:
                s.sim.step_phase(0)
            self._pass(1, ws, ps)
            self._pass(2, ws, pv)

    def read_fields(self, name):
        return np.concatenate([s.owned(s.sim.read_fields(name)) for s in self.slabs], axis=0)

    def read_peak_pressure(self):
        pk, rm = [], []
        for s in self.slabs:
            p, r = s.sim.read_peak_pressure()
            pk.append(s.owned(p)); rm.append(s.owned(r))
        return np.concatenate(pk, axis=0), np.concatenate(rm, axis=0)

    def close(self):
        for s in self.slabs:
            s.sim.close()
