"""Phased-array refocusing (second half) -- orchestration only.

Every arithmetic step runs in the CUDA kernels behind the C ABI: the point-source run with the phasor
sensor (``bvfdtd_step`` + ``BVFDTD_FLAG_PHASOR``), the Rayleigh sums plane -> elements and elements ->
plane (``bvfdtd_rayleigh``) and the corrected phase programming (``bvfdtd_refocus_weights``).  This
module only builds index lists, gathers / copies arrays and passes pointers.

Geometry convention: the entry plane is the z plane k_s of the grid; its cell (i, j) sits at
(i dx, j dx, 0) of the transducer frame, the array's surface points at z < 0 (behind the plane).
``geom`` is a dict: nx, ny, nz, pml, dx, dt, f0, table, index_map, k_s, target_cell (i, j, k),
steps, window (steps of the phasor / rms window at the end of the run).
"""
from __future__ import annotations

import numpy as np

from . import binding as bv


def plane_cells(geom):
    """(n, 2) int array of the (i, j) of the entry plane's cells outside the PML mask."""
    P, nx, ny = geom["pml"], geom["nx"], geom["ny"]
    ii, jj = np.meshgrid(np.arange(P, nx - P), np.arange(P, ny - P))
    return np.stack([ii.ravel(), jj.ravel()], axis=1).astype(np.int64)


def _dev(a, dtype, device):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).to(device)


def refocus_weights(P, element, area, n_elem, f, u0=1.0, device="cuda:0"):
    """``bvfdtd_refocus_weights`` on host arrays: (w_pts complex64, delay float32, E complex64)."""
    import torch
    dev = torch.device(device)
    Pc = np.ascontiguousarray(P, dtype=np.complex64)
    re, im = _dev(Pc.real, np.float32, dev), _dev(Pc.imag, np.float32, dev)
    w, d, E = _refocus_weights_device(re, im, _dev(element, np.int32, dev), _dev(area, np.float32, dev), n_elem, f, u0, dev)
    torch.cuda.synchronize(dev)
    wn, En = w.cpu().numpy(), E.cpu().numpy()
    return wn[:, 0] + 1j * wn[:, 1], d.cpu().numpy(), En[:, 0] + 1j * En[:, 1]


def _refocus_weights_device(re, im, element, area, n_elem, f, u0, dev):
    import torch
    n = re.numel()
    w = torch.empty((n, 2), dtype=torch.float32, device=dev)
    d = torch.empty(n_elem, dtype=torch.float32, device=dev)
    E = torch.empty((n_elem, 2), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    bv._check(bv.lib().bvfdtd_refocus_weights(n, re.data_ptr(), im.data_ptr(), element.data_ptr(), area.data_ptr(), int(n_elem),
                                              float(f), float(u0), w.data_ptr(), d.data_ptr(), E.data_ptr(), stream),
              "bvfdtd_refocus_weights")
    return w, d, E


def _rayleigh_device(src_xyz, src_w, rcv_xyz, f, dev, want_source):
    import torch
    n_r = rcv_xyz.shape[0]
    out = torch.empty((4, n_r), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    bv._check(bv.lib().bvfdtd_rayleigh(src_xyz.shape[0], src_xyz.data_ptr(), src_w.data_ptr(), n_r, rcv_xyz.data_ptr(), float(f),
                                       1500.0, 1000.0, out[0].data_ptr(), out[1].data_ptr(),
                                       out[2].data_ptr() if want_source else None, out[3].data_ptr() if want_source else None,
                                       stream), "bvfdtd_rayleigh")
    return out


def back_propagate(geom, el_xyz, element, area, n_elem, u0=1.0, device="cuda:0"):
    """Point source at the target -> phasors on the entry plane -> field at the array's surface
    points -> corrected phase programming.  Returns dict(w_pts, delay, E, plane_ij)."""
    import torch
    dev = torch.device(device)
    g = geom
    nx, ny = g["nx"], g["ny"]
    ti, tj, tk = g["target_cell"]
    sim = bv.Simulation(nx, ny, g["nz"], g["pml"], g["dx"], g["dt"], g["table"], g["index_map"], g["f0"],
                        rms_begin=g["steps"] - g["window"], flags=bv.FLAG_PHASOR, device=dev)
    sim.set_source(np.array([ti + nx * (tj + ny * tk)], np.int64), np.ones(1, np.float32), np.zeros(1, np.float32), 1, g["f0"], 3)
    sim.step(g["steps"])
    re, im = sim.read_phasor_device()
    ij = plane_cells(g)
    sel = _dev(ij[:, 0] + nx * ij[:, 1], np.int64, dev)
    w_plane = torch.stack([re[g["k_s"]].reshape(-1)[sel], im[g["k_s"]].reshape(-1)[sel]], dim=1).contiguous()   # gather only
    sim.close()
    plane_xyz = _dev(np.stack([ij[:, 0] * g["dx"], ij[:, 1] * g["dx"], np.zeros(len(ij))], 1), np.float32, dev)
    pts = _dev(el_xyz, np.float32, dev)
    f_el = _rayleigh_device(plane_xyz, w_plane, pts, g["f0"], dev, want_source=False)
    w, d, E = _refocus_weights_device(f_el[0], f_el[1], _dev(element, np.int32, dev), _dev(area, np.float32, dev), n_elem, g["f0"], u0, dev)
    torch.cuda.synchronize(dev)
    wn, En = w.cpu().numpy(), E.cpu().numpy()
    return dict(w_pts=wn[:, 0] + 1j * wn[:, 1], delay=d.cpu().numpy(), E=En[:, 0] + 1j * En[:, 1], plane_ij=ij)


def forward(geom, el_xyz, w_pts, device="cuda:0"):
    """The array with the complex point weights `w_pts` -> Rayleigh field on the entry plane -> stress
    source -> FDTD run; returns the steady-state pressure amplitude map (nz, ny, nx) on the host."""
    import torch
    dev = torch.device(device)
    g = geom
    nx, ny = g["nx"], g["ny"]
    ij = plane_cells(g)
    plane_xyz = _dev(np.stack([ij[:, 0] * g["dx"], ij[:, 1] * g["dx"], np.zeros(len(ij))], 1), np.float32, dev)
    wc = np.ascontiguousarray(w_pts, dtype=np.complex64)
    w = _dev(wc.view(np.float32).reshape(-1, 2), np.float32, dev)
    out = _rayleigh_device(_dev(el_xyz, np.float32, dev), w, plane_xyz, g["f0"], dev, want_source=True)
    torch.cuda.synchronize(dev)
    amp, delay = out[2].cpu().numpy(), out[3].cpu().numpy()
    sim = bv.Simulation(nx, ny, g["nz"], g["pml"], g["dx"], g["dt"], g["table"], g["index_map"], g["f0"],
                        rms_begin=g["steps"] - g["window"], device=dev)
    sim.set_source(ij[:, 0] + nx * (ij[:, 1] + ny * g["k_s"]), amp, delay, 1, g["f0"], 3)
    sim.step(g["steps"])
    _, rms = sim.read_peak_pressure(peak=False, rms=True)
    sim.close()
    return rms
