"""GPU tests of the runtime around the kernels: CUDA-graph replay of bvfdtd_step, the device guard of the entry
points, source lists longer than the workspace's source region."""
import numpy as np
import pytest

from oracle import fdtd_oracle as orc
from paper_2301_12727_b200 import build as bv_build
from paper_2301_12727_b200 import workloads as wl

from test_gpu_parity import compare_map, compare_state

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bv():
    bv_build.build()
    from paper_2301_12727_b200 import binding
    return binding


def _same(a, b, bv):
    for n in bv.FIELDS:
        assert np.array_equal(a.read_fields(n), b.read_fields(n)), n
    pa, ra = a.read_peak_pressure()
    pb, rb = b.read_peak_pressure()
    assert np.array_equal(pa, pb) and np.array_equal(ra, rb)
    assert a.step_index == b.step_index and a.rms_count == b.rms_count


@pytest.mark.parametrize("wave", [0, 1])
def test_graph_replay_is_bit_identical(bv, wave):
    """bvfdtd_step(n) replays captured CUDA graphs (8 steps per launch, then single steps), one graph per
    sensor regime; the injection takes the step index from a device counter.  Across the window edges
    (peak on at 5, rms on at 21, both off at 47) and over several calls it must equal the kernel-by-kernel
    path bit for bit, and the oracle within the usual bars."""
    w = wl.random_domain(70, 37, 44, 6, seed=21, steps=61, waveform=wave)
    w.peak_begin, w.rms_begin, w.sensor_end = 5, 21, 47
    g = bv.Simulation.from_workload(w)
    assert g.mode_bits() & bv.MODE_GRAPH
    plain = bv.Simulation.from_workload(w, tuning=bv.TUNE_NO_GRAPH)
    assert not plain.mode_bits() & bv.MODE_GRAPH
    one = bv.Simulation.from_workload(w)
    g.step(3); g.step(30); g.step(1); g.step(27)          # 3 + 30 + 1 + 27 = 61
    plain.step(61)
    for _ in range(61):
        one.step(1)                                        # n = 1 never uses a graph
    _same(g, plain, bv)
    _same(g, one, bv)
    o = orc.Oracle.from_workload(w)
    o.step(61)
    compare_state(g, o)
    peak, rms = g.read_peak_pressure()
    compare_map(peak, o.get("peak"))
    compare_map(rms, o.get("rms_amp"))
    assert g.rms_count == o.rms_count == 47 - 21
    # a new source list invalidates the graphs: keep stepping with half the cells
    for s in (g, plain):
        s.set_source(w.src_cell[::2], w.src_amp[::2], w.src_delay[::2], w.waveform, w.f_src, w.n_cycles)
        s.step(9)
    _same(g, plain, bv)
    for s in (g, plain, one):
        s.close()


def test_source_list_longer_than_the_workspace_region(bv):
    """the workspace holds up to 4 nx ny source cells; a longer list moves to a library-owned allocation"""
    nx, ny, nz, P = 40, 24, 40, 4
    w = wl.random_domain(nx, ny, nz, P, seed=5, steps=30, waveform=1)
    rng = np.random.default_rng(3)
    k, j, i = np.meshgrid(np.arange(P, nz - P), np.arange(P, ny - P), np.arange(P, nx - P), indexing="ij")
    cells = (i + nx * (j + ny * k)).ravel().astype(np.int64)
    cells = np.sort(rng.permutation(cells)[:4 * nx * ny + 500])
    assert cells.size > 4 * nx * ny
    w.src_cell = cells
    w.src_amp = rng.uniform(0.5, 1.5, cells.size).astype(np.float32)
    w.src_delay = (rng.uniform(0, 4, cells.size) * w.dt).astype(np.float32)
    sim = bv.Simulation.from_workload(w)
    sim.step(30)
    o = orc.Oracle.from_workload(w)
    o.step(30)
    compare_state(sim, o)
    # back to a short list (the owned copy is released), then none
    sim.set_source(cells[:10], w.src_amp[:10], w.src_delay[:10], w.waveform, w.f_src, w.n_cycles)
    o.set_source(cells[:10], w.src_amp[:10], w.src_delay[:10], w.waveform, w.f_src, w.n_cycles)
    sim.step(12); o.step(12)
    compare_state(sim, o)
    sim.close()


def test_context_on_a_device_that_is_not_current(bv):
    """every entry point runs on the device that owns the workspace, whatever device is current"""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    w = wl.random_domain(48, 40, 44, 6, seed=99, steps=20, waveform=1)
    torch.cuda.set_device(0)
    sim = bv.Simulation.from_workload(w, device="cuda:1")
    ref = bv.Simulation.from_workload(w, device="cuda:0")
    assert torch.cuda.current_device() == 0
    sim.step(20); ref.step(20)
    _same(sim, ref, bv)
    assert torch.cuda.current_device() == 0
    sim.close(); ref.close()
