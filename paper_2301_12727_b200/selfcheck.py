"""``python -m paper_2301_12727_b200.selfcheck [case ...]`` -- small runs of every launch plan of the hot path
through the C ABI, on one GPU: the default path, the dense sweep, the forced three-CTA velocity plan with a thick
PML, the fused single sweep (graph replay and kernel by kernel).  Each case checks that the fields are finite and
non-zero and that the plan is bit-identical to the plain two-pass, kernel-by-kernel run of the same workload.

It is also the target of the sanitizer runs recorded under ``profiles/`` (``compute-sanitizer --tool memcheck |
racecheck | synccheck python -m paper_2301_12727_b200.selfcheck``): small enough to finish under a sanitizer,
wide enough to touch every kernel instantiation.  No oracle, no CPU arithmetic: this is not a parity test
(those are ``tests/``)."""
from __future__ import annotations

import sys

import numpy as np

from . import binding as bv
from . import build
from . import workloads as wl


def _run(w, steps, flags=0, tuning=0, split=None):
    sim = bv.Simulation.from_workload(w, flags=flags, tuning=tuning)
    for n in (split or [steps]):
        sim.step(n)
    out = {n: sim.read_fields(n) for n in ("vx", "vz", "sxx", "syy", "sxy", "rxx", "ryz", "p")}
    out["peak"], out["rms"] = sim.read_peak_pressure()
    mode = sim.kernel_mode()
    cov = sim.fused_coverage()
    assert sim.padding_nonzeros() == 0, "a kernel wrote into the zero gaps of the layout"
    sim.close()
    return out, mode, cov


def _case(name, w, steps, flags=0, tuning=0, split=None, want_fused=False):
    ref, _, _ = _run(w, steps, tuning=bv.TUNE_NO_FUSED | bv.TUNE_NO_GRAPH | bv.TUNE_VEL_2CTA)
    got, mode, cov = _run(w, steps, flags=flags, tuning=tuning, split=split)
    assert all(np.isfinite(a).all() for a in got.values()), name
    assert float(np.abs(got["p"]).max()) > 0.0, name
    for n in ref:
        assert np.array_equal(ref[n], got[n]), (name, n)
    again, _, _ = _run(w, steps, flags=flags, tuning=tuning, split=split)      # run to run: no race shows
    for n in got:
        assert np.array_equal(again[n], got[n]), (name, n, "not deterministic")
    if want_fused:
        assert "fused" in mode and cov > 0.2, (name, mode, cov)
    print(f"selfcheck {name}: ok ({mode}; fused tile-plane fraction {cov:.2f})")


CASES = {
    "default": lambda: _case("default", wl.random_domain(64, 64, 64, 8, seed=11, steps=24, waveform=0), 24, split=[5, 19]),
    "dense": lambda: _case("dense", wl.blocky_domain(70, 30, 61, 5, seed=2, steps=16), 16, flags=bv.FLAG_DENSE),
    "three_cta": lambda: _case("three_cta", wl.random_domain(150, 60, 80, 24, seed=84, steps=12, waveform=1), 12,
                               tuning=bv.TUNE_VEL_3CTA),
    "stress16": lambda: _case("stress16", wl.blocky_domain(131, 45, 66, 6, seed=3, steps=12), 12, tuning=bv.TUNE_STRESS_16),
    "fused_graph": lambda: _case("fused_graph", wl.fluid_domain(150, 60, 70, 8, seed=1, steps=19), 19,
                                 tuning=bv.TUNE_FUSED, split=[3, 16], want_fused=True),
    "fused_plain": lambda: _case("fused_plain", wl.fluid_domain(131, 45, 66, 6, seed=2, steps=11, waveform=0), 11,
                                 tuning=bv.TUNE_FUSED | bv.TUNE_NO_GRAPH, want_fused=True),
}


def main(argv):
    build.build()
    names = argv or list(CASES)
    for n in names:
        CASES[n]()
    print("selfcheck: all cases passed")
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
