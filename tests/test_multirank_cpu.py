"""N > 1 host logic on CPU (gloo, world_size 2): bench.py's replicas-only aggregation.

The path does not shard ("replicas only"): every rank advances its own
replica and the whole-job rate is world * cells * steps / (max over ranks of the device time).
The only cross-rank operations are the barrier and the max reduction, exercised here."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    import bench
    rank, world = bench.dist_init("gloo")
    assert world == 2
    bench.barrier()
    ms_local = 10.0 if rank == 0 else 25.0          # rank 1 is the slow replica
    value, ms = bench.aggregate_rate(1000000, 50, ms_local, world, "cpu")
    assert abs(bench.reduce_max(float(rank), "cpu") - 1.0) < 1e-12
    bench.barrier()
    print(json.dumps({"rank": rank, "value": value, "ms": ms}))
""") % ROOT


def test_two_rank_aggregate_rate_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(out.strip().splitlines()[-1])
    import json
    res = [json.loads(o) for o in outs]
    expect = 2 * 1000000 * 50 / 25e-3 / 1e9         # both replicas' cell-steps over the slowest rank's time
    for r in res:
        assert abs(r["ms"] - 25.0) < 1e-9
        assert abs(r["value"] - expect) < 1e-9 * expect


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 1 exits 0 without output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
               MASTER_PORT="29534")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert p.returncode == 0, p.stderr[-2000:]
    assert p.stdout.strip() == ""
