"""Multi-process (gloo, world size 2) test of bench.py's replica plumbing: barrier, max-over-ranks time,
sum-over-ranks units, per-rank seeds, and the reference arm's rank gating.  Runs on CPU."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import bench
rank, local_rank, world = bench.env_rank()
dist = bench.dist_init(world, "gloo")
bench.dist_barrier(dist)
# rank r claims (r + 1) * 100 units in (r + 1) * 10 ms: the job is all units over the slowest rank's time
value, ms = bench.aggregate_throughput(dist, (rank + 1) * 100.0, (rank + 1) * 10.0)
mx = bench.dist_max(dist, float(rank))
sm = bench.dist_sum(dist, 1.0)
bench.dist_barrier(dist)
print(json.dumps(dict(rank=rank, world=world, value=value, ms=ms, mx=mx, sm=sm)))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _launch(code, world, extra_env=None, args=()):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, "-c", code, *args], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    return outs


def test_replica_aggregation_world2():
    outs = _launch(WORKER % dict(root=ROOT), 2)
    res = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    for d in res:
        assert d["world"] == 2
        assert d["ms"] == pytest.approx(20.0)                 # slowest rank
        assert d["value"] == pytest.approx(300.0 / 20e-3)     # all ranks' units over that time
        assert d["mx"] == pytest.approx(1.0) and d["sm"] == pytest.approx(2.0)


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.dist_init(1, "gloo") is None
    value, ms = bench.aggregate_throughput(None, 50.0, 5.0)
    assert ms == 5.0 and value == pytest.approx(1e4)


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the JSON line, rank 1 exits 0 silently."""
    code = ("import sys; sys.path.insert(0, %r); sys.argv = ['bench.py', '--impl', 'reference', '--workload', 'tiny', "
            "'--steps', '1', '--warmup', '0', '--gpus', '2']; import bench; sys.exit(bench.main())" % ROOT)
    outs = _launch(code, 2)
    line = json.loads(outs[0].strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["vs_baseline"] is None
    assert outs[1].strip() == ""
