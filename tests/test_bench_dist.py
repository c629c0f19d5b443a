"""bench.py's multi-rank plumbing ("replicas only"): world_size-2 gloo run on CPU.
The timed quantity is the MAX over ranks, the units are the SUM over ranks."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["TPCCLUS_ROOT"])
import bench
rank, world, local = bench.dist_setup(backend="gloo")
assert world == 2 and rank in (0, 1)
bench.dist_barrier(world)
ms, units = bench.dist_max_sum(10.0 + 5.0 * rank, 100.0 * (rank + 1), world)
bench.dist_barrier(world)
print(json.dumps({"rank": rank, "ms": ms, "units": units}))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo_max_time_sum_units():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), TPCCLUS_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    import json

    for o, _ in outs:
        r = json.loads(o.strip().splitlines()[-1])
        assert r["ms"] == 15.0 and r["units"] == 300.0, r


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.dist_max_sum(3.5, 7.0, 1) == (3.5, 7.0)
