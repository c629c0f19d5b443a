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


def test_bare_gpus_flag_launches_the_ranks_itself():
    """`python bench.py --gpus 2` without torchrun's environment starts the two ranks itself (one process per
    GPU through torch.distributed.run on 127.0.0.1).  Exercised on CPU with the reference arm (rank 0 times the
    oracle on config 0 and prints the line, rank 1 exits 0 without work)."""
    import json

    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference",
                        "--config", "0", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [json.loads(x) for x in p.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2
    assert lines[0]["value"] > 0 and lines[0]["cpu_baseline"]["kind"] == "oracle"
