"""The N > 1 path of bench.py (independent replicas: barrier + max-over-ranks, no data-path
collective) with world_size 2 on the gloo backend, CPU only."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
from paper_1808_10375_b200.replicas import ReplicaGroup
g = ReplicaGroup("gloo")
g.barrier()
ms = 10.0 + 5.0 * g.rank                      # rank 1 is the slow one
mx = g.max_over_ranks(ms)
g.barrier()
print(json.dumps({"rank": g.rank, "world": g.world, "seed": g.seed, "max": mx, "value": g.aggregate(1000, 4, mx)}), flush=True)
g.close()
""" % ROOT


def _free_port():
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_replicas_gloo():
    import json
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(r), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=120)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert [d["rank"] for d in outs] == [0, 1] and all(d["world"] == 2 for d in outs)
    assert [d["seed"] for d in outs] == [0, 1]                   # each replica its own data set
    assert all(d["max"] == 15.0 for d in outs)                   # the slowest rank's time, on every rank
    assert all(abs(d["value"] - 2 * 1000 * 4 / 15e-3) < 1e-6 for d in outs)   # whole-job aggregate, weak scaling


def test_single_process_needs_no_process_group():
    from paper_1808_10375_b200.replicas import ReplicaGroup
    env = {k: os.environ.pop(k) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK") if k in os.environ}
    try:
        g = ReplicaGroup("gloo")
        assert g.world == 1 and g.max_over_ranks(3.5) == 3.5
        g.barrier()
        assert g.aggregate(10, 2, 4.0) == 10 * 2 / 4e-3
        g.close()
    finally:
        os.environ.update(env)
