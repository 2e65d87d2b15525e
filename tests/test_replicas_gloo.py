"""N > 1 path of bench.py ("replicas only") on CPU: world_size 2, gloo backend.

What crosses ranks in the bench is the barrier and the MAX over ranks of the timed duration; the whole-job value is
world x (units per rank) / max time.  Two real processes rendezvous on 127.0.0.1.
"""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
from paper_2510_16721_b200.replicas import Ranks
r = Ranks("gloo")
assert r.world == 2 and r.dist is not None
r.barrier()
t = [0.25, 0.40][r.rank]                      # this rank's "device time"
mx = r.max_over_ranks(t)
v = r.throughput(1000.0, t)
r.barrier()
print(json.dumps({"rank": r.rank, "max": mx, "value": v}))
r.close()
""" % ROOT


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_two_rank_max_and_whole_job_value():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["max"] == 0.40                       # both ranks see the slower rank's time
        assert abs(o["value"] - 2 * 1000.0 / 0.40) < 1e-9
    assert sorted(o["rank"] for o in outs) == [0, 1]


def test_single_rank_needs_no_process_group():
    from paper_2510_16721_b200.replicas import Ranks
    env = {k: os.environ.pop(k) for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK") if k in os.environ}
    try:
        r = Ranks("gloo")
        assert r.world == 1 and r.dist is None
        assert r.max_over_ranks(1.5) == 1.5
        assert r.throughput(10.0, 2.0) == 5.0
        r.barrier()
        r.close()
    finally:
        os.environ.update(env)
