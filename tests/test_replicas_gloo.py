"""N > 1 path on CPU: two gloo ranks run the bench protocol of "replicas only" -- distinct
seeds per rank, SUM of trials over MAX of time -- and bench.py's reference arm leaves non-zero ranks idle."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
from paper_1509_04692_b200.replicas import Replicas
from paper_1509_04692_b200 import workloads as wl
R = Replicas(backend="gloo")
w = wl.pentagons(8, seed=R.seed)
R.barrier()
trials, seconds = 1000.0 * (R.rank + 1), 0.5 * (R.rank + 1)      # rank 1 is the slow one
value, trials_all, t_max = R.aggregate(trials, seconds)
R.barrier()
print(json.dumps(dict(rank=R.rank, world=R.world, seed=R.seed, q0=float(w.quat4[0, 0]), value=value, trials=trials_all, t=t_max)))
R.close()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_gloo_ranks_aggregate_like_bench():
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(r), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER.format(root=ROOT)], env=env, stdout=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, _ = p.communicate(timeout=300)
        assert p.returncode == 0
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert [d["seed"] for d in outs] == [1, 2] and outs[0]["q0"] != outs[1]["q0"]      # independent replicas
    for d in outs:
        assert d["world"] == 2 and d["trials"] == 3000.0 and d["t"] == 1.0 and d["value"] == 3000.0


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, WORLD_SIZE="2", RANK="1", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "1", "--config", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
