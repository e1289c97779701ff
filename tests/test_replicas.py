"""World-size-2 CPU test (gloo) of the replicas-only multi-GPU plumbing: barrier, max over ranks, aggregate rate,
per-rank seeds.  The CUDA hot path has no collective; this is the host logic bench.py --gpus N relies on."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, %r)
import numpy as np
import workloads as wl
from paper_2403_07666_b200.replicas import Group, replica_seed
g = Group("gloo")
g.barrier()
t = 1.0 + 0.5 * g.rank                       # rank 1 is the slower replica
mx = g.max_over_ranks(t)
rate = g.aggregate_rate(1000.0, t)
w = wl.shrunk(0, 1, 1, 4)
s = wl.jc0_scale(replica_seed(w.seed, g.rank), w.geometry.n_rings, 0.01)
g.barrier()
print(json.dumps({"rank": g.rank, "world": g.world, "max": mx, "rate": rate, "s0": float(s[0])}))
g.close()
'''


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_over_gloo(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda d: d["rank"])
    assert [d["world"] for d in outs] == [2, 2]
    assert outs[0]["max"] == outs[1]["max"] == 1.5             # the slower rank sets the time
    assert abs(outs[0]["rate"] - 2 * 1000.0 / 1.5) < 1e-9      # whole-job units over the max time
    assert outs[0]["s0"] != outs[1]["s0"]                      # different seeded Jc0 perturbation per replica


def test_single_process_group_is_a_noop():
    from paper_2403_07666_b200.replicas import Group, env_rank, replica_seed
    assert env_rank() == (0, 0, 1) or "RANK" in os.environ
    g = Group()
    g.barrier()
    assert g.max_over_ranks(2.5) == 2.5 and g.aggregate_rate(10.0, 2.0) == 5.0
    assert replica_seed(1002, 0) == 1002 and replica_seed(1002, 3) == 1302
