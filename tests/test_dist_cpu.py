"""World-size-2 check of the benchmark's multi-rank host logic on CPU (gloo): distinct replica seeds, barrier,
max-over-ranks timing and the whole-job aggregate."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
from paper_2606_15622_b200 import dist as D, workloads
ws, rank, _ = D.world()
assert D.init("gloo") == 2
seed = D.replica_seed(3, rank)
cfg, st = workloads.cavity(n=8, ppc=10, seed=seed)
D.barrier()
ms = 10.0 + 5.0 * rank                       # rank 1 is the slow one
ms_max = D.max_over_ranks(ms)
assert ms_max == 15.0, ms_max
val = D.aggregate_throughput(st["x"].shape[0], 4, ms_max, ws)
assert abs(val - 2 * 640 * 4 / 15e-3) < 1e-6
chk = D.max_over_ranks(float(st["vx"][:16].astype("float64").sum()))
print("rank", rank, "seed", seed, "sum", float(st["vx"][:16].astype("float64").sum()), "max", chk)
D.shutdown()
'''


def test_two_rank_gloo(tmp_path):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    procs = []
    for rank in range(2):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE="2", RANK=str(rank),
                   LOCAL_RANK=str(rank))
        procs.append(subprocess.Popen([sys.executable, str(w), ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
    sums = [float(o.split("sum")[1].split()[0]) for o in outs]
    assert sums[0] != sums[1]                 # the two replicas really are different ensembles
