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


SLAB_WORKER = r'''
import sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch
from paper_2606_15622_b200 import dist as D, workloads
ws, rank, _ = D.world()
assert D.init("gloo") == 2
cfg, st = workloads.cavity(n=12, ppc=15, seed=4)
ny = cfg["ny"]
bounds = D.slab_row_bounds(ny, ws)
assert bounds == [0, 6, 12]
rng = np.random.default_rng(9)
row = rng.integers(0, ny, size=st["x"].shape[0])          # destination rows after a (made-up) streaming step
held = rng.integers(0, ws, size=row.shape[0])             # which rank holds each particle before the exchange
def partitioned(r):
    idx = np.nonzero(held == r)[0]
    dest = np.searchsorted(np.array(bounds), row[idx], side="right") - 1
    order = idx[np.argsort(dest, kind="stable")]           # what fp_slab_partition does on the device
    starts = [0] + list(np.cumsum(np.bincount(dest, minlength=ws)))
    return {k: torch.from_numpy(st[k][order].copy()) for k in D.FIELDS}, [int(v) for v in starts]
mine, starts = partitioned(rank)
got, counts = D.exchange_slab_particles(mine, starts)
both = [partitioned(r) for r in range(ws)]
want = D.exchange_in_process([b[0] for b in both], [b[1] for b in both])[rank]
for k in D.FIELDS:
    assert torch.equal(got[k], want[k]), k
assert counts == [both[r][1][rank + 1] - both[r][1][rank] for r in range(ws)]
# every received particle belongs to this rank's rows, and nothing is lost over the two ranks
pid = got["pid"].numpy()
lookup = {int(p): int(r) for p, r in zip(st["pid"], row)}
assert all(bounds[rank] <= lookup[int(p)] < bounds[rank + 1] for p in pid)
tot = D.max_over_ranks(0.0)                               # keeps the ranks in step
n_all = torch.tensor([pid.shape[0]], dtype=torch.int64)
torch.distributed.all_reduce(n_all)
assert int(n_all) == st["x"].shape[0]
print("rank", rank, "received", pid.shape[0], "from", counts)
D.shutdown()
'''


def test_slab_exchange_two_rank_gloo(tmp_path):
    """NEXT-4 host logic: the all-to-all of partitioned particles hands every rank the particles of its rows, in ascending
    source order, identical to the in-process exchange the one-GPU slab test uses (tests/test_gpu_slab.py)."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    w = tmp_path / "slab_worker.py"
    w.write_text(SLAB_WORKER)
    procs = []
    for rank in range(2):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE="2", RANK=str(rank),
                   LOCAL_RANK=str(rank))
        procs.append(subprocess.Popen([sys.executable, str(w), ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o


def test_slab_row_bounds():
    import pytest
    from paper_2606_15622_b200 import dist as D
    assert D.slab_row_bounds(48, 1) == [0, 48]
    assert D.slab_row_bounds(48, 3) == [0, 16, 32, 48]
    b = D.slab_row_bounds(50, 8)
    assert b[0] == 0 and b[-1] == 50 and all(6 <= b[i + 1] - b[i] <= 7 for i in range(8))
    with pytest.raises(ValueError):
        D.slab_row_bounds(4, 5)
