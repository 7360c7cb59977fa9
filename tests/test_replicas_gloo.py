"""World-size-2 `gloo` test of the only multi-process logic this path has (replicas only):
rendezvous from the torchrun environment, the barrier, max-over-ranks of the elapsed time, sum-over-ranks of the
units, one scene seed per replica.  Runs on CPU; the data plane has no collective to test."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
from paper_2306_01301_b200 import replicas
rank, local_rank, ws = replicas.init("gloo")
assert ws == 2 and rank == int(os.environ["RANK"]) and local_rank == int(os.environ["LOCAL_RANK"])
replicas.barrier()
ms, units = replicas.aggregate(10.0 + 5.0 * rank, 1000.0 * (rank + 1))
assert ms == 15.0 and units == 3000.0, (ms, units)          # max over ranks, sum over ranks
seeds = [replicas.replica_seed(3, r) for r in range(ws)]
assert seeds[0] == 3 and len(set(seeds)) == ws              # rank 0 plans the named config, the others their own scene
replicas.barrier()
replicas.shutdown()
print("rank", rank, "ok", ms, units)
"""


def test_two_replicas_over_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER.format(root=ROOT)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for rank, p in enumerate(procs):
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        assert f"rank {rank} ok 15.0 3000.0" in out


def test_single_process_needs_no_group():
    from paper_2306_01301_b200 import replicas
    env = {k: os.environ.pop(k) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE") if k in os.environ}
    try:
        assert replicas.world() == (0, 0, 1)
        assert replicas.aggregate(7.0, 11.0) == (7.0, 11.0)
        replicas.barrier()
    finally:
        os.environ.update(env)
