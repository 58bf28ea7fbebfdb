"""The only cross-rank logic of the repository (replicas only): barrier
and the SUM / MAX reduction of per-rank work and time into one whole-job figure, exercised with
two CPU processes over gloo -- the path `bench.py --gpus N` takes under torchrun with NCCL."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
from paper_2410_19075_b200 import replicas
rank, ws = replicas.init("gloo")
assert ws == 2 and rank == int(os.environ["RANK"])
replicas.barrier()
# rank r processed (r + 1) * 1000 units in (r + 1) * 10 ms
units, ms_max, rate = replicas.aggregate((rank + 1) * 1000, (rank + 1) * 10.0, "cpu")
replicas.barrier()
print(json.dumps(dict(rank=rank, units=units, ms=ms_max, rate=rate)), flush=True)
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_two_rank_aggregate_over_gloo():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:                      # every rank sees the whole-job figure
        assert o["units"] == 3000.0     # SUM of the units
        assert o["ms"] == 20.0          # MAX of the times
        assert abs(o["rate"] - 3000.0 / 20e-3) < 1e-6
    assert sorted(o["rank"] for o in outs) == [0, 1]


def test_single_process_is_the_identity():
    from paper_2410_19075_b200 import replicas
    env = {k: os.environ.pop(k) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE") if k in os.environ}
    try:
        assert replicas.world() == (0, 0, 1)
        replicas.barrier()                       # no process group: a no-op
        assert replicas.aggregate(500, 25.0) == (500.0, 25.0, 500.0 / 25e-3)
    finally:
        os.environ.update(env)
