"""N > 1 path of bench.py (replicas only): world_size-2 gloo run on CPU of the rank plumbing --
environment parsing, barrier, max-over-ranks of the step time and the whole-job aggregate."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
from paper_2607_06523_b200 import replicas
rank, world, local = replicas.env_rank()
assert replicas.init("gloo")
replicas.barrier()
ms = 2.0 + rank                      # rank 1 is the slow one
mx = replicas.max_over_ranks(ms)
agg = replicas.aggregate_throughput(1000.0, mx, world)
replicas.barrier()
print(json.dumps({"rank": rank, "world": world, "local": local, "max_ms": mx, "agg": agg}))
import torch.distributed as dist
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_rank_gloo_max_and_aggregate(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    import json
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for r, o in enumerate(outs):
        assert o["rank"] == r and o["world"] == 2 and o["local"] == r
        assert o["max_ms"] == 3.0                      # the slowest rank's time on every rank
        assert abs(o["agg"] - 1000.0 * 2 / 3e-3) < 1e-6


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    from paper_2607_06523_b200 import replicas
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.env_rank() == (0, 1, 0)
    assert replicas.init("gloo") is False
    assert replicas.max_over_ranks(1.5) == 1.5
    assert replicas.aggregate_throughput(10.0, 2.0, 1) == 5000.0
