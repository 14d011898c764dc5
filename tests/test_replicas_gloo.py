"""N > 1 path of bench.py (replicas only) on CPU: world_size 2, gloo.  Each rank draws its own event
(seed + rank), there is no data-path collective, and the job's time is the max over ranks."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["VH_ROOT"])
import numpy as np
import torch
import torch.distributed as dist
import bench
from paper_1608_06577_b200 import inputs
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
prm, init, _ = inputs.config_3d(8, 8, 4, n_hot=3, seed=inputs.BASE_SEED + rank, radius=0.3, eta_half=0.1)
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))
val = bench.aggregate_value(prm["nx"] * prm["ny"] * prm["nz"], 4, world, ms * 1e-3)
sums = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
dist.all_gather(sums, torch.tensor([float(init["e"].sum())], dtype=torch.float64))
if rank == 0:
    print(json.dumps({"ms": ms, "value": val, "sums": [float(s) for s in sums]}))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_replicas_on_gloo(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), VH_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    import json

    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["ms"] == 15.0                                   # max over ranks, not rank 0's own 10 ms
    assert res["value"] == 8 * 8 * 4 * 4 * 2 / 15.0e-3         # both replicas' cell-updates over the slowest rank's time
    assert res["sums"][0] != res["sums"][1]                    # different events per rank (seed + rank)
