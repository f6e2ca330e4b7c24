"""The N > 1 path of bench.py on CPU: replicas only, one process per rank, `gloo`.

north_star fixes the hot path to one GPU without sharding or collectives, so `bench.py --gpus N`
runs N independent replicas; what the ranks share is the rendezvous, the barrier and the
max-over-ranks timing.  Two CPU processes exercise exactly that, with the oracle standing in for the
device (tests may call it): both replicas integrate the same seeded model and must agree bit for bit.
"""
import os
import subprocess
import sys
import textwrap
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent

WORKER = textwrap.dedent('''
    import os, sys, time, json, hashlib
    sys.path.insert(0, %r)
    import numpy as np
    import torch
    import torch.distributed as dist
    import bench
    import cn_workloads as W
    from oracle import OracleModel
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    desc = W.config4(n_cell=64, n_types=2)              # every rank: an independent replica
    o = OracleModel(desc)
    dist.barrier()
    o.run(2.0, 0.025)
    ms_local = 10.0 * (rank + 1)                        # rank 1 is the slow one
    value, ms_max = bench.aggregate(ms_local, len(desc["parent"]), 80, world, dist, device="cpu")
    h = hashlib.sha256(o.get_v().tobytes()).hexdigest()
    hs = [None] * world
    dist.all_gather_object(hs, h)
    if rank == 0:
        print(json.dumps({"value": value, "ms_max": ms_max, "same": len(set(hs)) == 1,
                          "n_node": len(desc["parent"]), "world": world}))
    dist.destroy_process_group()
''') % str(ROOT)


def test_two_replicas_barrier_and_max_over_ranks(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                          "--nproc-per-node", "2", "--master-addr", "127.0.0.1", "--master-port",
                          "29517", str(w)], capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["world"] == 2 and r["same"]
    assert r["ms_max"] == 20.0                                   # the slower rank sets the time
    assert abs(r["value"] - 2 * r["n_node"] * 80 / 20e-3) < 1e-6  # units of ALL ranks / max time
