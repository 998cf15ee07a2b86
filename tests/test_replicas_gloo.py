"""N > 1 path on CPU: world_size-2 gloo.  The deposition does not shard (DESIGN.md "Multi-GPU":
replicas only), so the only multi-rank logic is the bookkeeping of bench.py --gpus N:
barrier, MAX of the per-rank times, SUM of the per-rank units, per-replica seeds."""
import os
import socket
import subprocess
import sys

import numpy as np

from paper_1908_02219_b200 import replicas as R
from paper_1908_02219_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import sys, json
sys.path.insert(0, %(root)r)
from paper_1908_02219_b200 import replicas as R
rank, local_rank, world = R.init("gloo")
R.barrier()
ms, units = R.combine(10.0 + 5.0 * rank, 1000.0 * (rank + 1))
R.barrier()
print(json.dumps({"rank": rank, "world": world, "ms": ms, "units": units,
                  "seed": R.replica_seed(0, rank)}), flush=True)
R.finalize()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_combine_world2_gloo():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % {"root": ROOT}], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["world"] == 2
        assert o["ms"] == 15.0          # MAX over ranks
        assert o["units"] == 3000.0     # SUM over ranks
    assert outs[0]["seed"] != outs[1]["seed"]


def test_combine_single_process_identity():
    assert R.combine(3.5, 7.0) == (3.5, 7.0)
    assert R.env_rank()[2] >= 1


def test_replicas_get_different_markers():
    import dataclasses
    cfg = W.scaled(W.CONFIGS["cfg0"], 1000)
    a = W.generate(dataclasses.replace(cfg, seed=R.replica_seed(cfg.seed, 0)))
    b = W.generate(dataclasses.replace(cfg, seed=R.replica_seed(cfg.seed, 1)))
    assert not np.array_equal(a["s"], b["s"])
    assert abs(a["s"].mean() - b["s"].mean()) < 0.05
