"""Multi-process host logic of bench.py (no GPU): the path does not shard without an all-to-all (DESIGN.md
"Multi-GPU": replicas only), so the only distributed code is the timing aggregation — max over ranks of the
device time, sum over ranks of the work.  Covered here with world_size 2 over gloo on 127.0.0.1."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
ms, units = bench.aggregate(10.0 + 5.0 * rank, 1000.0 * (rank + 1), dist)
r, lr, w = bench.dist_env()
dist.barrier()
print(json.dumps({"rank": rank, "ms": ms, "units": units, "env": [r, lr, w]}))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_aggregate_world_size_2_gloo():
    import json
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 15.0            # max over ranks
        assert o["units"] == 3000.0       # whole-job work
        assert o["env"] == [o["rank"], o["rank"], 2]


def test_aggregate_single_process():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.0, 7.0, None) == (3.0, 7.0)


def test_reference_arm_other_ranks_exit_without_work():
    """`bench.py --impl reference` under torchrun: rank 0 alone runs the oracle, the others exit 0 silently."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], env=env,
                       capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
