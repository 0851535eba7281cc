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


TRANSPOSE_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch
import torch.distributed as dist
from paper_1810_12707_b200 import dist as D
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
N, nf = 16, 3
nyc, nxp = D.compact_extents(N)
def ident(f, z, y, x):            # a unique value per (field, z, ky, kx)
    return ((f * N + z) * nyc + y) * nxp + x + 0.5j
full = np.fromfunction(lambda f, z, y, x: ident(f, z, y, x), (nf, N, nyc, nxp), dtype=np.complex128)
(ya, yb), (za, zb) = D.ranges(N, world, rank)
ok = True
# bricks -> slabs: I hold all z of my ky range; afterwards all ky of my z range
work = np.full((nf, N, nyc, nxp), np.nan + 0j)
work[:, :, ya:yb, :] = full[:, :, ya:yb, :]      # includes my own block (my ky x my z), which is not exchanged
sc, rc = D.split_counts(N, world, rank, D.BRICKS_TO_SLABS, nf)
send = torch.from_numpy(D.pack_host(work, N, world, rank, D.BRICKS_TO_SLABS))
assert send.numel() == sum(sc)
recv = torch.empty(sum(rc), dtype=torch.float64)
D.all_to_all(recv, send, rc, sc)
D.unpack_host(work, recv.numpy(), N, world, rank, D.BRICKS_TO_SLABS)
ok &= bool(np.array_equal(work[:, za:zb], full[:, za:zb]))
# slabs -> bricks: the way back
work2 = np.full((nf, N, nyc, nxp), np.nan + 0j)
work2[:, za:zb] = full[:, za:zb]
sc, rc = D.split_counts(N, world, rank, D.SLABS_TO_BRICKS, nf)
send = torch.from_numpy(D.pack_host(work2, N, world, rank, D.SLABS_TO_BRICKS))
recv = torch.empty(sum(rc), dtype=torch.float64)
D.all_to_all(recv, send, rc, sc)
D.unpack_host(work2, recv.numpy(), N, world, rank, D.SLABS_TO_BRICKS)
ok &= bool(np.array_equal(work2[:, :, ya:yb], full[:, :, ya:yb]))
dist.barrier()
print(json.dumps({"rank": rank, "ok": ok, "ky": [ya, yb], "z": [za, zb]}))
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


import pytest


@pytest.mark.parametrize("world", [2, 3])
def test_slab_decomposition_transposes_over_gloo(world):
    """Host logic of the multi-GPU slab decomposition (paper_1810_12707_b200/dist.py): partition, split sizes, packed
    layout and ONE all_to_all_single per exchange turn 'all z of my ky range' into 'all ky of my z range' and back,
    with uneven shares (world = 3 does not divide N = 16 nor nyc = 11)."""
    import json
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", TRANSPOSE_WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    assert all(o["ok"] for o in outs)
    outs.sort(key=lambda o: o["rank"])
    assert outs[0]["ky"][0] == 0 and outs[-1]["ky"][1] == 11 and outs[0]["z"][0] == 0 and outs[-1]["z"][1] == 16
    for a, b in zip(outs, outs[1:]):
        assert a["ky"][1] == b["ky"][0] and a["z"][1] == b["z"][0]


def test_partition_is_balanced_and_counts_match():
    sys.path.insert(0, ROOT)
    from paper_1810_12707_b200 import dist as D
    for N, world in [(16, 2), (64, 3), (512, 8), (1024, 8), (256, 5)]:
        nyc, nxp = D.compact_extents(N)
        ky = [D.ranges(N, world, r)[0] for r in range(world)]
        zz = [D.ranges(N, world, r)[1] for r in range(world)]
        assert ky[0][0] == 0 and ky[-1][1] == nyc and zz[0][0] == 0 and zz[-1][1] == N
        assert max(b - a for a, b in ky) - min(b - a for a, b in ky) <= 1
        assert max(b - a for a, b in zz) - min(b - a for a, b in zz) <= 1
        for d in (0, 1):
            tot_s = tot_r = 0
            for r in range(world):
                s, rc = D.split_counts(N, world, r, d, 11)
                for peer in range(world):       # what r sends to peer is what peer expects from r
                    assert s[peer] == D.split_counts(N, world, peer, d, 11)[1][r]
                tot_s += sum(s); tot_r += sum(rc)
            own = sum(2 * 11 * (D.ranges(N, world, r)[1][1] - D.ranges(N, world, r)[1][0])
                      * (D.ranges(N, world, r)[0][1] - D.ranges(N, world, r)[0][0]) * nxp for r in range(world))
            assert tot_s == tot_r == 2 * 11 * N * nyc * nxp - own      # everything but the ranks' own blocks travels


def test_algorithmic_bytes_match_the_measured_dram_traffic():
    """bench.sweep_bytes (the algorithmic bytes behind every roofline fraction) against the DRAM bytes per launch that
    ncu measured (profiles/traffic_r02.json, from the committed captures): equal to within 4 %, i.e. no
    kernel re-reads what it should stream once, and the accounting does not flatter the fractions."""
    import json
    sys.path.insert(0, ROOT)
    import bench
    traffic = json.load(open(os.path.join(ROOT, "profiles", "traffic_r02.json")))
    for N in (256, 512):
        sb = bench.sweep_bytes(N, prune=True)
        launches = {"strided_inverse": 2, "strided_forward": 2, "x_fused": 1, "assemble": 1}
        for fam, n in launches.items():
            alg = sb[fam] / n
            meas = traffic[str(N)][fam]
            assert abs(meas / alg - 1.0) <= 0.04, (N, fam, meas / alg)
    # unpruned accounting: SURVEY.md's 148 field sweeps + the 32 of the separate forward z pass
    f = 8.0 * 512 ** 3
    assert abs(sum(bench.sweep_bytes(512, prune=False).values()) / f - 180.0) < 1e-9
    assert bench.unpruned_reference_bytes(512) == 1184.0 * 512 ** 3
