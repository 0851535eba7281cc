"""Slab decomposition over several GPUs, tested on ONE GPU: `world` virtual ranks run the
protocol of paper_1810_12707_b200/dist.py one after the other in one process (no kernel waits on another rank), the
all-to-all is a set of device copies.  The result must equal the undecomposed chunked pipeline BITWISE — the same
kernels see the same data, only who computes which brick / slab changes — and the oracle within the usual tolerance."""
import math

import numpy as np
import pytest

from paper_1810_12707_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1810_12707_b200 import build, binding, dist
    build.build()
    return binding, dist


def make_ranks(dist, cfg, world, dt=None, per_rank=False):
    return dist.Lockstep([dist.DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, dt or cfg.dt, rank=r, world=world,
                                       per_rank_storage=per_rank) for r in range(world)])


@pytest.mark.parametrize("per_rank", [False, True])
@pytest.mark.parametrize("N,world", [(32, 2), (32, 3), (64, 4), (128, 8), (64, 7)])
def test_decomposed_step_is_bitwise_the_single_gpu_step(mods, N, world, per_rank):
    """per_rank: MHD_FLAG_RANKS — every rank allocates only its share (brick- and slab-shaped work arrays)."""
    binding, dist = mods
    cfg = inputs.config3(N, kmax=4) if N >= 64 else inputs.config2(N)
    ref = binding.MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, flags=binding.MHD_FLAG_OUT_OF_CORE)
    ref.set_fields(cfg.prim, "primitive")
    grp = make_ranks(dist, cfg, world, per_rank=per_rank)
    if per_rank:
        full = binding.MHD(cfg.N, flags=binding.MHD_FLAG_OUT_OF_CORE).workspace_bytes
        assert grp.ranks[0].workspace_bytes < full * (3.0 / world + 0.35)      # 1/G state + 2/G work + staging
    grp.set_fields(cfg.prim, "primitive")
    U0r, U0g = ref.get_fields(), grp.get_fields()
    for f in range(8):
        assert np.array_equal(U0r[f], U0g[f]), ("after set_fields", f)
    ref.step(3); grp.step(3)            # Euler start + AB2, phase A of steps 2, 3 fused into phase C
    ref.step(2); grp.step(2)            # a second call: phase A runs on its own again
    Ur, Ug = ref.get_fields("primitive"), grp.get_fields("primitive")
    for f in range(8):
        assert np.array_equal(Ur[f], Ug[f]), ("after 5 steps", f)


def test_decomposed_run_matches_oracle(orc, mods):
    binding, dist = mods
    cfg = inputs.config1(32)
    o = orc.Oracle(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
    o.set_fields(cfg.prim, "primitive")
    grp = make_ranks(dist, cfg, 4)
    grp.set_fields(cfg.prim, "primitive")
    o.step(10); grp.step(10)
    Uo, Ug = o.get_fields(), grp.get_fields()
    scale = max(np.linalg.norm(x) for x in Uo)
    for f in range(8):
        assert np.linalg.norm(Ug[f] - Uo[f]) <= 1e-12 * scale


def test_library_partition_and_packing_match_the_host_logic(mods):
    """mhd_dist_ranges / mhd_dist_counts / mhd_dist_pack against dist.ranges / split_counts / pack_host (the host
    logic that the gloo test exercises with a real all_to_all_single)."""
    import torch
    binding, dist = mods
    N, world = 32, 3
    cfg = inputs.config2(N)
    nyc, nxp = dist.compact_extents(N)
    for rank in range(world):
        g = dist.DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, rank=rank, world=world)
        for r in range(world):
            assert g.ranges(r) == dist.ranges(N, world, r)
        for d in (0, 1):
            for nf in (8, 11, 16):
                assert g.counts(d, nf) == dist.split_counts(N, world, rank, d, nf)
        # fill the work arrays through the public path: slab part of set_fields writes work[0..7] on own z planes
        binding.MHD.set_fields(g, cfg.prim, "primitive")
        send, sc, rc = g.pack(dist.SLABS_TO_BRICKS, 8)
        g.stream.synchronize()
        # unpack into a second context of the same rank and pack again: the round trip is the identity on the blocks
        (ya, yb), (za, zb) = g.ranges()
        assert send.numel() == sum(sc) == 2 * 8 * (zb - za) * (nyc - (yb - ya)) * nxp       # all but the own block
        h = dist.DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, rank=rank, world=world)
        # the receive side of BRICKS_TO_SLABS has the geometry of the send side of SLABS_TO_BRICKS
        h.unpack(dist.BRICKS_TO_SLABS, 8, send)
        again, _, _ = h.pack(dist.SLABS_TO_BRICKS, 8)
        h.stream.synchronize()
        assert torch.equal(send, again)
        # layout: [peer][f][z][ky][kx]: compare with pack_host on a work array rebuilt from the blocks
        work = np.zeros((8, N, nyc, nxp), dtype=np.complex128)
        dist.unpack_host(work, send.cpu().numpy(), N, world, rank, dist.BRICKS_TO_SLABS)
        assert np.array_equal(dist.pack_host(work, N, world, rank, dist.SLABS_TO_BRICKS), send.cpu().numpy())


def test_decomposed_context_refuses_the_undecomposed_calls(mods):
    binding, dist = mods
    cfg = inputs.config1(32)
    g = dist.DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, rank=0, world=2)
    with pytest.raises(RuntimeError):
        g.phase(dist.PHASE_A)                       # no fields yet
    binding.MHD.set_fields(g, cfg.prim, "primitive")
    with pytest.raises(RuntimeError):
        binding.MHD.step(g, 1)                      # must be driven through the phases
    with pytest.raises(RuntimeError):
        g.rhs()
    with pytest.raises(RuntimeError):
        g.diagnostics()
    inc = binding.MHD(cfg.N)                        # an in-core context cannot be decomposed
    rc = inc._L.mhd_dist_config(inc._h, 0, 2)
    assert rc == -1


@pytest.mark.parametrize("per_rank", [False, True])
@pytest.mark.parametrize("N,world", [(32, 2), (64, 3), (128, 8), (64, 5)])
def test_direct_exchange_is_bitwise_too(mods, N, world, per_rank):
    """mhd_dist_peers: the z passes and the forward y pass store every row straight into its owner's workspace (what
    P2P stores over NVLink do between GPUs; here the virtual ranks share one GPU's address space): no pack, no
    collective, no unpack — and still the bits of the undecomposed step."""
    binding, dist = mods
    cfg = inputs.config3(N, kmax=4) if N >= 64 else inputs.config2(N)
    ref = binding.MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, flags=binding.MHD_FLAG_OUT_OF_CORE)
    ref.set_fields(cfg.prim, "primitive")
    grp = make_ranks(dist, cfg, world, per_rank=per_rank)
    grp.connect_peers()
    assert all(r.direct for r in grp.ranks)
    grp.set_fields(cfg.prim, "primitive")
    ref.step(3); grp.step(3)
    ref.step(2); grp.step(2)
    Ur, Ug = ref.get_fields("primitive"), grp.get_fields("primitive")
    for f in range(8):
        assert np.array_equal(Ur[f], Ug[f]), ("after 5 steps", f)
    assert all(r.exchanged_bytes == grp.ranks[0].exchanged_bytes for r in grp.ranks[:1])
    # the step itself moved nothing through packed buffers: only set_fields / get_fields did (8 fields, twice)
    sent = grp.ranks[0].exchanged_bytes
    grp.step(2)
    assert grp.ranks[0].exchanged_bytes == sent


IPC_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch
import torch.distributed as dist
from paper_1810_12707_b200 import dist as D, inputs
dist.init_process_group("gloo")                      # host-side barriers and handle exchange only
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)                             # both processes on the one GPU: CUDA IPC maps the peer's workspace
cfg = inputs.config2(32)
g = D.DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, rank=rank, world=world, device="cuda:0",
              per_rank_storage=True)
g.connect_peers_ipc()
assert g.direct
# set / get use the packed exchange: gloo all_to_all_single needs host tensors, so route it through the host here
def exchange_via_host(direction, nf):
    send, sc, rc = g.pack(direction, nf)
    g.stream.synchronize()
    recv = torch.empty(sum(rc), dtype=torch.float64)
    D.all_to_all(recv, send.cpu(), rc, sc)
    buf = torch.empty(max(1, recv.numel()), dtype=torch.float64, device="cuda:0")
    buf[:recv.numel()].copy_(recv)
    g.unpack(direction, nf, buf)
    g.stream.synchronize()
g.exchange = exchange_via_host
g.set_fields(cfg.prim, "primitive")
g.step(3)
g.step(2)
out = g.get_fields("primitive")
(za, zb) = g.ranges()[1]
np.save(os.environ["OUT_PREFIX"] + str(rank) + ".npy", np.stack([o[za:zb] for o in out]))
dist.barrier()
print(json.dumps({"rank": rank, "z": [za, zb], "direct": g.direct}))
dist.destroy_process_group()
"""


def test_direct_exchange_between_two_processes_over_cuda_ipc(mods, tmp_path):
    """Two PROCESSES (ranks 0, 1) on the one GPU: each maps the other's workspace through CUDA IPC (the mechanism that
    gives NVLink peer access between GPUs) and the step runs with direct stores and host barriers only — no kernel
    waits on the other rank.  Result: bitwise the undecomposed step."""
    import json, os, socket, subprocess, sys
    binding, dist = mods
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    prefix = str(tmp_path / "rank")
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   OUT_PREFIX=prefix)
        procs.append(subprocess.Popen([sys.executable, "-c", IPC_WORKER % root], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    metas = []
    for p in procs:
        out, err = p.communicate(timeout=600)
        assert p.returncode == 0, err[-3000:]
        metas.append(json.loads(out.strip().splitlines()[-1]))
    cfg = inputs.config2(32)
    ref = binding.MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, flags=binding.MHD_FLAG_OUT_OF_CORE)
    ref.set_fields(cfg.prim, "primitive")
    ref.step(3); ref.step(2)
    Ur = ref.get_fields("primitive")
    for m in metas:
        za, zb = m["z"]
        got = np.load(prefix + str(m["rank"]) + ".npy")
        for f in range(8):
            assert np.array_equal(got[f], Ur[f][za:zb]), (m["rank"], f)


@pytest.mark.parametrize("mode", ["decompose", "decompose_packed", "replicas"])
def test_bench_with_two_ranks_on_one_gpu(mods, mode):
    """bench.py as the driver launches it for N = 2 (one process per rank, env RANK / WORLD_SIZE / MASTER_*), with both ranks
    on the one GPU and gloo instead of NCCL (NCCL refuses two ranks on a device): the whole multi-rank flow — build on rank 0,
    barriers, IPC peer mapping or packed exchange, max-over-ranks timing, one JSON line from rank 0."""
    import json, os, socket, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    extra = {"decompose": ["--decompose"], "decompose_packed": ["--decompose", "--packed-exchange"], "replicas": []}[mode]
    cmd = [sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--size", "128", "--steps", "4", "--warmup", "3",
           "--no-cpu", "--no-fft", "--no-e2e"] + extra
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   MHD_BENCH_BACKEND="gloo")
        procs.append(subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, cwd=root))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=900)
        assert p.returncode == 0, err[-3000:]
        outs.append(out.strip())
    assert outs[1] == ""                                   # only rank 0 prints
    line = json.loads(outs[0].splitlines()[-1])
    assert line["n_gpus"] == 2 and line["steps"] == 4 and line["value"] > 0
    if mode == "replicas":
        assert line["scaling"] == "weak" and line["config"]["parallelism"] == "replicas x2"
        assert abs(line["value"] * line["ms_per_step"] * 1e-3 / (2 * 128 ** 3) - 1.0) < 1e-9       # whole-job work / max time
    else:
        assert line["scaling"] == "strong" and line["config"]["parallelism"] == "slab decomposition x2"
        dec = line["out_of_core"]["decomposed"]
        assert dec["world"] == 2 and ("direct" in dec["exchange"]) == (mode == "decompose")
        assert abs(line["value"] * line["ms_per_step"] * 1e-3 / (128 ** 3) - 1.0) < 1e-9           # ONE problem over both ranks
        if mode == "decompose_packed":
            assert dec["sent_to_peers_bytes_per_step_per_rank"] > 0
        else:
            assert dec["sent_to_peers_bytes_per_step_per_rank"] == 0                                  # rows went by P2P stores
