"""Slab decomposition of the MHD step over several GPUs — thin driver.

One process per GPU.  Every phase of the path runs in libmhd's kernels (include/mhd.h, mhd_dist_*); this module only
sequences them and moves the packed blocks between ranks with ONE collective per exchange,
`torch.distributed.all_to_all_single` (NCCL over NVLink / NVSwitch on GPUs).  Per step: two all-to-alls, of 11 and 16
work fields, each rank sending (world-1)/world of its share.

The protocol is written once, as generators that yield the exchanges they need, and driven either by a real process
group (`DistMHD.step` etc.) or, for tests on a single GPU, by `Lockstep`, which runs `world` virtual ranks one after the
other in one process and performs the all-to-all as device copies — no kernel ever waits on another rank.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import binding as B

PHASE_A, PHASE_B, PHASE_C, PHASE_STORE, PHASE_STATE_Z = 0, 1, 2, 3, 4
BRICKS_TO_SLABS, SLABS_TO_BRICKS = 0, 1


# ---- host-side partition logic (mirrors mhd_dist_ranges / mhd_dist_counts; checked against them in the GPU tests) ------
def compact_extents(N: int):
    """(nyc, nxp): retained ky values 2*kc+1 and the padded retained kx count (kc+1 rounded up to 8)."""
    kc = N // 3
    return 2 * kc + 1, (kc + 1 + 7) // 8 * 8


def ranges(N: int, world: int, rank: int):
    """((ky_lo, ky_hi), (z_lo, z_hi)) of `rank`: contiguous, sizes differ by at most one."""
    nyc, _ = compact_extents(N)
    return (nyc * rank // world, nyc * (rank + 1) // world), (N * rank // world, N * (rank + 1) // world)


def split_counts(N: int, world: int, rank: int, direction: int, nf: int):
    """(send, recv): doubles exchanged with every peer.  BRICKS_TO_SLABS sends my ky range x the peer's z range."""
    _, nxp = compact_extents(N)
    (ya, yb), (za, zb) = ranges(N, world, rank)
    send, recv = [], []
    for s in range(world):
        (sa, sb), (ta, tb) = ranges(N, world, s)
        a = 2 * nf * (tb - ta) * (yb - ya) * nxp
        b = 2 * nf * (zb - za) * (sb - sa) * nxp
        if s == rank:
            a = b = 0        # the rank's own block (its ky range x its z range) never leaves the work arrays
        send.append(a if direction == BRICKS_TO_SLABS else b)
        recv.append(b if direction == BRICKS_TO_SLABS else a)
    return send, recv


def _block(N, world, me, peer, direction, unpack):
    """(z range, ky range) in the work arrays of the block exchanged with `peer` (same rule as ooc_dist_pack)."""
    mine_ky = (direction == BRICKS_TO_SLABS) != bool(unpack)
    rz, ry = (peer, me) if mine_ky else (me, peer)
    return ranges(N, world, rz)[1], ranges(N, world, ry)[0]


def pack_host(work: np.ndarray, N: int, world: int, rank: int, direction: int) -> np.ndarray:
    """Layout of the packed send buffer, on the host: work is [nf][N][nyc][nxp] complex128; the buffer is
    [peer 0 block | peer 1 block | ...], block = [f][z][ky][kx_c] (what mhd_dist_pack writes on the device)."""
    parts = []
    for s in range(world):
        if s == rank:
            continue
        (za, zb), (ya, yb) = _block(N, world, rank, s, direction, False)
        parts.append(np.ascontiguousarray(work[:, za:zb, ya:yb, :]).reshape(-1))
    return np.concatenate(parts).view(np.float64)


def unpack_host(work: np.ndarray, buf: np.ndarray, N: int, world: int, rank: int, direction: int) -> None:
    """Inverse of the exchange on the receiving side (what mhd_dist_unpack does on the device)."""
    c = buf.view(np.complex128)
    off = 0
    nf, _, _, nxp = work.shape
    for s in range(world):
        if s == rank:
            continue
        (za, zb), (ya, yb) = _block(N, world, rank, s, direction, True)
        n = nf * (zb - za) * (yb - ya) * nxp
        work[:, za:zb, ya:yb, :] = c[off:off + n].reshape(nf, zb - za, yb - ya, nxp)
        off += n


def all_to_all(recv, send, recv_counts, send_counts, group=None):
    """The one collective of the decomposition (host or device tensors; gloo or nccl)."""
    import torch.distributed as dist
    dist.all_to_all_single(recv, send, output_split_sizes=list(recv_counts), input_split_sizes=list(send_counts), group=group)


# ---- one rank ---------------------------------------------------------------------------------------------------------
class DistMHD(B.MHD):
    """Rank `rank` of `world`: a chunked-pipeline context (everything in device memory) restricted to its shares."""

    def __init__(self, N, L=2 * np.pi, gamma=5.0 / 3.0, mu=0.0, eta=0.0, dt=1e-3, rank=0, world=1, device="cuda:0",
                 stream=None, group=None, per_rank_storage=False):
        """per_rank_storage: allocate only this rank's share (MHD_FLAG_RANKS: 1/world of the state, 2/world of the work
        arrays) instead of full-size arrays of which the rank uses its share."""
        flags = B.MHD_FLAG_OUT_OF_CORE | (((int(world) - 1) << 4) if per_rank_storage and world > 1 else 0)
        super().__init__(N, L, gamma, mu, eta, dt, device=device, stream=stream, flags=flags)
        L_ = self._L
        L_.mhd_dist_config.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L_.mhd_dist_phase.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L_.mhd_dist_counts.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L_.mhd_dist_pack.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L_.mhd_dist_unpack.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L_.mhd_dist_ranges.argtypes = [C.c_void_p, C.c_int] + [C.POINTER(C.c_int)] * 4
        self.rank, self.world, self.group = int(rank), int(world), group
        self._check(L_.mhd_dist_config(self._h, self.rank, self.world))
        L_.mhd_dist_peers.argtypes = [C.c_void_p, C.POINTER(C.c_longlong)]
        self._pending_A = False      # phase A of the next step already ran inside phase C
        self.exchanged_bytes = 0     # bytes this rank has sent to OTHER ranks through the packed exchange
        self.direct = False          # rows stored straight into the owners' workspaces (set_peers)
        self._peer_keep = []

    # -- ABI calls ---------------------------------------------------------------------------------------
    def phase(self, which, arg=0):
        self._check(self._L.mhd_dist_phase(self._h, int(which), int(arg)))

    def counts(self, direction, nf):
        s = (C.c_longlong * self.world)()
        r = (C.c_longlong * self.world)()
        self._check(self._L.mhd_dist_counts(self._h, int(direction), int(nf), s, r))
        return list(s), list(r)

    def ranges(self, rank=None):
        v = [C.c_int() for _ in range(4)]
        self._check(self._L.mhd_dist_ranges(self._h, self.rank if rank is None else int(rank), *[C.byref(x) for x in v]))
        return (v[0].value, v[1].value), (v[2].value, v[3].value)

    def pack(self, direction, nf):
        send_counts, recv_counts = self.counts(direction, nf)
        n = sum(send_counts)
        send = self.torch.empty(max(n, 1), dtype=self.torch.float64, device=self.device)[:n]     # never a null pointer
        self._check(self._L.mhd_dist_pack(self._h, int(direction), int(nf), send.data_ptr()))
        return send, send_counts, recv_counts

    def unpack(self, direction, nf, recv):
        self._check(self._L.mhd_dist_unpack(self._h, int(direction), int(nf), recv.data_ptr()))

    def set_peers(self, peer_bases):
        """Direct exchange: peer_bases[s] = address, IN THIS PROCESS, of rank s's (256-byte aligned) workspace base
        (its own for s = rank); None switches back to the packed exchange."""
        if peer_bases is None:
            self._check(self._L.mhd_dist_peers(self._h, None))
            self.direct = False
            return
        d = (C.c_longlong * self.world)(*[int(b) - int(self._base) for b in peer_bases])
        self._check(self._L.mhd_dist_peers(self._h, d))
        self.direct = self.world > 1

    def connect_peers_ipc(self):
        """One process per GPU: map every peer's workspace into this process (CUDA IPC; NVLink peer access between GPUs)
        and switch to the direct exchange.  Handles travel through the process group as pickled objects."""
        import torch.distributed as dist
        torch = self.torch
        self.stream.synchronize()
        info = self.workspace.untyped_storage()._share_cuda_()          # (device, handle, size, offset, ...)
        mine = {"rank": self.rank, "share": info, "base_off": int(self._base) - int(self.workspace.data_ptr())}
        allinfo = [None] * self.world
        dist.all_gather_object(allinfo, mine, group=self.group)
        bases = []
        for s, inf in enumerate(allinfo):
            if s == self.rank:
                bases.append(int(self._base))
                continue
            peer_dev = int(inf["share"][0])
            if peer_dev != self.device.index:             # another GPU: kernels here must be allowed to store into it
                with torch.cuda.device(self.device):
                    self._L.mhd_dist_enable_peer_access.argtypes = [C.c_void_p, C.c_int]
                    self._check(self._L.mhd_dist_enable_peer_access(self._h, peer_dev))
            with torch.cuda.device(self.device):
                st = torch.UntypedStorage._new_shared_cuda(*inf["share"])
            self._peer_keep.append(st)                                   # keeps the mapping alive
            bases.append(int(st.data_ptr()) + inf["base_off"])
        self.set_peers(bases)
        dist.barrier(group=self.group)

    def barrier(self):
        """Where the packed protocol exchanges, the direct one only orders: my stores are done, so are my peers'."""
        import torch.distributed as dist
        self.stream.synchronize()
        if self.world > 1:
            dist.barrier(group=self.group)

    # -- the protocol, as generators that yield (direction, nfields) where an exchange is due ---------------------
    def _gen_set_fields(self, fields, kind):
        B.MHD.set_fields(self, fields, kind)              # own z planes: prim->cons, forward x and y passes
        yield (SLABS_TO_BRICKS, 8)
        self.phase(PHASE_STORE)                           # forward z + projection of own ky bricks
        self._pending_A = False

    def _gen_step(self, n):
        for s in range(int(n)):
            if not self._pending_A:
                if self.direct and s == 0:
                    yield ("barrier",)                    # peers may still read the rows phase A is about to store
                self.phase(PHASE_A)
            yield ("barrier",) if self.direct else (BRICKS_TO_SLABS, 11)
            self.phase(PHASE_B)
            yield ("barrier",) if self.direct else (SLABS_TO_BRICKS, 16)
            more = s + 1 < n
            self.phase(PHASE_C, 1 if more else 0)
            self._pending_A = more

    def _gen_get_fields(self, kind, where, out):
        self.phase(PHASE_STATE_Z)
        self._pending_A = False                           # work[0..7] was overwritten
        yield (BRICKS_TO_SLABS, 8)
        self._result = B.MHD.get_fields(self, kind, where, out)      # only this rank's z planes are written

    # -- driven by a real process group ----------------------------------------------------------------------------
    def exchange(self, direction, nf):
        if self.world == 1:
            return                                        # a single rank: its one block is already in place
        send, send_counts, recv_counts = self.pack(direction, nf)
        n = sum(recv_counts)
        recv = self.torch.empty(max(n, 1), dtype=self.torch.float64, device=self.device)[:n]
        import torch.distributed as dist
        if dist.get_backend(self.group) == "gloo":        # gloo moves host tensors (tests; NCCL is the production backend)
            self.stream.synchronize()
            host = self.torch.empty(n, dtype=self.torch.float64)
            all_to_all(host, send.cpu(), recv_counts, send_counts, self.group)
            recv.copy_(host)
        else:
            with self.torch.cuda.stream(self.stream):
                all_to_all(recv, send, recv_counts, send_counts, self.group)
        self.unpack(direction, nf, recv)
        self.exchanged_bytes += 8 * sum(send_counts)

    def _drive(self, gen):
        for req in gen:
            if req[0] == "barrier":
                self.barrier()
            else:
                self.exchange(*req)

    def set_fields(self, fields, kind="primitive"):
        self._drive(self._gen_set_fields(fields, kind))

    def step(self, n=1):
        self._drive(self._gen_step(n))

    def get_fields(self, kind="conservative", where="host", out=None):
        """Full-size arrays of which only this rank's z planes (self.ranges()[1]) are filled."""
        self._drive(self._gen_get_fields(kind, where, out))
        return self._result


# ---- `world` virtual ranks in one process (single-GPU tests of the decomposition) ------------------------------------------
class Lockstep:
    """Runs the same protocol for all ranks in lockstep; the all-to-all is a set of device copies."""

    def __init__(self, ranks):
        self.ranks = list(ranks)
        assert all(r.world == len(self.ranks) and r.rank == i for i, r in enumerate(self.ranks))

    def _exchange(self, direction, nf):
        torch = self.ranks[0].torch
        packed = [r.pack(direction, nf) for r in self.ranks]
        for r in self.ranks:
            r.stream.synchronize()
        for me, r in enumerate(self.ranks):
            _, _, recv_counts = packed[me]
            parts = []
            for s in range(len(self.ranks)):
                send_s, send_counts_s, _ = packed[s]
                off = sum(send_counts_s[:me])
                assert send_counts_s[me] == recv_counts[s]
                parts.append(send_s[off:off + send_counts_s[me]])
            recv = torch.cat(parts + [torch.empty(1, dtype=torch.float64, device=r.device)])   # never a null pointer
            r.unpack(direction, nf, recv)
            r.stream.synchronize()

    def _drive(self, gens):
        while True:
            reqs = []
            for g in gens:
                try:
                    reqs.append(next(g))
                except StopIteration:
                    reqs.append(None)
            if all(q is None for q in reqs):
                return
            assert all(q == reqs[0] for q in reqs), "ranks out of step"
            if reqs[0][0] == "barrier":
                for r in self.ranks:
                    r.stream.synchronize()
            else:
                self._exchange(*reqs[0])

    def connect_peers(self):
        """Virtual ranks share one address space: every rank can store into every other rank's workspace."""
        bases = [r._base for r in self.ranks]
        for r in self.ranks:
            r.set_peers(bases)

    def set_fields(self, fields, kind="primitive"):
        self._drive([r._gen_set_fields(fields, kind) for r in self.ranks])

    def step(self, n=1):
        self._drive([r._gen_step(n) for r in self.ranks])

    def get_fields(self, kind="conservative"):
        """Assembled full fields: every rank contributes its z planes."""
        N = self.ranks[0].N
        outs = [[np.zeros((N, N, N)) for _ in range(8)] for _ in self.ranks]
        self._drive([r._gen_get_fields(kind, "host", outs[i]) for i, r in enumerate(self.ranks)])
        full = [np.empty((N, N, N)) for _ in range(8)]
        for i, r in enumerate(self.ranks):
            za, zb = r.ranges()[1]
            for f in range(8):
                full[f][za:zb] = outs[i][f][za:zb]
        return full
