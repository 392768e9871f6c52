"""One GPU (process) per rank: the partitioned DVM step (include/ufs_dvm.h, "Partitioned mesh"; SURVEY.md 8(e), 8(f)-2;
PAPER.md:57 space-filling-curve partition, PAPER.md:185-187 multi-GPU advection with ghost cells).

Memory, streams and the transfer only: every copy that touches f on the device is the library's (ufs_dvm_halo_pack /
ufs_dvm_halo_unpack); what moves the packed buffers between ranks is torch.distributed (NCCL send / recv over NVLink), or
a plain device copy when several ranks are emulated on one device (tests, bench --emulate-ranks)."""
from typing import List, Optional

import numpy as np

from . import binding as B
from .inputs import Case, CELL_KINETIC, STORE_F32


class RankStepper(B.DvmStepper):
    """Rank `my_rank`'s part of `case`: f tensors of n_inner + n_ghost slabs, one packed send and one packed receive
    buffer per peer.  Canonical rows (load_canonical / read_canonical / moments) are the rank's own kinetic leaves in
    ascending leaf order (self.inner_leaves)."""

    def __init__(self, case: Case, rank_of_leaf: np.ndarray, my_rank: int, n_ranks: int, device="cuda:0",
                 kn: Optional[float] = None, storage: Optional[int] = None, stream=None, symmetric: bool = False, group=None):
        """symmetric: allocate the two f tensors as symmetric memory of the process group (every rank makes the same
        calls; sized for the largest rank) so that setup_push_distributed can hand the peers' mappings to the library."""
        import torch
        self.torch = torch
        self.case = case
        self.my_rank, self.n_ranks = int(my_rank), int(n_ranks)
        self.storage = case.storage if storage is None else storage
        self.dtype = torch.float32 if self.storage == STORE_F32 else torch.float64
        self.device = torch.device(device)
        desc, self._keep = B.make_desc(case, kn=kn, storage=self.storage)
        self.Nv = case.Nv
        h0 = B.ufs_dvm_create_part_host(desc, rank_of_leaf, my_rank, n_ranks)     # sizes first
        lay = B.ufs_dvm_part_layout(h0)
        B.ufs_dvm_destroy(h0)
        self.n_inner, self.n_ghost = lay["n_inner"], lay["n_ghost"]
        n_slabs = self.n_inner + self.n_ghost
        with torch.cuda.device(self.device):
            self.sums = None
            if symmetric:
                self.f, self.f_symm = _symmetric_f(torch, n_slabs, self.Nv, self.dtype, self.device, group)
                # the carried sums too (36 doubles per slab), so that the peers' step kernels can write the ghost rows
                self.sums, self.sums_symm = _symmetric_f(torch, n_slabs, 36, torch.float64, self.device, group)
            else:
                self.f = [torch.empty((n_slabs, self.Nv), dtype=self.dtype, device=self.device) for _ in range(2)]
            self.mom = torch.empty((5, max(self.n_inner, 1)), dtype=torch.float64, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.h = B.ufs_dvm_create_part(desc, rank_of_leaf, my_rank, n_ranks, [t.data_ptr() for t in self.f],
                                           self.stream.cuda_stream)
            if self.sums is not None:
                B.ufs_dvm_sums_use(self.h, self.sums[0].data_ptr(), self.sums[1].data_ptr())
            self.peers = []
            self.send_buf, self.recv_buf = {}, {}
            elem = 4 if self.storage == STORE_F32 else 8
            for p in range(n_ranks):
                sb, rb = B.ufs_dvm_halo_bytes(self.h, p)
                if sb or rb:
                    self.peers.append(p)
                    self.send_buf[p] = torch.empty(sb // elem, dtype=self.dtype, device=self.device)
                    self.recv_buf[p] = torch.empty(rb // elem, dtype=self.dtype, device=self.device)
        lay = B.ufs_dvm_part_layout(self.h)
        self.leaf_of_slab = lay["leaf_of_slab"]
        self.first_global_slab = lay["first_global_slab"]
        self.n_kinetic, self.cell_of_slab, self.vel_of_slot = B.ufs_dvm_layout(self.h, self.Nv)
        assert self.n_kinetic == self.n_inner
        self.inner_leaves = np.sort(self.cell_of_slab)
        row_of_leaf = np.full(case.n_leaves, -1, np.int64)
        row_of_leaf[self.inner_leaves] = np.arange(self.n_inner)
        self.row_of_slab = row_of_leaf[self.cell_of_slab]

    def moments(self) -> np.ndarray:
        if self.n_inner == 0:
            return np.zeros((5, 0))
        return super().moments()[:, :self.n_inner]

    # -- the library's side of the exchange
    def pack(self, peer: int):
        B.ufs_dvm_halo_pack(self.h, peer, self.send_buf[peer].data_ptr())

    def unpack(self, peer: int):
        B.ufs_dvm_halo_unpack(self.h, peer, self.recv_buf[peer].data_ptr())

    def halo_done(self):
        B.ufs_dvm_halo_done(self.h)

    def setup_push(self, peer_f, dest_slab, peer_sums=None):
        """Switch this rank to the fused ghost exchange (ufs_dvm_halo_push_setup): peer_f[p] = (address of rank p's f
        buffer 0, of its buffer 1) as this device reaches them, dest_slab[p] = rank p's recv_slab list for this rank;
        None for ranks that need nothing from this one.  peer_sums[p] = rank p's ufs_dvm_sums_dev pair: the ghost cells'
        sums are pushed as well."""
        pick = lambda xs, b: None if xs is None else [None if x is None else x[b] for x in xs]
        B.ufs_dvm_halo_push_setup(self.h, pick(peer_f, 0), pick(peer_f, 1), dest_slab, pick(peer_sums, 0), pick(peer_sums, 1))
        self.push = True

    def halo_bytes(self):
        """Bytes this rank sends / receives per step."""
        return (sum(t.numel() * t.element_size() for t in self.send_buf.values()),
                sum(t.numel() * t.element_size() for t in self.recv_buf.values()))


def _symmetric_f(torch, n_slabs, Nv, dtype, device, group):
    """Two f tensors in symmetric memory (torch.distributed._symmetric_memory): same size on every rank (the largest
    rank's), rendezvous over the group; returns the tensors cut to this rank's slabs and the rendezvous handles."""
    import torch.distributed as dist
    import torch.distributed._symmetric_memory as symm
    most = torch.tensor([n_slabs], dtype=torch.int64, device=device)
    dist.all_reduce(most, op=dist.ReduceOp.MAX, group=group)
    rows = max(int(most.item()), 1)
    name = dist.group.WORLD.group_name if group is None else group.group_name
    full = [symm.empty((rows, Nv), dtype=dtype, device=device) for _ in range(2)]
    handles = [symm.rendezvous(t, name) for t in full]
    return [t[:n_slabs] for t in full], handles


def exchange_local(ranks: List[RankStepper]):
    """Ghost exchange between ranks emulated on ONE device and one stream: pack, device copy, unpack, in stream order
    (no kernel waits on another one)."""
    for r in ranks:
        for p in r.peers:
            r.pack(p)
    for r in ranks:
        with r.torch.cuda.stream(r.stream):
            for p in r.peers:
                r.recv_buf[p].copy_(ranks[p].send_buf[r.my_rank])
        for p in r.peers:
            r.unpack(p)
        r.halo_done()


def exchange_distributed(rank: RankStepper, group=None):
    """Ghost exchange between real ranks: packed buffers by grouped send / recv (NCCL over NVLink / NVSwitch when the
    process group is nccl), enqueued on the handle's stream."""
    import torch.distributed as dist
    torch = rank.torch
    with torch.cuda.stream(rank.stream):
        for p in rank.peers:
            rank.pack(p)
        ops = []
        for p in rank.peers:
            if rank.send_buf[p].numel():
                ops.append(dist.P2POp(dist.isend, rank.send_buf[p], p, group=group))
            if rank.recv_buf[p].numel():
                ops.append(dist.P2POp(dist.irecv, rank.recv_buf[p], p, group=group))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for p in rank.peers:
            rank.unpack(p)
        rank.halo_done()


def setup_push_local(ranks: List[RankStepper], push_sums: bool = True):
    """Fused ghost exchange between ranks emulated on ONE device: every rank's step kernel stores its boundary cells
    straight into the other ranks' ghost slabs (the same address space: the peers' own pointers), and with push_sums their
    velocity sums into the other ranks' sums arrays."""
    n = len(ranks)
    for r in ranks:
        peer_f, dest, sums = [None] * n, [None] * n, [None] * n
        for p in r.peers:
            if B.ufs_dvm_halo_bytes(r.h, p)[0]:
                peer_f[p] = (ranks[p].f[0].data_ptr(), ranks[p].f[1].data_ptr())
                dest[p] = B.ufs_dvm_halo(ranks[p].h, r.my_rank)["recv_slab"]
                sums[p] = B.ufs_dvm_sums_dev(ranks[p].h)
        r.setup_push(peer_f, dest, sums if push_sums else None)


def step_pushed_local(ranks: List[RankStepper], dt: float):
    """One step of every rank under the fused exchange, ranks emulated on one device and ONE stream: the stream order is
    the barrier between the step kernels and the ghost sums (no kernel waits on another one)."""
    for r in ranks:
        r.step(dt, 1)
    for r in ranks:
        r.halo_done()


def setup_push_distributed(rank: RankStepper, group=None):
    """Fused ghost exchange between real ranks of one node.  The two f tensors of `rank` must have been allocated by
    torch.distributed._symmetric_memory.empty (rank.f_symm = the two rendezvous handles): every rank's buffers are then
    mapped into every other rank's address space over NVLink, and the peers' recv_slab lists travel once, on the host,
    by all_gather_object.  The carried sums live in symmetric memory as well (ufs_dvm_sums_use), so the ghost cells' sums
    are pushed too."""
    import torch.distributed as dist
    n = rank.n_ranks
    mine = {p: B.ufs_dvm_halo(rank.h, p)["recv_slab"] for p in rank.peers}
    everyone = [None] * n
    dist.all_gather_object(everyone, mine, group=group)
    peer_f, dest, sums = [None] * n, [None] * n, [None] * n
    for p in rank.peers:
        if B.ufs_dvm_halo_bytes(rank.h, p)[0]:
            peer_f[p] = tuple(int(rank.f_symm[b].buffer_ptrs[p]) for b in range(2))
            sums[p] = tuple(int(rank.sums_symm[b].buffer_ptrs[p]) for b in range(2))
            dest[p] = everyone[p][rank.my_rank]
    rank.setup_push(peer_f, dest, sums)
    rank.push_token = rank.torch.zeros(1, dtype=rank.torch.int32, device=rank.device)


def step_pushed_distributed(rank: RankStepper, dt: float, group=None):
    """One step under the fused exchange: the step kernel pushes while it computes; a barrier on the stream (NCCL) stands
    between every rank's step kernel and the ghost sums / the next step."""
    import torch.distributed as dist
    with rank.torch.cuda.stream(rank.stream):
        rank.step(dt, 1)
        dist.all_reduce(rank.push_token, group=group)     # ordered after the step kernel on this stream, on every rank
        rank.halo_done()
