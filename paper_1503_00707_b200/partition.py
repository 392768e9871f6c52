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
                 kn: Optional[float] = None, storage: Optional[int] = None, stream=None):
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
            self.f = [torch.empty((n_slabs, self.Nv), dtype=self.dtype, device=self.device) for _ in range(2)]
            self.mom = torch.empty((5, max(self.n_inner, 1)), dtype=torch.float64, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.h = B.ufs_dvm_create_part(desc, rank_of_leaf, my_rank, n_ranks, [t.data_ptr() for t in self.f],
                                           self.stream.cuda_stream)
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

    def halo_bytes(self):
        """Bytes this rank sends / receives per step."""
        return (sum(t.numel() * t.element_size() for t in self.send_buf.values()),
                sum(t.numel() * t.element_size() for t in self.recv_buf.values()))


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
