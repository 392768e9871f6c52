"""Host logic of the partitioned mesh (flatten.cpp: partition_leaves, restrict_to_rank; SURVEY.md 8(e), 8(f)-2;
PAPER.md:57 N-order partition with weights, PAPER.md:185-187 inner cells before ghost cells, one ghost gather per step).

* the partition covers every leaf once, cuts the N-order curve into consecutive ranges and balances the weights
  to within one leaf;
* the halo lists equal a brute-force derivation from all leaf pairs (tests/helpers.brute_force_faces), peer by peer,
  chunk mask by chunk mask, and what one rank sends is what the other expects, in the same order;
* a world-size-2 gloo run: each rank steps the ORACLE on its own part of the mesh (inner leaves + ghost leaves + the
  non-kinetic leaves around them), exchanging before every step exactly the chunks the library's halo lists name; the
  stitched result is bit-equal to the one-domain oracle.  Data the lists do not name is never right on the receiving
  side (ghost rows start from garbage), so a missing chunk or a wrong mask changes the result."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from tests.helpers import brute_force_faces, periodic_case, random_tree

P = (True, True, True)


def _cases():
    lv, ijk = random_tree(np.random.default_rng(5), 2, 4, P, 0.3)
    return {"small3_walls_solid": inputs.small(3), "small5_mask": inputs.small(5),
            "random_periodic": periodic_case(lv, ijk, nv=(6, 6, 6))}


def _periodic_flags(case):
    return tuple(case.bc[2 * a] == inputs.BC_PERIODIC for a in range(3))


# ----------------------------------------------------------------------------------------------- the partition
@pytest.mark.parametrize("name", ["small3_walls_solid", "small5_mask", "random_periodic"])
@pytest.mark.parametrize("n_ranks", [1, 2, 3, 7])
def test_partition_is_a_balanced_cut_of_the_n_order_curve(name, n_ranks):
    case = _cases()[name]
    desc, keep = B.make_desc(case)
    wk, wf = 1.0, 0.05
    rol = B.ufs_dvm_partition(desc, n_ranks, wk, wf)
    assert rol.shape == (case.n_leaves,) and rol.min() >= 0 and rol.max() < n_ranks     # every leaf, one rank each
    order = inputs.morton_order(case.level, case.ijk)                                   # numpy N-order (inputs.py)
    along = rol[order]
    assert np.all(np.diff(along) >= 0)                                                  # consecutive ranges of the curve
    w = np.where(case.kind == inputs.CELL_KINETIC, wk, np.where(case.kind == inputs.CELL_FLUID, wf, 0.0))
    per_rank = np.bincount(rol, weights=w, minlength=n_ranks)
    assert np.abs(per_rank - w.sum() / n_ranks).max() <= w.max() + 1e-9                 # within one leaf of the mean
    # kinetic >> fluid weights: with w_fluid = 0 the kinetic leaves alone are balanced
    rol0 = B.ufs_dvm_partition(desc, n_ranks, 1.0, 0.0)
    kin = np.bincount(rol0[case.kind == inputs.CELL_KINETIC], minlength=n_ranks)
    assert kin.max() - kin.min() <= 1


def test_partition_rejects_bad_arguments():
    case = inputs.small(3)
    desc, keep = B.make_desc(case)
    with pytest.raises(B.UfsDvmError):
        B.ufs_dvm_partition(desc, 0)
    with pytest.raises(B.UfsDvmError):
        B.ufs_dvm_partition(desc, 2, w_kinetic=0.0)
    # ownership that is not a range of the curve is refused
    rol = B.ufs_dvm_partition(desc, 2)
    order = inputs.morton_order(case.level, case.ijk)
    kin_along = order[case.kind[order] == inputs.CELL_KINETIC]
    bad = rol.copy(); bad[kin_along[0]] = 1; bad[kin_along[-1]] = 0
    with pytest.raises(B.UfsDvmError) as e:
        B.ufs_dvm_create_part_host(desc, bad, 0, 2)
    assert e.value.code == B.EINVAL


# ----------------------------------------------------------------------------------------------- halo lists
def _brute_force_needs(case, rol, n_ranks):
    """needs[r][p] = {leaf: octant mask} of the kinetic leaves of rank p that rank r's kinetic leaves read: over a face
    on axis a the high cell reads the low cell's groups with xi_a > 0 (bit a set), the low cell the high cell's groups
    with xi_a < 0."""
    live = case.kind != inputs.CELL_SOLID
    faces = brute_force_faces(case.level, case.ijk, _periodic_flags(case), live=live)
    up = [sum(1 << o for o in range(8) if (o >> a) & 1) for a in range(3)]
    needs = [[dict() for _ in range(n_ranks)] for _ in range(n_ranks)]
    kin = case.kind == inputs.CELL_KINETIC
    for lo, hi, a, _ in faces:
        if not (kin[lo] and kin[hi]) or rol[lo] == rol[hi]:
            continue
        d = needs[rol[hi]][rol[lo]]; d[lo] = d.get(lo, 0) | up[a]
        d = needs[rol[lo]][rol[hi]]; d[hi] = d.get(hi, 0) | (0xFF ^ up[a])
    return needs


@pytest.mark.parametrize("name", ["small3_walls_solid", "small5_mask", "random_periodic"])
@pytest.mark.parametrize("n_ranks", [2, 3, 5])
def test_halo_lists_equal_the_brute_force_derivation(name, n_ranks):
    case = _cases()[name]
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, n_ranks)
    needs = _brute_force_needs(case, rol, n_ranks)
    hs = [B.ufs_dvm_create_part_host(desc, rol, r, n_ranks) for r in range(n_ranks)]
    try:
        lays = [B.ufs_dvm_part_layout(h) for h in hs]
        n_all = 0
        for r in range(n_ranks):
            lay = lays[r]
            # inner cells first: the rank's kinetic leaves in N-order; ghosts after
            inner = lay["leaf_of_slab"][:lay["n_inner"]]
            assert set(inner.tolist()) == set(np.nonzero((rol == r) & (case.kind == inputs.CELL_KINETIC))[0].tolist())
            n_all += lay["n_inner"]
            ghosts = lay["leaf_of_slab"][lay["n_inner"]:]
            assert np.array_equal(rol[ghosts], lay["owner_of_ghost"])
            want_all = {}
            for p in range(n_ranks):
                hl = B.ufs_dvm_halo(hs[r], p)
                got = {int(lay["leaf_of_slab"][s]): int(m) for s, m in zip(hl["recv_slab"], hl["recv_mask"])}
                assert got == needs[r][p], f"rank {r} <- {p}"
                assert np.all(hl["recv_slab"] >= lay["n_inner"])
                want_all.update(got)
                # what p sends to r is what r expects from p, entry by entry
                hp = B.ufs_dvm_halo(hs[p], r)
                sent = [(int(lays[p]["leaf_of_slab"][s]), int(m)) for s, m in zip(hp["send_slab"], hp["send_mask"])]
                recv = [(int(lay["leaf_of_slab"][s]), int(m)) for s, m in zip(hl["recv_slab"], hl["recv_mask"])]
                assert sent == recv
                assert np.all(hp["send_slab"] < lays[p]["n_inner"])
                sb, _ = B.ufs_dvm_halo_bytes(hs[p], r)
                _, rb = B.ufs_dvm_halo_bytes(hs[r], p)
                chunk = (case.Nv // 8) * 8
                # chunks, then (streaming kernels) the 36 carried sums of every listed cell
                tail = 36 * 8 if B.ufs_dvm_kernel_name(hs[p]) in ("k_tiles", "k_rows", "k_stream") else 0
                assert sb == rb == sum(bin(m).count("1") for _, m in sent) * chunk + len(sent) * tail
            assert set(ghosts.tolist()) == set(want_all)              # no ghost nobody reads, none missing
            if want_all:
                assert max(bin(m).count("1") for m in want_all.values()) <= 8
        assert n_all == int((case.kind == inputs.CELL_KINETIC).sum())
    finally:
        for h in hs:
            B.ufs_dvm_destroy(h)


def test_one_face_ghost_gets_only_its_four_upwind_chunks():
    """Uniform periodic grid cut in two along the curve: a ghost that touches the rank across one face only is listed
    with exactly four octant chunks."""
    lv, ijk = random_tree(np.random.default_rng(0), 2, 2, P, 0.0)
    case = periodic_case(lv, ijk, nv=(6, 6, 6))
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, 2)
    h = B.ufs_dvm_create_part_host(desc, rol, 0, 2)
    hl = B.ufs_dvm_halo(h, 1)
    counts = np.array([bin(int(m)).count("1") for m in hl["recv_mask"]])
    assert counts.min() == 4 and (counts == 4).sum() > 0
    B.ufs_dvm_destroy(h)


@pytest.mark.parametrize("name,n_ranks", [("small3_walls_solid", 2), ("small3_walls_solid", 5), ("small5_mask", 3)])
def test_push_entries_pair_every_send_slab_with_the_peers_ghost_slab(name, n_ranks):
    """ufs_dvm_halo_push_setup on host-only handles (made-up buffer addresses): one entry per (sent cell, peer) with the
    send list's octant mask and the address of the ghost slab the PEER's receive list names for it, in both f buffers; the
    tiles with entries first."""
    case = _cases()[name]
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, n_ranks)
    hs = [B.ufs_dvm_create_part_host(desc, rol, r, n_ranks) for r in range(n_ranks)]
    slab_bytes = case.Nv * 8
    base = lambda p, b: 4096 * (1 + 2 * p + b) * (1 << 32)
    try:
        for r in range(n_ranks):
            with pytest.raises(B.UfsDvmError):
                B.ufs_dvm_push_entries(hs[r])                       # not set up yet
            dest = [None if p == r else B.ufs_dvm_halo(hs[p], r)["recv_slab"] for p in range(n_ranks)]
            sbase = lambda p, b: base(p, b) + (1 << 30)
            B.ufs_dvm_halo_push_setup(hs[r], [None if p == r else base(p, 0) for p in range(n_ranks)],
                                      [None if p == r else base(p, 1) for p in range(n_ranks)], dest)
            assert not B.ufs_dvm_push_entries(hs[r])["sums0"].any()          # no sums arrays given: no sums pushed
            with pytest.raises(B.UfsDvmError):                              # both or neither
                B.ufs_dvm_halo_push_setup(hs[r], [None if p == r else base(p, 0) for p in range(n_ranks)],
                                          [None if p == r else base(p, 1) for p in range(n_ranks)], dest,
                                          [None if p == r else sbase(p, 0) for p in range(n_ranks)], None)
            B.ufs_dvm_halo_push_setup(hs[r], [None if p == r else base(p, 0) for p in range(n_ranks)],
                                      [None if p == r else base(p, 1) for p in range(n_ranks)], dest,
                                      [None if p == r else sbase(p, 0) for p in range(n_ranks)],
                                      [None if p == r else sbase(p, 1) for p in range(n_ranks)])
            ent = B.ufs_dvm_push_entries(hs[r])
            want = set()
            for p in range(n_ranks):
                if p == r:
                    continue
                hl = B.ufs_dvm_halo(hs[r], p)
                for s, m, d in zip(hl["send_slab"], hl["send_mask"], dest[p]):
                    want.add((int(s), int(m), base(p, 0) + int(d) * slab_bytes, base(p, 1) + int(d) * slab_bytes,
                              sbase(p, 0) + int(d) * 36 * 8, sbase(p, 1) + int(d) * 36 * 8))    # a sums row: 36 doubles
            got = list(zip(ent["slab"].tolist(), ent["mask"].tolist(), ent["dst0"].tolist(), ent["dst1"].tolist(),
                           ent["sums0"].tolist(), ent["sums1"].tolist()))
            assert len(got) == len(set(got)) and set(got) == want
            t = B.ufs_dvm_tiles(hs[r])
            sent = np.zeros(B.ufs_dvm_part_layout(hs[r])["n_inner"], bool)
            sent[ent["slab"]] = True
            has = np.array([sent[t["s0"][i]:t["s0"][i] + t["nc"][i]].any() for i in range(t["n_tiles"])])
            assert ent["n_push_tiles"] == has.sum() and np.all(has[:has.sum()]) and not np.any(has[has.sum():])
            # inside each group the tiles keep their N-order
            for grp in (t["s0"][:has.sum()], t["s0"][has.sum():]):
                assert np.all(np.diff(grp) > 0)
            # a second set-up with the same arguments changes nothing
            B.ufs_dvm_halo_push_setup(hs[r], [None if p == r else base(p, 0) for p in range(n_ranks)],
                                      [None if p == r else base(p, 1) for p in range(n_ranks)], dest)
            ent2 = B.ufs_dvm_push_entries(hs[r])
            assert all(np.array_equal(ent[k], ent2[k]) for k in ("slab", "mask", "dst0", "dst1"))
            assert not ent2["sums0"].any()
    finally:
        for h in hs:
            B.ufs_dvm_destroy(h)


# ----------------------------------------------------------------------------------------------- two ranks, gloo
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _octant_of_velocity(case):
    """Sign group (bit a set: xi_a > 0) of every canonical velocity index."""
    nv = case.nv
    kz, ky, kx = np.meshgrid(np.arange(nv[2]), np.arange(nv[1]), np.arange(nv[0]), indexing="ij")
    return ((kx >= nv[0] // 2) * 1 + (ky >= nv[1] // 2) * 2 + (kz >= nv[2] // 2) * 4).ravel()


def _rank_worker(rank, world, port, which, nsteps, out, fused=False):
    import torch
    import torch.distributed as dist
    from oracle.dvm_oracle import Oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    case = _cases()[which]
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, world)
    h = B.ufs_dvm_create_part_host(desc, rol, rank, world)
    lay = B.ufs_dvm_part_layout(h)
    n_in = lay["n_inner"]
    slabs = lay["leaf_of_slab"]                                   # inner then ghost leaves
    full = Oracle(case)                                           # the oracle's own neighbour search, whole mesh
    around = full.leaf_neighbours(slabs[:n_in])
    ids = np.unique(np.concatenate([slabs, around]))
    # ghost cells = the foreign kinetic leaves among the inner cells' neighbours
    foreign = around[(case.kind[around] == inputs.CELL_KINETIC) & (rol[around] != rank)]
    assert set(foreign.tolist()) == set(slabs[n_in:].tolist())
    sub = inputs.sub_case(case, ids)
    o = Oracle(sub, window=True)
    kin_ids = ids[case.kind[ids] == inputs.CELL_KINETIC]          # oracle rows of the part
    row = {int(l): i for i, l in enumerate(kin_ids)}
    f0_all = inputs.initial_f(case)                               # rows: kinetic leaves of the whole case
    glob_row = np.full(case.n_leaves, -1, np.int64); glob_row[case.kinetic_leaves()] = np.arange(case.kinetic_leaves().size)
    f = f0_all[glob_row[kin_ids]].copy()
    ghost_rows = np.array([row[int(l)] for l in slabs[n_in:]], np.int64)
    f[ghost_rows] *= 0.37                                         # garbage until the exchange fills what is needed
    octv = _octant_of_velocity(case)
    halos = {p: B.ufs_dvm_halo(h, p) for p in range(world) if p != rank}
    if fused:
        # fused exchange (ufs_dvm_halo_push_setup on the host-only handle): what travels, and WHERE it lands in the peer, comes
        # from this rank's push entries -- made-up buffer addresses, decoded back to (peer, ghost slab) -- not from the
        # peer's own receive list.  The peers' receive lists are the set-up input, exchanged once.
        recv_lists = [None] * world
        dist.all_gather_object(recv_lists, {p: hl["recv_slab"] for p, hl in halos.items()})
        slab_bytes = case.Nv * 8
        base = lambda p, b: ((p + 1) << 44) + (b << 43)
        B.ufs_dvm_halo_push_setup(h, [None if p == rank else base(p, 0) for p in range(world)],
                                  [None if p == rank else base(p, 1) for p in range(world)],
                                  [None if p == rank else recv_lists[p][rank] for p in range(world)])
        ent = B.ufs_dvm_push_entries(h)
        assert np.all(ent["dst1"] - ent["dst0"] == (1 << 43))
        peer_of = (ent["dst0"] >> np.uint64(44)).astype(np.int64) - 1
        dest_of = ((ent["dst0"] & np.uint64((1 << 43) - 1)) // np.uint64(slab_bytes)).astype(np.int64)
        assert np.all((ent["dst0"] & np.uint64((1 << 43) - 1)) % np.uint64(slab_bytes) == 0)
        for p, hl in halos.items():
            mine = np.nonzero(peer_of == p)[0]
            mine = mine[np.argsort(dest_of[mine], kind="stable")]
            # the same chunks as the send list, each with the ghost slab the peer expects it in
            assert sorted(zip(ent["slab"][mine].tolist(), ent["mask"][mine].tolist())) == sorted(zip(hl["send_slab"].tolist(), hl["send_mask"].tolist()))
            halos[p] = dict(hl, send_slab=ent["slab"][mine], send_mask=ent["mask"][mine], send_dest=dest_of[mine])
    for _ in range(nsteps):
        reqs, recv = [], {}
        for p, hl in halos.items():
            parts = [f[row[int(slabs[s])]][(int(m) >> octv) & 1 == 1] for s, m in zip(hl["send_slab"], hl["send_mask"])]
            send = torch.from_numpy(np.concatenate(parts) if parts else np.zeros(0))
            n_recv = sum(int(((int(m) >> octv) & 1).sum()) for m in hl["recv_mask"])
            recv[p] = torch.empty(n_recv, dtype=torch.float64)
            reqs += [dist.isend(send, p), dist.irecv(recv[p], p)]
        for q in reqs:
            q.wait()
        dests = {}
        if fused:      # the senders' destinations travel with the data: the receiver places every chunk where it was pushed
            for p, hl in halos.items():
                theirs = torch.empty(len(hl["recv_slab"]), dtype=torch.int64)
                rq = [dist.isend(torch.from_numpy(np.ascontiguousarray(hl["send_dest"], np.int64)), p), dist.irecv(theirs, p)]
                for q in rq:
                    q.wait()
                dests[p] = theirs.numpy()
        for p, hl in halos.items():
            buf, at = recv[p].numpy(), 0
            where = dests[p] if fused else hl["recv_slab"]
            assert sorted(where.tolist()) == sorted(hl["recv_slab"].tolist())
            mask_of = {int(s): int(m) for s, m in zip(hl["recv_slab"], hl["recv_mask"])}
            for s in where:
                m = mask_of[int(s)]
                sel = (int(m) >> octv) & 1 == 1
                k = int(sel.sum())
                f[row[int(slabs[s])], sel] = buf[at:at + k]
                at += k
            assert at == buf.size
        f = o.step(f, case.dt, 1)
    inner_rows = np.array([row[int(l)] for l in slabs[:n_in]], np.int64)
    out.put((rank, slabs[:n_in].copy(), f[inner_rows].copy()))
    dist.barrier()
    dist.destroy_process_group()
    B.ufs_dvm_destroy(h)


@pytest.mark.parametrize("which,nsteps,fused", [("random_periodic", 4, False), ("small3_walls_solid", 2, False),
                                                ("small3_walls_solid", 2, True)])
def test_two_rank_gloo_run_stitched_equals_the_one_domain_oracle(which, nsteps, fused):
    from oracle.dvm_oracle import Oracle
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_worker, args=(r, 2, port, which, nsteps, out, fused)) for r in range(2)]
    for p in procs:
        p.start()
    got = [out.get(timeout=600) for _ in range(2)]
    for p in procs:
        p.join(timeout=600)
        assert p.exitcode == 0
    case = _cases()[which]
    f0 = inputs.initial_f(case)
    ref = Oracle(case).step(f0, case.dt, nsteps)
    glob_row = np.full(case.n_leaves, -1, np.int64); glob_row[case.kinetic_leaves()] = np.arange(ref.shape[0])
    seen = np.zeros(ref.shape[0], bool)
    for rank, leaves, f in got:
        rows = glob_row[leaves]
        assert not seen[rows].any()
        seen[rows] = True
        assert np.array_equal(f, ref[rows]), f"rank {rank}: stitched part differs from the one-domain oracle"
    assert seen.all()
