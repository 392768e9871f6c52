"""The partitioned DVM step on the device (ufs_dvm_create_part, ufs_dvm_halo_pack / unpack / done; SURVEY.md 8(e),
8(f)-2): R ranks emulated on ONE device and one stream -- every rank's handle steps its own part, the
ghost chunks travel through the library's pack and unpack kernels with a device copy in between (no kernel waits on
another one) -- and the stitched result must match the one-domain CPU oracle within the storage type's tolerance, on
meshes with 2:1 faces, walls, SOLID leaves, the kinetic/fluid mask and fp32 storage."""
import numpy as np
import pytest

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from paper_1503_00707_b200.partition import RankStepper, exchange_local, setup_push_local, step_pushed_local
from tests.helpers import assert_moments_close, rel_linf

pytestmark = pytest.mark.gpu
TOL = {inputs.STORE_F64: 1e-12, inputs.STORE_F32: 2e-5}


def _run_partitioned(case, n_ranks, nsteps, w_fluid=0.0, push=False, push_sums=True, own_sums=False):
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, n_ranks, 1.0, w_fluid)
    f0 = inputs.initial_f(case)
    if case.storage == inputs.STORE_F32:
        f0 = f0.astype(np.float32).astype(np.float64)
    kin = case.kinetic_leaves()
    glob_row = np.full(case.n_leaves, -1, np.int64); glob_row[kin] = np.arange(kin.size)
    ranks = [RankStepper(case, rol, r, n_ranks) for r in range(n_ranks)]
    keep_sums = []
    try:
        for r in ranks:
            assert B.ufs_dvm_kernel_name(r.h) == "k_tiles"
            if own_sums:
                # the carried sums in caller-owned arrays (ufs_dvm_sums_use; what a symmetric allocation would be)
                import torch
                mine = [torch.full((r.n_inner + r.n_ghost, 36), float("nan"), dtype=torch.float64, device=r.device) for _ in range(2)]
                B.ufs_dvm_sums_use(r.h, mine[0].data_ptr(), mine[1].data_ptr())
                assert B.ufs_dvm_sums_dev(r.h) == (mine[0].data_ptr(), mine[1].data_ptr())
                keep_sums.append(mine)
            r.load_canonical(f0[glob_row[r.inner_leaves]])
        if push:
            # fused exchange: one ordinary exchange for the first step's ghosts, from then on the step kernels write the
            # boundary cells into the peers' ghost slabs themselves -- no pack, copy or unpack launch after this point
            setup_push_local(ranks, push_sums=push_sums)
            exchange_local(ranks)
            before = [B.ufs_dvm_launch_count(r.h) for r in ranks]
            for _ in range(nsteps):
                step_pushed_local(ranks, case.dt)
            for r, b in zip(ranks, before):
                # k_prep, k_tiles on the boundary tiles, k_tiles on the rest; the ghost sums only if the peers do not push them
                per_step = 3 + (1 if r.n_ghost and not push_sums else 0)
                first = 1 if r.n_inner else 0                  # the sums pass of the initial f
                assert B.ufs_dvm_launch_count(r.h) - b <= nsteps * per_step + first
        else:
            for _ in range(nsteps):
                exchange_local(ranks)
                for r in ranks:
                    r.step(case.dt, 1)
        f = np.empty_like(f0)
        mom = np.empty((5, kin.size))
        for r in ranks:
            r.sync()
            f[glob_row[r.inner_leaves]] = r.read_canonical()
            mom[:, glob_row[r.inner_leaves]] = r.moments()
        sent = sum(r.halo_bytes()[0] for r in ranks)
        for r, mine in zip(ranks, keep_sums):
            cur = B.ufs_dvm_current(r.h)
            rows = mine[cur][:r.n_inner, :35].cpu().numpy()
            assert np.all(np.isfinite(rows)) and np.all(rows[:, 0] > 0)     # the step kernel wrote the caller's arrays
        return f0, f, mom, sent
    finally:
        for r in ranks:
            r.close()


@pytest.mark.parametrize("cfg,n_ranks", [(3, 2), (3, 3), (4, 2), (5, 3)])
def test_partitioned_step_matches_the_one_domain_oracle(cfg, n_ranks):
    case = inputs.small(cfg)
    nsteps = 3
    f0, f, mom, sent = _run_partitioned(case, n_ranks, nsteps, w_fluid=0.02)
    assert sent > 0
    o = Oracle(case)
    f_ref = o.step(f0, case.dt, nsteps)
    tol = TOL[case.storage]
    assert np.all(np.isfinite(f))
    assert rel_linf(f, f_ref) <= tol
    assert_moments_close(mom, o.moments(f_ref), tol, eps_storage=6e-8 if case.storage == inputs.STORE_F32 else 2.3e-16)


def test_one_rank_partition_is_the_plain_step():
    """n_ranks = 1: no ghosts, no exchange; bit-equal to the unpartitioned handle."""
    case = inputs.small(3)
    f0, f, mom, sent = _run_partitioned(case, 1, 2)
    assert sent == 0
    st = B.DvmStepper(case)
    st.load_canonical(f0)
    st.step(case.dt, 2)
    st.sync()
    assert np.array_equal(st.read_canonical(), f)
    st.close()


def test_step_without_fresh_ghosts_is_refused():
    case = inputs.small(3)
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, 2)
    ranks = [RankStepper(case, rol, r, 2) for r in range(2)]
    try:
        f0 = inputs.initial_f(case)
        kin = case.kinetic_leaves()
        glob_row = np.full(case.n_leaves, -1, np.int64); glob_row[kin] = np.arange(kin.size)
        for r in ranks:
            r.load_canonical(f0[glob_row[r.inner_leaves]])
        with pytest.raises(B.UfsDvmError) as e:
            ranks[0].step(case.dt, 1)                     # no exchange yet
        assert e.value.code == B.EINVAL and "ghost" in str(e.value)
        exchange_local(ranks)
        with pytest.raises(B.UfsDvmError):
            ranks[0].step(case.dt, 2)                     # one step at a time
        for r in ranks:
            r.step(case.dt, 1)
        with pytest.raises(B.UfsDvmError):
            ranks[0].step(case.dt, 1)                     # stale again after the step
    finally:
        for r in ranks:
            r.close()


@pytest.mark.parametrize("push", [False, True])
def test_partitioned_config3_at_stated_size_four_ranks(push):
    """Config 3 literal (26 312 leaves: inflow, outflow, specular sides, SOLID body, 2:1 faces) cut into four ranks on one
    device, 5 steps with the ghost exchange before each (packed, or fused into the step kernel); the stitched whole field
    against the one-domain oracle."""
    case = inputs.config3(lmax=7)
    f0, f, mom, sent = _run_partitioned(case, 4, 5, push=push)
    assert sent > 0
    o = Oracle(case)
    f_ref = o.step(f0, case.dt, 5)
    assert np.all(np.isfinite(f))
    assert rel_linf(f, f_ref) <= 1e-12
    assert_moments_close(mom, o.moments(f_ref), 1e-12)


@pytest.mark.parametrize("cfg,n_ranks,push_sums", [(3, 2, True), (3, 3, False), (4, 2, True), (4, 4, False), (5, 3, True),
                                                   (5, 3, False)])
def test_fused_exchange_matches_the_one_domain_oracle(cfg, n_ranks, push_sums):
    """ufs_dvm_halo_push_setup: the step kernel stores the boundary cells into the peers' ghost slabs (peer memory; here the
    ranks share one device) -- 2:1 faces, walls, a SOLID body, the kinetic/fluid mask (k_tiles' FLUID instantiation), fp32;
    with the cells' sums pushed as well, or formed from the ghost slabs by ufs_dvm_halo_done."""
    case = inputs.small(cfg)
    nsteps = 4
    f0, f, mom, sent = _run_partitioned(case, n_ranks, nsteps, w_fluid=0.02, push=True, push_sums=push_sums)
    o = Oracle(case)
    f_ref = o.step(f0, case.dt, nsteps)
    tol = TOL[case.storage]
    assert np.all(np.isfinite(f))
    assert rel_linf(f, f_ref) <= tol
    assert_moments_close(mom, o.moments(f_ref), tol, eps_storage=6e-8 if case.storage == inputs.STORE_F32 else 2.3e-16)


def test_fused_exchange_is_bit_equal_to_the_packed_exchange():
    """The same rows reach the same ghost slabs and the same owner's sums reach the same ghost rows either way: the two
    exchanges give bit-identical fields."""
    case = inputs.small(3)
    _, f_a, mom_a, _ = _run_partitioned(case, 3, 3)
    _, f_b, mom_b, _ = _run_partitioned(case, 3, 3, push=True)
    assert np.array_equal(f_a, f_b)
    assert np.array_equal(mom_a, mom_b)


@pytest.mark.parametrize("push,own_sums", [(False, False), (True, False), (True, True)])
@pytest.mark.parametrize("cfg,n_ranks", [(3, 3), (4, 2), (5, 3)])
def test_partitioned_run_is_bit_identical_to_the_one_domain_run(cfg, n_ranks, push, own_sums):
    """The ghost rows of the sums hold the owners' own carried sums (behind the chunks of the packed exchange, or pushed by
    the peers' step kernels), so a cell sees exactly what it sees in the unpartitioned run -- the same f in its upwind
    sources, the same sums behind its Maxwellian -- and the stitched field is the one-domain device run bit for bit
    (walls, SOLID body, 2:1 faces; fp32 storage; the kinetic/fluid mask)."""
    case = inputs.small(cfg)
    nsteps = 4
    f0, f, mom, _ = _run_partitioned(case, n_ranks, nsteps, w_fluid=0.02, push=push, own_sums=own_sums)
    st = B.DvmStepper(case)
    try:
        st.load_canonical(f0)
        st.step(case.dt, nsteps)
        st.sync()
        assert np.array_equal(st.read_canonical(), f)
        assert np.array_equal(st.moments(), mom)
    finally:
        st.close()


def test_fused_exchange_push_entries_cover_the_send_lists():
    case = inputs.small(3)
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, 3)
    ranks = [RankStepper(case, rol, r, 3) for r in range(3)]
    try:
        setup_push_local(ranks)
        for r in ranks:
            t = B.ufs_dvm_tiles(r.h)
            counts = np.array([[(int(w) >> (4 * c)) & 15 for c in range(8)] for w in t["push_counts"]])
            assert np.all(counts[np.arange(8)[None, :] >= t["nc"][:, None]] == 0)
            n_send = sum(B.ufs_dvm_halo(r.h, p)["send_slab"].size for p in range(3))
            assert counts.sum() == n_send
            # the tiles with entries come first (they are stepped first, by the pushing instantiation)
            has = counts.sum(axis=1) > 0
            assert 0 < has.sum() < t["n_tiles"] and np.all(has[:has.sum()]) and not np.any(has[has.sum():])
            # every inner slab is in exactly one tile, whatever the order
            cover = np.zeros(r.n_inner, np.int64)
            for i in range(t["n_tiles"]):
                cover[t["s0"][i]:t["s0"][i] + t["nc"][i]] += 1
            assert np.all(cover == 1)
            # a tile's entries follow the previous tile's
            assert np.array_equal(t["push_first"], np.concatenate([[0], np.cumsum(counts.sum(axis=1))[:-1]]))
            # per cell: as many entries as peers that list it
            per_slab = np.zeros(r.n_inner, np.int64)
            for p in range(3):
                np.add.at(per_slab, B.ufs_dvm_halo(r.h, p)["send_slab"], 1)
            got = np.zeros(r.n_inner, np.int64)
            for i in range(t["n_tiles"]):
                got[t["s0"][i]:t["s0"][i] + t["nc"][i]] = counts[i, :t["nc"][i]]
            assert np.array_equal(got, per_slab)
    finally:
        for r in ranks:
            r.close()


def test_fused_exchange_refuses_what_it_cannot_serve():
    case = inputs.small(3)
    desc, keep = B.make_desc(case)
    st = B.DvmStepper(case)                                   # not partitioned
    try:
        with pytest.raises(B.UfsDvmError) as e:
            B.ufs_dvm_halo_push_setup(st.h, [None], [None], [None])
        assert e.value.code == B.EINVAL
    finally:
        st.close()
    rol = B.ufs_dvm_partition(desc, 2)
    ranks = [RankStepper(case, rol, r, 2) for r in range(2)]
    try:
        with pytest.raises(B.UfsDvmError) as e:               # rank 1 needs cells of rank 0 but no buffers are given
            B.ufs_dvm_halo_push_setup(ranks[0].h, [None, None], [None, None], [None, None])
        assert e.value.code == B.EINVAL and "rank 1" in str(e.value)
    finally:
        for r in ranks:
            r.close()


def test_distributed_plumbing_of_the_fused_exchange_with_a_one_rank_nccl_group():
    """setup_push_distributed / step_pushed_distributed with the only process group one GPU allows (world size 1, NCCL):
    f and the carried sums in torch's symmetric memory, rendezvous, ufs_dvm_sums_use, the recv lists by all_gather_object,
    the stream barrier.  No peer exists, so nothing crosses a wire; the result must be the plain step's, bit for bit."""
    import os
    import socket
    import torch
    import torch.distributed as dist
    pytest.importorskip("torch.distributed._symmetric_memory")
    from paper_1503_00707_b200.partition import exchange_distributed, setup_push_distributed, step_pushed_distributed
    assert not dist.is_initialized()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        case = inputs.small(3)
        desc, keep = B.make_desc(case)
        rol = B.ufs_dvm_partition(desc, 1)
        r = RankStepper(case, rol, 0, 1, symmetric=True)
        st = B.DvmStepper(case)
        try:
            assert B.ufs_dvm_sums_dev(r.h) == (r.sums[0].data_ptr(), r.sums[1].data_ptr())
            assert int(r.f_symm[0].buffer_ptrs[0]) == r.f[0].data_ptr()
            f0 = inputs.initial_f(case)
            r.load_canonical(f0)
            setup_push_distributed(r)
            exchange_distributed(r)
            for _ in range(3):
                step_pushed_distributed(r, case.dt)
            r.sync()
            st.load_canonical(f0)
            st.step(case.dt, 3)
            st.sync()
            assert np.array_equal(st.read_canonical(), r.read_canonical())
        finally:
            r.close()
            st.close()
    finally:
        dist.destroy_process_group()
