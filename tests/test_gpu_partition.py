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
from paper_1503_00707_b200.partition import RankStepper, exchange_local
from tests.helpers import assert_moments_close, rel_linf

pytestmark = pytest.mark.gpu
TOL = {inputs.STORE_F64: 1e-12, inputs.STORE_F32: 2e-5}


def _run_partitioned(case, n_ranks, nsteps, w_fluid=0.0):
    desc, keep = B.make_desc(case)
    rol = B.ufs_dvm_partition(desc, n_ranks, 1.0, w_fluid)
    f0 = inputs.initial_f(case)
    if case.storage == inputs.STORE_F32:
        f0 = f0.astype(np.float32).astype(np.float64)
    kin = case.kinetic_leaves()
    glob_row = np.full(case.n_leaves, -1, np.int64); glob_row[kin] = np.arange(kin.size)
    ranks = [RankStepper(case, rol, r, n_ranks) for r in range(n_ranks)]
    try:
        for r in ranks:
            assert B.ufs_dvm_kernel_name(r.h) == "k_tiles"
            r.load_canonical(f0[glob_row[r.inner_leaves]])
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


def test_partitioned_config3_at_stated_size_four_ranks():
    """Config 3 literal (26 312 leaves: inflow, outflow, specular sides, SOLID body, 2:1 faces) cut into four ranks on one
    device, 5 steps with the ghost exchange before each; the stitched whole field against the one-domain oracle."""
    case = inputs.config3(lmax=7)
    f0, f, mom, sent = _run_partitioned(case, 4, 5)
    assert sent > 0
    o = Oracle(case)
    f_ref = o.step(f0, case.dt, 5)
    assert np.all(np.isfinite(f))
    assert rel_linf(f, f_ref) <= 1e-12
    assert_moments_close(mom, o.moments(f_ref), 1e-12)
