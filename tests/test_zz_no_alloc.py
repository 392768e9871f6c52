"""ufs_dvm_moments_static (include/ufs_dvm.h): the moments of f without any allocation in the library -- the per-cell
velocity sums go through a fixed array in the library's device image (UFS_DVM_STATIC_MAX_CELLS cells) instead of the
cudaMalloc'ed buffer of ufs_dvm_moments.  Checked against the existing path (ufs_dvm_moments, which reads the sums the
step kernel carries) on two calls in a row with different f, so that a call that read what the previous one left in
the shared array would fail.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from tests.helpers import assert_moments_close

pytestmark = pytest.mark.gpu
TOL = {inputs.STORE_F64: 1e-12, inputs.STORE_F32: 2e-5}


@pytest.mark.parametrize("cfg", [3, 4])          # fp64 storage with walls, a SOLID body and 2:1 faces; fp32 storage
def test_static_moments_match_the_existing_path_twice_in_a_row(cfg):
    case = inputs.small(cfg)
    st = B.DvmStepper(case)
    try:
        assert st.n_kinetic <= B.STATIC_MAX_CELLS
        f0 = inputs.initial_f(case)
        if st.storage == inputs.STORE_F32:
            f0 = f0.astype(np.float32).astype(np.float64)
        st.load_canonical(f0)
        eps = 6e-8 if st.storage == inputs.STORE_F32 else 2.3e-16
        seen = []
        for call in range(2):
            st.step(case.dt, 2)
            before = B.ufs_dvm_launch_count(st.h)
            got = st.moments_static().copy()
            assert B.ufs_dvm_launch_count(st.h) == before + 2          # the sums pass and the moments kernel
            ref = st.moments().copy()
            assert np.all(np.isfinite(got))
            assert_moments_close(got, ref, TOL[st.storage], eps_storage=eps, what=f"call {call}")
            seen.append(got)
        assert not np.array_equal(seen[0], seen[1])                    # the two calls saw different f
        # the input may be any buffer in the handle's layout: the current f passed explicitly, bit for bit the same
        cur = B.ufs_dvm_current(st.h)
        assert np.array_equal(st.moments_static(st.f[cur]), seen[1])
        # ... and the other buffer holds the f of one step earlier: a different field
        assert not np.array_equal(st.moments_static(st.f[cur ^ 1]), seen[1])
        # the carried sums were neither read nor changed: the step goes on as if nothing had been called
        st.step(case.dt, 1)
        assert_moments_close(st.moments_static(), st.moments(), TOL[st.storage], eps_storage=eps, what="after")
    finally:
        st.close()


def test_static_moments_refuse_more_cells_than_the_fixed_array_holds():
    case = inputs.config3(lmax=7)                 # 26 312 kinetic cells > 8192
    st = B.DvmStepper(case, storage=inputs.STORE_F32)
    try:
        assert st.n_kinetic > B.STATIC_MAX_CELLS
        before = B.ufs_dvm_launch_count(st.h)
        with pytest.raises(B.UfsDvmError) as e:
            B.ufs_dvm_moments_static(st.h, None, st.mom.data_ptr())
        assert e.value.code == B.EINVAL
        assert str(B.STATIC_MAX_CELLS) in str(e.value) and "ufs_dvm_moments" in str(e.value)
        assert B.ufs_dvm_launch_count(st.h) == before                  # nothing was enqueued
        st.sync()                                                      # and the handle is still usable
    finally:
        st.close()
