"""Mesh change on the device (ufs_dvm_remesh) against the oracle's remap
(reading G20, pinned in tests/test_oracle_remap_pins.py): element by element on small tree pairs (fp64 and fp32
storage, refinement and coarsening over several levels, FLUID -> KINETIC leaves), then stepping on from the carried
state, and at stated size from config 3 (l_max 7) to config 3' (l_max 8)."""
import gc

import numpy as np
import pytest

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import harness, inputs
from tests.helpers import assert_moments_close, gpu_field_error, periodic_case, random_tree, rel_linf

pytestmark = pytest.mark.gpu
P = (True, True, True)


def _case(seed, p_split, nv=(24, 24, 24), kind_fn=None, fluid=False, storage=inputs.STORE_F64):
    lv, ijk = random_tree(np.random.default_rng(seed), 1, 3, P, p_split)
    kind = np.zeros(lv.shape[0], np.uint8) if kind_fn is None else kind_fn(lv, ijk)
    fm = None
    if fluid:
        c = (ijk + 0.5) / (2.0 ** lv)[:, None]
        fm = np.stack([1 + 0.3 * np.sin(2 * np.pi * c[:, 0]), 0.2 * np.cos(2 * np.pi * c[:, 1]), 0 * c[:, 0] + 0.1,
                       -0.1 * np.sin(2 * np.pi * c[:, 2]), 1 + 0.2 * np.cos(2 * np.pi * c[:, 0])], axis=1)
    case = periodic_case(lv, ijk, nv=nv, vlim=5.0, kn=0.2, kind=kind, fluid_moments=fm)
    case.storage = storage
    return case


def _remesh_and_compare(old, new, tol_map, tol_step, nsteps=2, seed=0):
    rng = np.random.default_rng(seed)
    kin = old.kinetic_leaves()
    f_old = inputs.maxwellian_canonical(old, old.prim0[kin]) * (1 + 0.3 * rng.uniform(-1, 1, (kin.size, old.Nv)))
    if old.storage == inputs.STORE_F32:
        f_old = f_old.astype(np.float32).astype(np.float64)
    st_old = B.DvmStepper(old)
    st_old.load_canonical(f_old)
    st_new = B.DvmStepper(new, remesh_from=st_old)
    counts = st_new.remesh_counts
    f_map = st_new.read_canonical()
    o_old, o_new = Oracle(old), Oracle(new)
    ref = o_new.remap_from(o_old, f_old)
    assert rel_linf(f_map, ref) <= tol_map
    # the carried state is a state like any other: step on (the velocity sums are rebuilt from it)
    st_new.step(new.dt, nsteps)
    st_new.sync()
    start = f_map if new.storage == inputs.STORE_F32 else ref     # fp32: the oracle starts from the device's bits
    f_ref = o_new.step(start, new.dt, nsteps)
    assert rel_linf(st_new.read_canonical(), f_ref) <= tol_step
    assert_moments_close(st_new.moments(), o_new.moments(f_ref), tol_step,
                         eps_storage=6e-8 if new.storage == inputs.STORE_F32 else 2.3e-16)
    # the old handle is still usable
    st_old.step(old.dt, 1)
    st_old.sync()
    st_new.close(); st_old.close()
    return counts


@pytest.mark.parametrize("so,sn,po,pn", [(1, 2, 0.3, 0.2), (3, 4, 0.0, 0.5), (5, 6, 0.5, 0.0)])
def test_remesh_matches_oracle_fp64(so, sn, po, pn):
    counts = _remesh_and_compare(_case(so, po), _case(sn, pn), 1e-15, 1e-12, seed=so)
    assert counts.sum() > 0 and counts[3] == 0
    if po == 0.0:
        assert counts[1] > 0 and counts[2] == 0        # only refinement
    if pn == 0.0:
        assert counts[2] > 0 and counts[1] == 0        # only coarsening


def test_remesh_matches_oracle_fp32_storage():
    old, new = _case(7, 0.3, storage=inputs.STORE_F32), _case(8, 0.3, storage=inputs.STORE_F32)
    _remesh_and_compare(old, new, 1e-7, 2e-5, seed=7)


def test_remesh_unchanged_mesh_is_a_copy():
    case = _case(9, 0.3)
    rng = np.random.default_rng(1)
    f = inputs.maxwellian_canonical(case, case.prim0) * (1 + 0.3 * rng.uniform(-1, 1, (case.n_leaves, case.Nv)))
    a = B.DvmStepper(case); a.load_canonical(f)
    b = B.DvmStepper(case, remesh_from=a)
    assert b.remesh_counts.tolist() == [case.n_leaves, 0, 0, 0]
    assert np.array_equal(b.read_canonical(), f)
    a.close(); b.close()


def test_remesh_mask_change_fluid_to_kinetic():
    half = lambda lv, ijk: np.where((ijk + 0.5)[:, 0] / 2.0 ** lv < 0.5, inputs.CELL_FLUID, inputs.CELL_KINETIC).astype(np.uint8)
    other = lambda lv, ijk: np.where((ijk + 0.5)[:, 1] / 2.0 ** lv < 0.3, inputs.CELL_FLUID, inputs.CELL_KINETIC).astype(np.uint8)
    old, new = _case(11, 0.3, kind_fn=half, fluid=True), _case(12, 0.25, kind_fn=other, fluid=True)
    counts = _remesh_and_compare(old, new, 1e-15, 1e-12, seed=11)
    assert counts[3] > 0


def test_remesh_refuses_other_velocity_grid_and_solid_sources():
    old = _case(13, 0.3)
    a = B.DvmStepper(old)
    a.load_canonical(inputs.maxwellian_canonical(old, old.prim0))
    with pytest.raises(B.UfsDvmError) as e:
        B.DvmStepper(_case(13, 0.3, nv=(12, 12, 12)), remesh_from=a)
    assert e.value.code == B.EINVAL
    a.close()
    blk = lambda lv, ijk: np.where(np.abs((ijk + 0.5) / (2.0 ** lv)[:, None] - 0.5).max(axis=1) < 0.2, inputs.CELL_SOLID, inputs.CELL_KINETIC).astype(np.uint8)
    old = _case(14, 0.3, kind_fn=blk)
    a = B.DvmStepper(old)
    a.load_canonical(inputs.maxwellian_canonical(old, old.prim0[old.kinetic_leaves()]))
    with pytest.raises(B.UfsDvmError) as e:
        B.DvmStepper(_case(14, 0.3), remesh_from=a)
    assert e.value.code == B.EINVAL and "SOLID" in str(e.value)
    a.close()


def test_remesh_config3_to_config3_l8_at_stated_size():
    """26 312 -> 152 240 kinetic leaves (sphere octree refined one more level around the body; the body itself is the
    old mesh's staircase, inputs.with_body_of: the l_max 8 sampling of the sphere would uncover 1948 leaves inside old
    SOLID leaves, which a mesh change refuses), fp64, after 3 steps on the coarse mesh; the whole new field against the
    oracle's remap of the device's old field."""
    import torch
    old = inputs.config3(lmax=7)
    new = inputs.with_body_of(old, inputs.config3(lmax=8))
    st_old = B.DvmStepper(old)
    harness.fill_initial_f_device(st_old, old)
    st_old.step(old.dt, 3)
    st_old.sync()
    f_old = st_old.read_canonical()
    st_new = B.DvmStepper(new, remesh_from=st_old)
    counts = st_new.remesh_counts
    assert counts.sum() == st_new.n_kinetic and counts[1] > 0
    ref = Oracle(new).remap_from(Oracle(old), f_old)
    dmax, rmax = gpu_field_error(st_new, ref)
    assert dmax <= 1e-15 * rmax
    st_new.step(new.dt, 1)           # and the new handle steps
    st_new.sync()
    for st in (st_new, st_old):
        st.close(); st.f = None; st.mom = None
    gc.collect(); torch.cuda.empty_cache()
