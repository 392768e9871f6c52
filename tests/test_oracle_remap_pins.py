"""Pins of the oracle's mesh-change map (oracle_dvm_remap; reading G20: the new value
is the volume average over the new leaf of the old piecewise-constant field).  Each pin is fixed by that definition,
not by the oracle: an independent dense-grid average, exact invariants, the closed-form Maxwellian of a FLUID leaf."""
import numpy as np
import pytest

from oracle.dvm_oracle import Oracle, OracleError
from paper_1503_00707_b200 import inputs
from tests.helpers import periodic_case, random_tree

P = (True, True, True)
NV = (4, 4, 4)


def _case(seed, p_split=0.3, base=1, lmax=4, kind_fn=None, fluid=False):
    lv, ijk = random_tree(np.random.default_rng(seed), base, lmax, P, p_split)
    kind = np.zeros(lv.shape[0], np.uint8) if kind_fn is None else kind_fn(lv, ijk)
    fm = None
    if fluid:
        c = (ijk + 0.5) / (2.0 ** lv)[:, None]
        fm = np.stack([1 + 0.3 * np.sin(2 * np.pi * c[:, 0]), 0.2 * np.cos(2 * np.pi * c[:, 1]), 0 * c[:, 0] + 0.1,
                       -0.1 * np.sin(2 * np.pi * c[:, 2]), 1 + 0.2 * np.cos(2 * np.pi * c[:, 0])], axis=1)
    return periodic_case(lv, ijk, nv=NV, kind=kind, fluid_moments=fm)


def _noisy_f(case, seed):
    rng = np.random.default_rng(seed)
    kin = case.kinetic_leaves()
    return inputs.maxwellian_canonical(case, case.prim0[kin]) * (1 + 0.5 * rng.uniform(-1, 1, (kin.size, case.Nv)))


def _dense(case, rows_value, lmax):
    """The piecewise-constant field of the kinetic leaves on the uniform level-lmax grid: [N,N,N,Nv] (NaN elsewhere)."""
    N = 1 << lmax
    out = np.full((N, N, N, case.Nv), np.nan)
    kin = case.kinetic_leaves()
    for r, j in enumerate(kin.tolist()):
        s = 1 << (lmax - int(case.level[j]))
        i0 = case.ijk[j].astype(np.int64) * s
        out[i0[0]:i0[0] + s, i0[1]:i0[1] + s, i0[2]:i0[2] + s] = rows_value[r]
    return out


@pytest.mark.parametrize("seed_old,seed_new", [(1, 2), (3, 4), (5, 5)])
def test_remap_equals_the_dense_grid_volume_average(seed_old, seed_new):
    old, new = _case(seed_old), _case(seed_new, p_split=0.2)
    f_old = _noisy_f(old, 10 + seed_old)
    got = Oracle(new).remap_from(Oracle(old), f_old)
    lmax = int(max(old.level.max(), new.level.max()))
    dense = _dense(old, f_old, lmax)
    kin = new.kinetic_leaves()
    refs = np.empty_like(got)
    for r, j in enumerate(kin.tolist()):
        s = 1 << (lmax - int(new.level[j]))
        i0 = new.ijk[j].astype(np.int64) * s
        refs[r] = dense[i0[0]:i0[0] + s, i0[1]:i0[1] + s, i0[2]:i0[2] + s].reshape(-1, new.Nv).mean(axis=0)
    assert np.abs(got - refs).max() <= 4e-16 * np.abs(refs).max()
    if seed_old == seed_new:                     # same tree rule, other split probability: still a real change
        assert new.n_leaves != old.n_leaves


def test_unchanged_mesh_is_the_identity_bit_for_bit():
    case = _case(7)
    f = _noisy_f(case, 1)
    assert np.array_equal(Oracle(case).remap_from(Oracle(case), f), f)


def test_remap_conserves_every_velocity_node():
    """sum_j V_j f_ij over the domain is the same before and after (both meshes tile the cube)."""
    old, new = _case(11), _case(12, p_split=0.15)
    f_old = _noisy_f(old, 3)
    f_new = Oracle(new).remap_from(Oracle(old), f_old)
    v_old = 8.0 ** (-old.level[old.kinetic_leaves()].astype(np.float64))
    v_new = 8.0 ** (-new.level[new.kinetic_leaves()].astype(np.float64))
    a, b = v_old @ f_old, v_new @ f_new
    assert np.abs(a - b).max() <= 1e-14 * np.abs(a).max()


def test_refine_then_coarsen_is_the_identity_to_roundoff():
    coarse = _case(21, lmax=3)
    lv, ijk = inputs.build_tree(4, 4, {}, P)            # every leaf of `coarse` refined down to level 4
    fine = periodic_case(lv, ijk, nv=NV)
    oc, of = Oracle(coarse), Oracle(fine)
    f = _noisy_f(coarse, 5)
    up = of.remap_from(oc, f)
    # injection: every fine leaf carries exactly its coarse ancestor's values
    assert set(np.unique(up[:, 0]).tolist()) <= set(f[:, 0].tolist())
    back = oc.remap_from(of, up)                       # mean of equal values: the identity to round-off
    assert np.abs(back - f).max() <= 1e-14 * np.abs(f).max()       # up to 512 equal terms summed in sequence


def test_uniform_state_stays_uniform():
    old, new = _case(31), _case(32)
    row = inputs.maxwellian_canonical(old, np.array([[1.3, 0.2, -0.1, 0.3, 0.9]]))[0]
    f_old = np.tile(row, (old.n_leaves, 1))
    f_new = Oracle(new).remap_from(Oracle(old), f_old)
    assert np.abs(f_new - row).max() <= 2e-16 * row.max()


def test_new_kinetic_leaf_over_an_old_fluid_leaf_gets_its_maxwellian():
    half = lambda lv, ijk: np.where((ijk + 0.5)[:, 0] / 2.0 ** lv < 0.5, inputs.CELL_FLUID, inputs.CELL_KINETIC).astype(np.uint8)
    old = _case(41, kind_fn=half, fluid=True)
    new = _case(41, fluid=True)                          # same tree, everything kinetic now
    f_old = _noisy_f(old, 2)
    f_new = Oracle(new).remap_from(Oracle(old), f_old)
    was_fluid = old.kind == inputs.CELL_FLUID
    ref = inputs.maxwellian_canonical(old, old.fluid_moments[was_fluid])
    assert np.abs(f_new[was_fluid] - ref).max() <= 1e-15 * ref.max()
    assert np.array_equal(f_new[~was_fluid], f_old)


def test_new_kinetic_leaf_over_a_solid_leaf_is_refused():
    blk = lambda lv, ijk: np.where(np.abs((ijk + 0.5) / (2.0 ** lv)[:, None] - 0.5).max(axis=1) < 0.2, inputs.CELL_SOLID, inputs.CELL_KINETIC).astype(np.uint8)
    old = _case(51, kind_fn=blk)
    assert (old.kind == inputs.CELL_SOLID).any()
    new = _case(51)
    with pytest.raises(OracleError):
        Oracle(new).remap_from(Oracle(old), _noisy_f(old, 1))
