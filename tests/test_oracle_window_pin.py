"""Pin of the oracle's `window` mode (oracle/dvm_oracle.c: a missing neighbour becomes a zero-gradient ghost and the
coverage check is skipped).  The full-size GPU parity of config 4 rests on it (windowed oracle), so it is
pinned here against the FULL oracle, which the pins of tests/test_oracle_pins.py fix: after S steps the value at a leaf
depends only on the leaves within S face-rings of it (first-order upwind stencil, Eq. 2; the collision
step is local), so stepping the S-ring sub-mesh in window mode must reproduce the full run at the centre BIT FOR BIT
-- same neighbours, same areas, same order of the sums.  Centres are chosen next to a 2:1 face (both sides), a SOLID
leaf, a FLUID leaf and a domain wall of every kind."""
import numpy as np
import pytest

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import harness, inputs
from tests.helpers import periodic_case, random_tree


def _stratified_centres(case, mesh, rng, per_class=2):
    """Kinetic leaves by what they touch: coarse / fine side of a 2:1 face, SOLID, FLUID, domain wall, interior."""
    kin = np.nonzero(case.kind == inputs.CELL_KINETIC)[0]
    owner, neigh, _, _, ratio = mesh.faces()
    classes = {"coarse_side": np.concatenate([owner[ratio == 1], neigh[ratio == -1]]),
               "fine_side": np.concatenate([neigh[ratio == 1], owner[ratio == -1]])}
    touch = {inputs.CELL_SOLID: [], inputs.CELL_FLUID: []}
    for j in kin.tolist():
        for q in mesh.leaf_neighbours([j]).tolist():
            if case.kind[q] in touch:
                touch[int(case.kind[q])].append(j)
    classes["next_to_solid"] = np.array(touch[inputs.CELL_SOLID], np.int64)
    classes["next_to_fluid"] = np.array(touch[inputs.CELL_FLUID], np.int64)
    n = (1 << case.level.astype(np.int64))
    at_wall = ((case.ijk == 0) | (case.ijk.astype(np.int64) == (n - 1)[:, None])).any(axis=1)
    classes["domain_wall"] = np.nonzero(at_wall)[0]
    classes["any"] = kin
    out = []
    for name, ids in classes.items():
        ids = np.intersect1d(ids, kin)
        if ids.size:
            out += [(name, int(c)) for c in rng.choice(ids, min(per_class, ids.size), replace=False)]
    return out


def _check_window_equals_full(case, f0, nsteps_list=(1, 2, 3), per_class=2, seed=0):
    full = Oracle(case)
    kin = case.kinetic_leaves()
    row_of_leaf = np.full(case.n_leaves, -1, np.int64)
    row_of_leaf[kin] = np.arange(kin.size)
    centres = _stratified_centres(case, full, np.random.default_rng(seed), per_class)
    assert centres
    seen = set()
    for S in nsteps_list:
        f_full = full.step(f0, case.dt, S)
        m_full = full.moments(f_full)
        for name, c in centres:
            ids = harness.window_leaves(case, c, S, full.leaf_neighbours)
            assert ids.size < case.n_leaves or S >= 3      # a real window, not the whole mesh
            sub = harness.sub_case(case, ids)
            kin_ids = ids[case.kind[ids] == inputs.CELL_KINETIC]
            o = Oracle(sub, window=True)
            f_win = o.step(f0[row_of_leaf[kin_ids]], case.dt, S)
            k = int(np.searchsorted(kin_ids, c))
            assert np.array_equal(f_win[k], f_full[row_of_leaf[c]]), f"{case.name} {name} leaf {c} S={S}"
            assert np.array_equal(o.moments(f_win)[:, k], m_full[:, row_of_leaf[c]])
            seen.add(name)
    return seen


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_window_mode_equals_full_oracle_on_small_configs(cfg):
    case = inputs.small(cfg)
    seen = _check_window_equals_full(case, inputs.initial_f(case), seed=cfg)
    assert "coarse_side" in seen and "fine_side" in seen
    if cfg == 3:
        assert "next_to_solid" in seen and "domain_wall" in seen
    if cfg == 5:
        assert "next_to_fluid" in seen


def test_window_mode_on_a_random_tree_with_walls_and_noise():
    """Random 2:1 tree, specular / inflow / outflow walls, a SOLID block, a non-Maxwellian noisy state."""
    lv, ijk = random_tree(np.random.default_rng(21), 2, 4, (False, False, False), 0.3)
    c = (ijk + 0.5) / (2.0 ** lv)[:, None]
    kind = np.where(np.abs(c - 0.5).max(axis=1) < 0.13, inputs.CELL_SOLID, inputs.CELL_KINETIC).astype(np.uint8)
    bc = (inputs.BC_INFLOW, inputs.BC_OUTFLOW, inputs.BC_SPECULAR, inputs.BC_SPECULAR, inputs.BC_OUTFLOW, inputs.BC_SPECULAR)
    inflow = np.zeros((6, 5)); inflow[0] = (1.2, 0.7, 0.0, 0.1, 0.9)
    case = periodic_case(lv, ijk, nv=(6, 6, 6), kn=0.2, bc=bc, kind=kind, inflow=inflow)
    rng = np.random.default_rng(5)
    kin = case.kinetic_leaves()
    f0 = inputs.maxwellian_canonical(case, case.prim0[kin]) * (1 + 0.3 * rng.uniform(-1, 1, (kin.size, case.Nv)))
    seen = _check_window_equals_full(case, f0, per_class=3, seed=9)
    assert {"coarse_side", "fine_side", "next_to_solid", "domain_wall"} <= seen


def test_window_mode_is_not_vacuous():
    """A window that is too small (S - 1 rings for S steps) must differ from the full run: the ghost at the window
    edge is felt.  Guards against a check that passes because nothing is compared."""
    case = inputs.small(4)
    f0 = inputs.initial_f(case)
    full = Oracle(case)
    kin = case.kinetic_leaves()
    row_of_leaf = np.full(case.n_leaves, -1, np.int64); row_of_leaf[kin] = np.arange(kin.size)
    c = int(kin[len(kin) // 2])
    S = 2
    f_full = full.step(f0, case.dt, S)
    ids = harness.window_leaves(case, c, S - 1, full.leaf_neighbours)
    kin_ids = ids[case.kind[ids] == inputs.CELL_KINETIC]
    o = Oracle(harness.sub_case(case, ids), window=True)
    f_win = o.step(f0[row_of_leaf[kin_ids]], case.dt, S)
    k = int(np.searchsorted(kin_ids, c))
    assert not np.array_equal(f_win[k], f_full[row_of_leaf[c]])
