"""Host logic of the mesh change (flatten.cpp: build_remap): applying the library's map with numpy
must give the oracle's remap (pinned in tests/test_oracle_remap_pins.py) on random old/new tree pairs, including
multi-level refinement and coarsening, FLUID -> KINETIC leaves and the refusal of SOLID sources."""
import numpy as np
import pytest

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from tests.helpers import periodic_case, random_tree

P = (True, True, True)


def _case(seed, p_split, kind_fn=None, fluid=False, lmax=4):
    lv, ijk = random_tree(np.random.default_rng(seed), 1, lmax, P, p_split)
    kind = np.zeros(lv.shape[0], np.uint8) if kind_fn is None else kind_fn(lv, ijk)
    fm = None
    if fluid:
        c = (ijk + 0.5) / (2.0 ** lv)[:, None]
        fm = np.stack([1 + 0.3 * np.sin(2 * np.pi * c[:, 0]), 0.2 * np.cos(2 * np.pi * c[:, 1]), 0 * c[:, 0] + 0.1,
                       -0.1 * np.sin(2 * np.pi * c[:, 2]), 1 + 0.2 * np.cos(2 * np.pi * c[:, 0])], axis=1)
    return periodic_case(lv, ijk, nv=(6, 4, 4), kind=kind, fluid_moments=fm)


def _apply_plan(old, new, f_old_rows):
    d_o, k1 = B.make_desc(old); d_n, k2 = B.make_desc(new)
    ho, hn = B.ufs_dvm_create_host(d_o), B.ufs_dvm_create_host(d_n)
    try:
        n_o, cell_o, _ = B.ufs_dvm_layout(ho, old.Nv)
        n_n, cell_n, _ = B.ufs_dvm_layout(hn, new.Nv)
        off, src, wgt, gl = B.ufs_dvm_remap_plan(ho, hn, n_n)
    finally:
        B.ufs_dvm_destroy(ho); B.ufs_dvm_destroy(hn)
    row_o = np.full(old.n_leaves, -1, np.int64); row_o[old.kinetic_leaves()] = np.arange(n_o)
    row_n = np.full(new.n_leaves, -1, np.int64); row_n[new.kinetic_leaves()] = np.arange(n_n)
    out = np.zeros((n_n, new.Nv))
    for s in range(n_n):
        acc = np.zeros(new.Nv)
        for k in range(off[s], off[s + 1]):
            if src[k] >= 0:
                acc += wgt[k] * f_old_rows[row_o[cell_o[src[k]]]]
            else:
                leaf = gl[-1 - src[k]]
                acc += wgt[k] * inputs.maxwellian_canonical(old, old.fluid_moments[leaf][None, :])[0]
        out[row_n[cell_n[s]]] = acc
    return out, (off, src, wgt)


@pytest.mark.parametrize("so,sn,po,pn", [(1, 2, 0.3, 0.2), (3, 4, 0.15, 0.35), (5, 5, 0.3, 0.3), (6, 7, 0.0, 0.4), (8, 9, 0.4, 0.0)])
def test_library_map_equals_the_oracle_remap(so, sn, po, pn):
    old, new = _case(so, po), _case(sn, pn)
    rng = np.random.default_rng(so)
    f_old = inputs.maxwellian_canonical(old, old.prim0) * (1 + 0.5 * rng.uniform(-1, 1, (old.n_leaves, old.Nv)))
    got, (off, src, wgt) = _apply_plan(old, new, f_old)
    ref = Oracle(new).remap_from(Oracle(old), f_old)
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()
    # every new slab's weights sum to one; a single source always has weight one
    sums = np.add.reduceat(wgt, off[:-1])
    assert np.allclose(sums, 1.0, rtol=0, atol=1e-15)
    if so == sn and po == pn:
        assert np.all(np.diff(off) == 1) and np.all(wgt == 1.0)


def test_map_with_fluid_sources_and_mask_change():
    half = lambda lv, ijk: np.where((ijk + 0.5)[:, 0] / 2.0 ** lv < 0.5, inputs.CELL_FLUID, inputs.CELL_KINETIC).astype(np.uint8)
    other = lambda lv, ijk: np.where((ijk + 0.5)[:, 1] / 2.0 ** lv < 0.3, inputs.CELL_FLUID, inputs.CELL_KINETIC).astype(np.uint8)
    old, new = _case(11, 0.3, kind_fn=half, fluid=True), _case(12, 0.25, kind_fn=other, fluid=True)
    rng = np.random.default_rng(3)
    kin = old.kinetic_leaves()
    f_old = inputs.maxwellian_canonical(old, old.prim0[kin]) * (1 + 0.5 * rng.uniform(-1, 1, (kin.size, old.Nv)))
    got, (off, src, wgt) = _apply_plan(old, new, f_old)
    assert (src < 0).any()
    ref = Oracle(new).remap_from(Oracle(old), f_old)
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()


def test_solid_source_is_refused():
    blk = lambda lv, ijk: np.where(np.abs((ijk + 0.5) / (2.0 ** lv)[:, None] - 0.5).max(axis=1) < 0.2, inputs.CELL_SOLID, inputs.CELL_KINETIC).astype(np.uint8)
    old, new = _case(21, 0.3, kind_fn=blk), _case(21, 0.3)
    d_o, k1 = B.make_desc(old); d_n, k2 = B.make_desc(new)
    ho, hn = B.ufs_dvm_create_host(d_o), B.ufs_dvm_create_host(d_n)
    with pytest.raises(B.UfsDvmError) as e:
        B.ufs_dvm_remap_plan(ho, hn, new.n_leaves)
    assert e.value.code == B.EINVAL and "SOLID" in str(e.value)
    B.ufs_dvm_destroy(ho); B.ufs_dvm_destroy(hn)


def test_config3_to_l8_with_the_old_body_is_a_pure_refinement_map():
    """The stated-size mesh change of tests/test_gpu_remesh.py, host side: with the old staircase body kept
    (inputs.with_body_of) every new kinetic leaf has exactly one source of weight one; without it the map is refused
    because the finer sampling of the sphere uncovers leaves inside old SOLID leaves."""
    old, fine = inputs.config3(lmax=7), inputs.config3(lmax=8)
    new = inputs.with_body_of(old, fine)
    assert (new.kind == inputs.CELL_SOLID).sum() > (fine.kind == inputs.CELL_SOLID).sum()
    ho = B.ufs_dvm_create_host(B.make_desc(old)[0])
    try:
        hn = B.ufs_dvm_create_host(B.make_desc(new)[0])
        n_n, _, _ = B.ufs_dvm_layout(hn, new.Nv)
        off, src, wgt, gl = B.ufs_dvm_remap_plan(ho, hn, n_n)
        B.ufs_dvm_destroy(hn)
        assert n_n == new.kinetic_leaves().size and np.all(np.diff(off) == 1)
        assert np.all(wgt == 1.0) and np.all(src >= 0) and gl.size == 0
        hf = B.ufs_dvm_create_host(B.make_desc(fine)[0])
        with pytest.raises(B.UfsDvmError) as e:
            B.ufs_dvm_remap_plan(ho, hf, fine.kinetic_leaves().size)
        B.ufs_dvm_destroy(hf)
        assert e.value.code == B.EINVAL and "SOLID" in str(e.value)
    finally:
        B.ufs_dvm_destroy(ho)
