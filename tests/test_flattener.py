"""Host logic of the C-ABI library (no GPU): symbols, mesh validation, face lists, layout."""
import ctypes as C

import numpy as np
import pytest

from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from tests.helpers import brute_force_faces, periodic_case, random_tree

P = (True, True, True)


def _host(case, **kw):
    desc, keep = B.make_desc(case, **kw)
    return B.ufs_dvm_create_host(desc), keep


def test_library_exports_every_declared_symbol():
    import os, re
    L = B.lib()
    hdr = open(os.path.join(os.path.dirname(B.__file__), "..", "include", "ufs_dvm.h")).read()
    declared = set(re.findall(r"\b(ufs_dvm_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert getattr(L, name) is not None


def test_config1_faces_layout_and_counts():
    c = inputs.config1()
    h, _ = _host(c)
    ow, ng, ar, ax, ra = B.ufs_dvm_faces(h)
    assert (ra == 0).sum() == 1644 and (ra != 0).sum() == 96
    got = sorted(zip(ow.tolist(), ng.tolist(), ax.tolist(), ar.tolist()))
    assert got == brute_force_faces(c.level, c.ijk, P)
    n, cell, vel = B.ufs_dvm_layout(h, c.Nv)
    assert n == 568 and sorted(cell.tolist()) == list(range(568))
    assert sorted(vel.tolist()) == list(range(c.Nv))
    # octant grouping: each eighth of the slab holds one sign combination
    nv = c.nv[0]
    kx, ky, kz = vel % nv, (vel // nv) % nv, vel // (nv * nv)
    octant = (kx >= nv // 2) + 2 * (ky >= nv // 2) + 4 * (kz >= nv // 2)
    assert np.array_equal(octant, np.repeat(np.arange(8), c.Nv // 8))
    # Morton order: depth-first, child index x + 2y + 4z
    lmax = int(c.level.max())
    sh = lmax - c.level[cell].astype(np.int64)
    xyz = c.ijk[cell].astype(np.int64) << sh[:, None]
    key = np.zeros(n, np.int64)
    for b in range(lmax):
        for a in range(3):
            key |= ((xyz[:, a] >> b) & 1) << (3 * b + a)
    assert np.all(np.diff(key) > 0)
    assert B.ufs_dvm_kernel_info(h)["fast"] and B.ufs_dvm_kernel_info(h)["vec"] == 2
    B.ufs_dvm_destroy(h)


@pytest.mark.parametrize("seed,periodic", [(0, P), (1, (False, False, False)), (2, (True, False, True))])
def test_faces_random_trees_against_brute_force(seed, periodic):
    rng = np.random.default_rng(seed)
    lv, ijk = random_tree(rng, 1, 4, periodic, 0.12)
    bc = tuple(inputs.BC_PERIODIC if periodic[s // 2] else inputs.BC_OUTFLOW for s in range(6))
    kind = np.zeros(lv.shape[0], np.uint8)
    kind[rng.uniform(size=lv.shape[0]) < 0.1] = inputs.CELL_SOLID
    c = periodic_case(lv, ijk, bc=bc, kind=kind)
    h, _ = _host(c)
    ow, ng, ar, ax, ra = B.ufs_dvm_faces(h)
    got = sorted(zip(ow.tolist(), ng.tolist(), ax.tolist(), ar.tolist()))
    assert got == brute_force_faces(lv, ijk, periodic, live=kind != inputs.CELL_SOLID)
    assert np.all(ra == lv[ng].astype(int) - lv[ow].astype(int))
    B.ufs_dvm_destroy(h)


def test_boundary_face_counts_match_survey_config3():
    c = inputs.config3()
    h, _ = _host(c)
    ow, ng, ar, ax, ra = B.ufs_dvm_faces(h)
    assert (ra == 0).sum() == 70536 and (ra != 0).sum() == 9728
    cell, axis, side, area, kind, state = B.ufs_dvm_boundary_faces(h)
    cnt = {k: int((kind == k).sum()) for k in (1, 2, 3, 4, 5)}
    assert cnt == {1: 1024, 2: 256, 3: 256, 4: 3104, 5: 0}
    n, _, _ = B.ufs_dvm_layout(h, c.Nv)
    assert n == 26312
    B.ufs_dvm_destroy(h)


def test_mask_and_fluid_interface_faces():
    c = inputs.small(5)
    h, _ = _host(c)
    n, cell, _ = B.ufs_dvm_layout(h, c.Nv)
    assert n == int((c.kind == inputs.CELL_KINETIC).sum())
    assert np.all(c.kind[cell] == inputs.CELL_KINETIC)
    bcell, axis, side, area, kind, state = B.ufs_dvm_boundary_faces(h)
    fl = kind == B_FLUID
    assert fl.sum() > 0 and np.all(c.kind[state[fl]] == inputs.CELL_FLUID) and np.all(c.kind[bcell[fl]] == inputs.CELL_KINETIC)
    B.ufs_dvm_destroy(h)


B_FLUID = 5


def test_validation_errors():
    lv, ijk = inputs.build_tree(2, 2, {}, P)
    with pytest.raises(B.UfsDvmError) as e:
        _host(periodic_case(lv[:-1], ijk[:-1]))
    assert e.value.code == B.EMESH
    with pytest.raises(B.UfsDvmError) as e:                       # duplicate leaf = overlap
        _host(periodic_case(np.concatenate([lv, lv[:1]]), np.concatenate([ijk, ijk[:1]])))
    assert e.value.code == B.EMESH
    # face 2:1 violation
    oct_ = [(i, j, k) for k in range(2) for j in range(2) for i in range(2)]
    lvb = np.array([1] * 7 + [2] * 7 + [3] * 8, np.uint8)
    ijkb = np.array(oct_[1:] + oct_[:-1] + [(2 + i, 2 + j, 2 + k) for (i, j, k) in oct_], np.uint32)
    with pytest.raises(B.UfsDvmError) as e:
        _host(periodic_case(lvb, ijkb, bc=(inputs.BC_OUTFLOW,) * 6))
    assert e.value.code == B.EMESH
    # diagonal-only 2:1 violation (second constraint): level-1 cube, octant (0,0,0) split to
    # level 2, its child (1,1,0) split to level 3: those leaves touch the level-1 octant (1,1,0) only
    # along an edge
    lvd = np.array([1] * 7 + [2] * 7 + [3] * 8, np.uint8)
    l2 = [c for c in oct_ if c != (1, 1, 0)]
    ijkd = np.array(oct_[1:] + l2 + [(2 + i, 2 + j, 0 + k) for (i, j, k) in oct_], np.uint32)
    # make it face-balanced: the level-3 block at (2..3,2..3,0..1) has face neighbours at level 2 inside
    # octant (0,0,0) on -x,-y,+z, the domain boundary on -z, and level-1 leaves across +x and +y faces --
    # so this tree also violates the face rule; use the oracle-independent property instead: EMESH either way
    with pytest.raises(B.UfsDvmError) as e:
        _host(periodic_case(lvd, ijkd, bc=(inputs.BC_OUTFLOW,) * 6))
    assert e.value.code == B.EMESH
    # specular needs a symmetric grid
    c = periodic_case(lv, ijk, bc=(inputs.BC_SPECULAR,) * 2 + (inputs.BC_PERIODIC,) * 4)
    c.vmin = (-3.0, -4.0, -4.0)
    with pytest.raises(B.UfsDvmError) as e:
        _host(c)
    assert e.value.code == B.EINVAL
    # periodic on one side only
    with pytest.raises(B.UfsDvmError):
        _host(periodic_case(lv, ijk, bc=(inputs.BC_PERIODIC, inputs.BC_OUTFLOW) + (inputs.BC_PERIODIC,) * 4))
    # device calls on a host-only handle
    h, _ = _host(periodic_case(lv, ijk))
    assert B.lib().ufs_dvm_step(h, 0.1, 1) == B.EINVAL
    assert "host-only" in B.ufs_dvm_last_error(h)
    B.ufs_dvm_destroy(h)


def test_diagonal_balance_is_checked():
    """A tree that is face-balanced but not edge-balanced must be rejected (PAPER.md:45 rule 2)."""
    # level-2 base (4^3); refine cell (1,1,1) to level 3 and its child (3,3,3)->level 4.  Level-4 leaves at
    # (6..7)^3 touch the level-2 cell (2,2,2) at a corner only; face neighbours of the level-4 block are the
    # level-3 siblings (inside) and the level-2 cells (2,1,1),(1,2,1),(1,1,2) across faces -> that IS a face
    # violation too.  Build instead a corner-only violation by also refining those three face neighbours
    # and the three edge neighbours (2,2,1),(2,1,2),(1,2,2) once, leaving (2,2,2) at level 2.
    split2 = np.zeros((4, 4, 4), bool)
    for c in [(1, 1, 1), (2, 1, 1), (1, 2, 1), (1, 1, 2), (2, 2, 1), (2, 1, 2), (1, 2, 2)]:
        split2[c] = True
    split3 = np.zeros((8, 8, 8), bool)
    split3[3, 3, 3] = True
    # assemble the unbalanced leaf list by hand (inputs.build_tree would balance it)
    leaves = []
    for i in range(4):
        for j in range(4):
            for k in range(4):
                if not split2[i, j, k]:
                    leaves.append((2, i, j, k))
                else:
                    for a in range(2):
                        for b in range(2):
                            for cc in range(2):
                                I, J, K = 2 * i + a, 2 * j + b, 2 * k + cc
                                if split3[I, J, K]:
                                    leaves += [(4, 2 * I + x, 2 * J + y, 2 * K + z) for x in range(2) for y in range(2) for z in range(2)]
                                else:
                                    leaves.append((3, I, J, K))
    arr = np.array(leaves)
    c = periodic_case(arr[:, 0].astype(np.uint8), arr[:, 1:].astype(np.uint32), bc=(inputs.BC_OUTFLOW,) * 6)
    # the oracle only needs face neighbours and accepts this tree ...
    from oracle.dvm_oracle import Oracle
    Oracle(c)
    # ... the library enforces both rules of PAPER.md:45
    with pytest.raises(B.UfsDvmError) as e:
        _host(c)
    assert e.value.code == B.EMESH


def test_generic_layout_for_odd_and_asymmetric_grids():
    lv, ijk = inputs.build_tree(1, 1, {}, P)
    c = periodic_case(lv, ijk, nv=(5, 4, 3))
    c.vmin, c.vmax = (-4.0, -3.0, -2.0), (4.0, 5.0, 2.0)
    h, _ = _host(c)
    info = B.ufs_dvm_kernel_info(h)
    assert not info["fast"]
    n, cell, vel = B.ufs_dvm_layout(h, c.Nv)
    assert sorted(vel.tolist()) == list(range(c.Nv))
    B.ufs_dvm_destroy(h)
