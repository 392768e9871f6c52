"""Host logic of the tile records (flatten.cpp: build_tiles): a numpy
transport step that gathers every cell's four streams THROUGH the tile records (piece lists + per-cell index tables)
must reproduce the oracle's transport (Eq. 2) on trees with 2:1 faces, walls of every kind, SOLID and
FLUID leaves.  Also: tiles partition the slabs in order, complete sibling octets are kept whole, and no piece list is
longer than pmax."""
import numpy as np
import pytest

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from tests.helpers import periodic_case, random_tree

PIECE_TABLE = 0x80000000
PIECE_FLUID = 0x40000000      # a fluid ghost: its Maxwellian is formed on chip from factor rows, nothing is copied
PIECE_INDEX = 0x3fffffff


def _host(case, storage=None):
    d, keep = B.make_desc(case, storage=storage)
    return B.ufs_dvm_create_host(d), keep


def _transport_through_tiles(case, h, f0_rows, dt):
    """f* of every kinetic leaf (Case row order, canonical velocity order) computed from the tile records only."""
    n_kin, cell_of_slab, vel_of_slot = B.ufs_dvm_layout(h, case.Nv)
    T = B.ufs_dvm_tiles(h)
    nv = case.nv[0]
    nh = nv // 2
    CH = nh ** 3
    kin = case.kinetic_leaves()
    row_of_leaf = np.full(case.n_leaves, -1, np.int64); row_of_leaf[kin] = np.arange(kin.size)
    row_of_slab = row_of_leaf[cell_of_slab]
    f = f0_rows[row_of_slab][:, vel_of_slot].reshape(n_kin, 8, CH)         # slab, octant chunk, in-chunk offset
    # |xi| by rank (x fastest inside a chunk), ghost tables in slot order
    xi = np.abs(case.xi_nodes(0))[nh:]
    ax, ay, az = xi[None, None, :], xi[None, :, None], xi[:, None, None]
    tables = {}
    for s in range(6):
        if case.bc[s] == inputs.BC_INFLOW:
            tables[len(tables)] = inputs.maxwellian_canonical(case, case.inflow[s][None, :])[0][vel_of_slot].reshape(8, CH)
    out = np.zeros_like(f)
    seen = np.zeros(n_kin, bool)
    for t in range(T["n_tiles"]):
        s0, nc = int(T["s0"][t]), int(T["nc"][t])
        for o in range(8):
            def chunk(code):
                c = code & PIECE_INDEX
                if code & PIECE_TABLE:
                    return tables[c // 8][c % 8]
                if code & PIECE_FLUID:
                    assert c % 8 == o
                    leaf = int(T["fluid_leaf"][c // 8])
                    assert case.kind[leaf] == inputs.CELL_FLUID
                    return inputs.maxwellian_canonical(case, case.fluid_moments[leaf][None, :])[0][vel_of_slot].reshape(8, CH)[o]
                return f[c // 8, c % 8]
            pcs = T["pieces"][t, o]
            for c in range(nc):
                ix = T["cellidx"][t, o, c]
                assert int(pcs[ix[0]]) == (s0 + c) * 8 + o                  # own chunk
                own = chunk(int(pcs[ix[0]])).reshape(nh, nh, nh)
                level = int(T["level"][t][c])
                assert level == case.level[cell_of_slab[s0 + c]]
                dth = dt * (1 << level) / case.domain_len
                acc = own * (1.0 - dth * (ax + ay + az))
                for a, w in enumerate((ax, ay, az)):
                    four = (ix[1] >> a) & 1
                    src = np.zeros(CH)
                    for k in range(4 if four else 1):
                        b = int(ix[4 + 4 * a + k])
                        assert b != 0xFF
                        is_fluid = bool(int(pcs[b]) & PIECE_FLUID)
                        # the per-cell fluid mask (bytes 2..3, bit 4a + k) and flag bit 3 say the same
                        assert bool(((int(ix[2]) | (int(ix[3]) << 8)) >> (4 * a + k)) & 1) == is_fluid
                        assert not is_fluid or (ix[1] & 0x08)
                        src = src + chunk(int(pcs[b]))
                    if not four:
                        assert all(int(x) == 0xFF for x in ix[5 + 4 * a: 8 + 4 * a])
                    acc = acc + dth * w * (0.25 if four else 1.0) * src.reshape(nh, nh, nh)
                out[s0 + c, o] = acc.reshape(CH)
        seen[s0:s0 + nc] = True
    assert seen.all()
    inv = np.empty(case.Nv, np.int64); inv[vel_of_slot] = np.arange(case.Nv)
    res = np.empty_like(f0_rows)
    res[row_of_slab] = out.reshape(n_kin, case.Nv)[:, inv]
    return res, T


def _check_structure(case, h, T, storage):
    n_kin, cell_of_slab, _ = B.ufs_dvm_layout(h, case.Nv)
    assert T["n_tiles"] > 0 and T["s0"][0] == 0
    assert np.array_equal(T["s0"][1:], (T["s0"] + T["nc"])[:-1]) and T["s0"][-1] + T["nc"][-1] == n_kin
    assert T["nc"].min() >= 1 and T["nc"].max() <= 8
    assert T["np"].max() <= T["pmax"]
    # complete sibling octets (children 0..7 of one parent in N-order, all kinetic) are never split or merged
    lv, ijk = case.level[cell_of_slab].astype(np.int64), case.ijk[cell_of_slab].astype(np.int64)
    starts = set(T["s0"].tolist())
    n_oct = 0
    for s in range(n_kin - 7):
        if lv[s] == 0 or (ijk[s] & 1).any():
            continue
        ok = all(lv[s + i] == lv[s] and np.array_equal(ijk[s + i], ijk[s] + [(i & 1), (i >> 1) & 1, (i >> 2) & 1]) for i in range(1, 8))
        if ok:
            n_oct += 1
            t = int(np.searchsorted(T["s0"], s))
            fits = T["nc"][t] == 8 and T["s0"][t] == s
            # (an octet whose piece lists exceed pmax -- finer neighbours all around -- may be cut)
            assert fits or T["pmax"] < 8 + 12 * 4
            assert s in starts
    return n_oct


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_transport_through_tile_records_matches_oracle_small_configs(cfg):
    case = inputs.small(cfg)
    h, _ = _host(case)
    assert B.ufs_dvm_kernel_name(h) == "k_tiles"
    f0 = inputs.initial_f(case)
    rng = np.random.default_rng(cfg)
    f0 = f0 * (1 + 0.2 * rng.uniform(-1, 1, f0.shape))       # no symmetry can hide a wrong source
    got, T = _transport_through_tiles(case, h, f0, case.dt)
    ref = Oracle(case).transport(f0, case.dt)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    n_oct = _check_structure(case, h, T, case.storage)
    assert n_oct > 0
    B.ufs_dvm_destroy(h)


def test_tiles_on_a_random_periodic_tree_fp32_pmax():
    """fp32 storage: the ring holds more pieces (pmax 40), so octets with finer neighbours stay whole."""
    lv, ijk = random_tree(np.random.default_rng(8), 2, 4, (True, True, True), 0.25)
    case = periodic_case(lv, ijk, nv=(24, 24, 24), vlim=5.0, kn=0.2)
    h, _ = _host(case, storage=inputs.STORE_F32)
    assert B.ufs_dvm_kernel_name(h) == "k_tiles"
    rng = np.random.default_rng(2)
    f0 = inputs.maxwellian_canonical(case, case.prim0) * (1 + 0.3 * rng.uniform(-1, 1, (case.n_leaves, case.Nv)))
    got, T = _transport_through_tiles(case, h, f0, case.dt)
    ref = Oracle(case).transport(f0, case.dt)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    assert T["pmax"] == 40
    assert _check_structure(case, h, T, inputs.STORE_F32) > 0
    B.ufs_dvm_destroy(h)


def test_shared_pieces_are_counted_once():
    """A uniform periodic grid: every tile is an octet and lists exactly 20 pieces per octant (8 own + 12 outside)."""
    lv, ijk = inputs.build_tree(3, 3, {}, (True,) * 3)
    case = periodic_case(lv, ijk, nv=(24, 24, 24), vlim=5.0)
    h, _ = _host(case)
    T = B.ufs_dvm_tiles(h)
    assert T["n_tiles"] == 64 and np.all(T["nc"] == 8) and np.all(T["np"] == 20)
    B.ufs_dvm_destroy(h)


def test_other_grids_do_not_get_tiles():
    case = inputs.config1()              # 12^3: six positive nodes per axis -> k_rows
    h, _ = _host(case)
    assert B.ufs_dvm_kernel_name(h) == "k_rows" and B.ufs_dvm_tiles(h)["n_tiles"] == 0
    B.ufs_dvm_destroy(h)
