"""The lattice-Boltzmann variant through its C ABI (include/ufs_lbm.h).

CPU: the library exports every declared symbol, validates its arguments, and its layout (N-order rows, lattice columns
and weights) is what the oracle and the problem recipes assume.  GPU: parity with oracle/lbm_oracle.py element by element
("CPU and GPU results coincide within a machine precision") on D3Q19 and D3Q27, fp64 and fp32 storage,
periodic 2:1 trees, walls of every kind with SOLID leaves and an equilibrium inflow, with and without collisions."""
import math
import os
import re

import numpy as np
import pytest

from oracle import lbm_oracle as LO
from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from paper_1503_00707_b200 import lbm as K
from tests.helpers import rel_linf

TOL = {inputs.STORE_F64: 1e-12, inputs.STORE_F32: 2e-5}


def test_library_exports_every_declared_lbm_symbol():
    L = K.lib()
    hdr = open(os.path.join(os.path.dirname(B.__file__), "..", "include", "ufs_lbm.h")).read()
    declared = set(re.findall(r"\b(ufs_lbm_[a-z_]+)\s*\(", hdr))
    assert declared == set(K.EXPORTS)
    for name in declared:
        assert getattr(L, name) is not None


@pytest.mark.parametrize("q", [19, 27])
def test_layout_lattice_and_weights(q):
    case = inputs.lbm_case(inputs.small(3), q)
    d, keep = K.make_desc(case)
    h = K.ufs_lbm_create_host(d)
    n, cell, qq, c, w = K.ufs_lbm_layout(h)
    K.ufs_lbm_destroy(h)
    kin = case.kinetic_leaves()
    assert qq == q and n == kin.size and sorted(cell.tolist()) == kin.tolist()
    order = inputs.morton_order(case.level, case.ijk)
    assert np.array_equal(cell, order[case.kind[order] == inputs.CELL_KINETIC])      # rows in N-order
    assert np.array_equal(c.astype(np.int64), inputs.lattice_velocities(q))
    co, wo, _ = LO.lattice(q)
    assert np.array_equal(c.astype(float), co) and np.abs(w - wo).max() < 1e-16 and abs(w.sum() - 1) < 1e-15


def test_bad_arguments_are_refused():
    case = inputs.lbm_case(inputs.small(3), 19)
    d, keep = K.make_desc(case)
    d.lattice = 15
    with pytest.raises(B.UfsDvmError) as e:
        K.ufs_lbm_create_host(d)
    assert e.value.code == B.EINVAL
    d.lattice = 19; d.tau = 0.0
    with pytest.raises(B.UfsDvmError):
        K.ufs_lbm_create_host(d)
    masked = inputs.small(5)                         # has FLUID leaves
    c2 = inputs.lbm_case(masked, 19); c2.kind = masked.kind.copy()
    with pytest.raises(B.UfsDvmError) as e:
        K.ufs_lbm_create_host(K.make_desc(c2)[0])
    assert e.value.code == B.EINVAL and "FLUID" in str(e.value)


# ------------------------------------------------------------------------------------------------- GPU parity
def _check(case, nsteps, tau=None, storage=None):
    storage = case.storage if storage is None else storage
    tau = inputs.lbm_tau(case) if tau is None else tau
    f0 = LO.initial_f(case)
    if storage == inputs.STORE_F32:
        f0 = f0.astype(np.float32).astype(np.float64)
    st = K.LbmStepper(case, tau=tau, storage=storage)
    st.load_canonical(f0)
    st.step(case.dt, nsteps)
    st.sync()
    f_gpu, m_gpu = st.read_canonical(), st.moments()
    assert K.ufs_lbm_launch_count(st.h) == nsteps + 1
    st.close()
    o = LO.LbmOracle(case, tau)
    f_ref = o.step(f0, case.dt, nsteps)
    m_ref = o.moments(f_ref)
    tol = TOL[storage]
    assert np.all(np.isfinite(f_gpu))
    assert rel_linf(f_gpu, f_ref) <= tol
    assert rel_linf(m_gpu[0], m_ref[0]) <= tol
    pmax = np.sqrt((m_ref[1:] ** 2).sum(axis=0)).max()
    assert np.abs(m_gpu[1:] - m_ref[1:]).max() <= tol * max(pmax, 1e-3 * m_ref[0].max())
    assert np.abs(f_gpu - f0).max() > 1e-6 * np.abs(f0).max()      # the step did something


@pytest.mark.gpu
@pytest.mark.parametrize("q", [19, 27])
@pytest.mark.parametrize("tree", ["config1", "small3", "small4"])
def test_lbm_matches_oracle_fp64(q, tree):
    base = {"config1": inputs.config1, "small3": lambda: inputs.small(3), "small4": lambda: inputs.small(4)}[tree]()
    case = inputs.lbm_case(base, q, nsteps=6)
    _check(case, 6, storage=inputs.STORE_F64)


@pytest.mark.gpu
@pytest.mark.parametrize("q", [19, 27])
def test_lbm_matches_oracle_fp32_storage(q):
    _check(inputs.lbm_case(inputs.small(3), q), 5, storage=inputs.STORE_F32)


@pytest.mark.gpu
def test_lbm_transport_only():
    _check(inputs.lbm_case(inputs.small(3), 27), 4, tau=math.inf)


@pytest.mark.gpu
def test_lbm_conserves_mass_on_the_periodic_tree():
    case = inputs.lbm_case(inputs.config1(), 19, noise_rel=2e-2)
    st = K.LbmStepper(case)
    st.load_canonical(LO.initial_f(case))
    vol = 8.0 ** (-case.level[case.kinetic_leaves()].astype(np.float64))
    m0 = st.moments()
    st.step(case.dt, 20)
    m1 = st.moments()
    st.close()
    assert np.abs(((m1 - m0) * vol).sum(axis=1)).max() <= 1e-13 * (m0[0] * vol).sum()


@pytest.mark.gpu
def test_lbm_on_the_million_leaf_octree_windows_and_conservation():
    """The bench workload of the LBM variant (D3Q19 on the 1 009 261-leaf periodic config-4 octree, fp64): parity at
    sampled cells against the oracle on the sub-mesh within S = 3 face rings of each (values outside the domain of
    dependence cannot reach the sample after S steps; window mode pinned in tests/test_oracle_window_pin.py), then
    conservation of total mass and momentum over 20 steps."""
    from oracle.dvm_oracle import Oracle
    from paper_1503_00707_b200 import harness
    S = 3
    case = inputs.lbm_case(inputs.config4(), 19, noise_rel=0.0)
    st = K.LbmStepper(case)
    # f(t=0): the equilibrium of the case's (rho, u) fields, formed by the oracle side and handed to the device
    f0 = LO.initial_f(case)
    st.load_canonical(f0)
    mesh = Oracle(case, kn=math.inf)                      # neighbour search of the whole mesh (for the windows)
    rng = np.random.default_rng(inputs.SEED_BASE + 919)
    kin = case.kinetic_leaves()
    picks = []
    for l in np.unique(case.level[kin]).tolist():
        ids = kin[case.level[kin] == l]
        picks.append(rng.choice(ids, 16, replace=False))
    picks.append(np.array([st.cell_of_row[0], st.cell_of_row[-1]]))
    centres = np.unique(np.concatenate(picks))
    row_of_leaf = np.full(case.n_leaves, -1, np.int64); row_of_leaf[kin] = np.arange(kin.size)
    vol = 8.0 ** (-case.level[kin].astype(np.float64))
    m0 = st.moments()
    st.step(case.dt, S)
    st.sync()
    f_gpu = st.read_canonical()
    worst = 0.0
    for c in centres.tolist():
        ids = harness.window_leaves(case, c, S, mesh.leaf_neighbours)
        sub = inputs.sub_case(case, ids); sub.meta = case.meta
        o = LO.LbmOracle(sub, inputs.lbm_tau(case), window=True)
        f_ref = o.step(f0[row_of_leaf[ids]], case.dt, S)
        k = int(np.searchsorted(ids, c))
        err = np.abs(f_gpu[row_of_leaf[c]] - f_ref[k]).max() / np.abs(f_ref[k]).max()
        worst = max(worst, err)
        assert err <= 1e-12, f"leaf {c} (level {case.level[c]}): {err:.3e}"
    del mesh
    st.step(case.dt, 20 - S)
    m1 = st.moments()
    st.close()
    tot0, tot1 = (m0 * vol).sum(axis=1), (m1 * vol).sum(axis=1)
    assert np.all(np.isfinite(m1))
    assert np.abs(tot1 - tot0).max() <= 1e-12 * tot0[0]
