"""Pins of the lattice-Boltzmann oracle (oracle/lbm_oracle.py) against what the lattice mathematics
fixes, none of them the oracle's own formula retyped:

* the weights are THE solution of the isotropy conditions of a D3Q19 / D3Q27 lattice with c_s^2 = 1/3 (solved here as a
  linear system per shell, independently);
* the moments of the second-order equilibrium: sum f_eq = rho, sum c f_eq = rho u, sum c c f_eq =
  rho (c_s^2 I + u u) -- the property the expansion is built to have;
* relaxation conserves rho and rho u, an equilibrium is its fixed point, homogeneous relaxation is geometric;
* a uniform equilibrium at rest and in motion is steady on a periodic 2:1 tree (transport + collision together);
* the whole step conserves mass and momentum on a periodic tree; a specular box conserves mass;
* D3Q19 is D3Q27's transport restricted to 19 velocities (the eight corners never mix in);
* 1-D streaming along x on a uniform periodic grid: every population moves with its own c_x by the closed form of the
  first-order upwind scheme (the same closed form that pins the DVM transport, P3)."""
import itertools

import numpy as np
import pytest

from oracle import lbm_oracle as LO
from paper_1503_00707_b200 import inputs
from tests.helpers import periodic_case, random_tree

P = (True, True, True)


def _tree_case(seed=3, p_split=0.3, lmax=3):
    lv, ijk = random_tree(np.random.default_rng(seed), 1, lmax, P, p_split)
    return periodic_case(lv, ijk, nv=(6, 6, 6))


@pytest.mark.parametrize("q", [19, 27])
def test_weights_solve_the_isotropy_conditions(q):
    c, w, active = LO.lattice(q)
    assert c.shape == (q, 3) and len(set(map(tuple, c.tolist()))) == q
    assert np.array_equal(c, inputs.lattice_velocities(q).astype(float))          # same index meaning on both sides
    # independent derivation: one weight per shell |c|^2; conditions sum w = 1, sum w cx^2 = 1/3, sum w cx^4 = 3 sum w cx^2 cy^2
    # (4th-order isotropy), and for D3Q27 additionally sum w cx^2 cy^2 cz^2 = 1/27 (6th-order moment of the product form)
    shells = sorted(set(int(round((ci ** 2).sum())) for ci in c))
    rows, rhs = [], []
    def row(fn):
        return [sum(fn(ci) for ci in c if int(round((ci ** 2).sum())) == s) for s in shells]
    rows.append(row(lambda ci: 1.0)); rhs.append(1.0)
    rows.append(row(lambda ci: ci[0] ** 2)); rhs.append(1.0 / 3.0)
    rows.append(row(lambda ci: ci[0] ** 4 - 3.0 * ci[0] ** 2 * ci[1] ** 2)); rhs.append(0.0)
    if q == 27:
        rows.append(row(lambda ci: ci[0] ** 2 * ci[1] ** 2 * ci[2] ** 2)); rhs.append(1.0 / 27.0)
    sol = np.linalg.solve(np.array(rows), np.array(rhs))
    for s, ws in zip(shells, sol):
        got = {round(float(wi), 15) for ci, wi in zip(c, w) if int(round((ci ** 2).sum())) == s}
        assert len(got) == 1 and abs(got.pop() - ws) < 1e-15
    # full second- and fourth-order isotropy
    d = np.eye(3)
    for a, b in itertools.product(range(3), repeat=2):
        assert abs((w * c[:, a] * c[:, b]).sum() - d[a, b] / 3.0) < 1e-15
    for a, b, g, e in itertools.product(range(3), repeat=4):
        want = (d[a, b] * d[g, e] + d[a, g] * d[b, e] + d[a, e] * d[b, g]) / 9.0
        assert abs((w * c[:, a] * c[:, b] * c[:, g] * c[:, e]).sum() - want) < 1e-15
    assert all(abs((w * c[:, a]).sum()) < 1e-16 for a in range(3))


@pytest.mark.parametrize("q", [19, 27])
def test_equilibrium_moments(q):
    rng = np.random.default_rng(q)
    rho = rng.uniform(0.5, 2.0, 50)
    u = rng.uniform(-0.15, 0.15, (50, 3))
    feq = LO.equilibrium(q, rho, u)
    c, w, _ = LO.lattice(q)
    assert np.abs(feq.sum(axis=1) - rho).max() < 1e-15
    assert np.abs(feq @ c - rho[:, None] * u).max() < 1e-15
    for a, b in itertools.product(range(3), repeat=2):
        m2 = (feq * c[:, a] * c[:, b]).sum(axis=1)
        assert np.abs(m2 - rho * ((a == b) / 3.0 + u[:, a] * u[:, b])).max() < 1e-15
    # at rest: f_eq = w rho
    assert np.abs(LO.equilibrium(q, rho, 0 * u) - rho[:, None] * w[None, :]).max() < 1e-16
    # the moments routine is the plain sums
    r2, m2 = LO.moments(q, feq)
    assert np.array_equal(r2, sum(feq[:, i] for i in range(q)))


@pytest.mark.parametrize("q", [19, 27])
def test_relaxation_invariants_and_geometric_decay(q):
    case = inputs.lbm_case(_tree_case(), q, omega=0.6)
    tau = inputs.lbm_tau(case)
    o = LO.LbmOracle(case, tau)
    rng = np.random.default_rng(1)
    f = LO.initial_f(case) * (1 + 0.3 * rng.uniform(-1, 1, (o.n, q)))
    g = o.collide(f, case.dt)
    r0, m0 = LO.moments(q, f); r1, m1 = LO.moments(q, g)
    assert np.abs(r1 - r0).max() < 1e-15 and np.abs(m1 - m0).max() < 1e-15
    feq = LO.equilibrium(q, r0, m0 / r0[:, None])
    assert np.abs(o.collide(feq, case.dt) - feq).max() < 1e-15                    # fixed point (to round-off)
    # homogeneous relaxation: moments conserved => f^n = f_eq + (1 - omega)^n (f - f_eq)
    h = f.copy()
    for _ in range(5):
        h = o.collide(h, case.dt)
    assert np.abs(h - (feq + (1 - 0.6) ** 5 * (f - feq))).max() < 1e-15


@pytest.mark.parametrize("q", [19, 27])
@pytest.mark.parametrize("u", [(0.0, 0.0, 0.0), (0.05, -0.03, 0.02)])
def test_uniform_equilibrium_is_steady_on_a_2to1_periodic_tree(q, u):
    case = inputs.lbm_case(_tree_case(), q, noise_rel=0.0)
    case.prim0[:, 0] = 1.3; case.prim0[:, 1:4] = u
    o = LO.LbmOracle(case, inputs.lbm_tau(case))
    f0 = LO.initial_f(case)
    f1 = o.step(f0, case.dt, 4)
    assert np.abs(f1 - f0).max() <= 2e-15 * np.abs(f0).max()


@pytest.mark.parametrize("q", [19, 27])
def test_step_conserves_mass_and_momentum_on_a_periodic_tree(q):
    case = inputs.lbm_case(_tree_case(seed=5), q, noise_rel=5e-2)
    o = LO.LbmOracle(case, inputs.lbm_tau(case))
    f0 = LO.initial_f(case)
    f1 = o.step(f0, case.dt, 3)
    vol = 8.0 ** (-case.level[case.kinetic_leaves()].astype(np.float64))
    m0, m1 = o.moments(f0), o.moments(f1)
    assert np.abs(((m1 - m0) * vol).sum(axis=1)).max() <= 1e-14 * (m0[0] * vol).sum()


def test_specular_box_with_a_solid_block_conserves_mass():
    lv, ijk = random_tree(np.random.default_rng(2), 2, 3, (False,) * 3, 0.3)
    c = (ijk + 0.5) / (2.0 ** lv)[:, None]
    kind = np.where(np.abs(c - 0.5).max(axis=1) < 0.2, inputs.CELL_SOLID, inputs.CELL_KINETIC).astype(np.uint8)
    tree = periodic_case(lv, ijk, nv=(6, 6, 6), bc=(inputs.BC_SPECULAR,) * 6, kind=kind)
    case = inputs.lbm_case(tree, 19, noise_rel=2e-2)
    o = LO.LbmOracle(case, inputs.lbm_tau(case))
    f0 = LO.initial_f(case)
    f1 = o.step(f0, case.dt, 3)
    vol = 8.0 ** (-case.level[case.kinetic_leaves()].astype(np.float64))
    assert abs(((o.moments(f1)[0] - o.moments(f0)[0]) * vol).sum()) <= 1e-14 * (o.moments(f0)[0] * vol).sum()
    assert np.abs(f1 - f0).max() > 1e-6                       # and something did happen


def test_d3q19_transport_is_d3q27_transport_on_19_velocities():
    tree = _tree_case(seed=7)
    c19, c27 = inputs.lbm_case(tree, 19), inputs.lbm_case(tree, 27)
    o19, o27 = LO.LbmOracle(c19, 1.0), LO.LbmOracle(c27, 1.0)
    f27 = LO.initial_f(c27)
    _, _, a19 = LO.lattice(19); _, _, a27 = LO.lattice(27)
    pos = np.searchsorted(a27, a19)
    got = o19.transport(f27[:, pos], c19.dt)
    assert np.array_equal(got, o27.transport(f27, c27.dt)[:, pos])


def test_streaming_along_x_closed_form():
    """Uniform periodic level-3 grid, collisions off (tau = inf), f_i(x) = w_i (1 + eps sin 2 pi x): after n steps
    population i is M_i [1 + eps Im(g^n e^{2 pi i x})], g = 1 - c (1 - e^{-i s theta}), c = |c_x| dt / h, theta = 2 pi h
    (first-order upwind)."""
    lv, ijk = random_tree(np.random.default_rng(0), 3, 3, P, 0.0)
    tree = periodic_case(lv, ijk, nv=(6, 6, 6))
    case = inputs.lbm_case(tree, 27, noise_rel=0.0)
    o = LO.LbmOracle(case, float("inf"))
    c, w, _ = LO.lattice(27)
    x = case.centres()[case.kinetic_leaves(), 0]
    eps, n, h = 0.1, 6, 1.0 / 8
    f = w[None, :] * (1 + eps * np.sin(2 * np.pi * x))[:, None]
    for _ in range(n):
        f = o.collide(o.transport(f, case.dt), case.dt)       # dt / inf = 0: collide is the identity
    th = 2 * np.pi * h
    for i in range(27):
        cc, s = abs(c[i, 0]) * case.dt / h, np.sign(c[i, 0])
        g = 1 - cc * (1 - np.exp(-1j * s * th))
        want = w[i] * (1 + eps * np.imag(g ** n * np.exp(2j * np.pi * x)))
        assert np.abs(f[:, i] - want).max() < 5e-16
