"""Pins of the CPU oracle against what the paper and the mathematics fix.

The paper prints no worked numbers, so every pin is a closed form, an
invariant, a special case or a brute force that does not reuse the oracle's own formulas."""
import math

import numpy as np
import pytest
from scipy import optimize

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import inputs
from tests.helpers import (brute_force_faces, np_moments, periodic_case, random_tree, rel_linf, xi_grids)

P = (True, True, True)


def _noisy(case, seed, amp=0.3):
    rng = np.random.default_rng(seed)
    f = inputs.maxwellian_canonical(case, case.prim0[case.kinetic_leaves()])
    return f * (1 + amp * rng.uniform(-1, 1, f.shape))


def _volumes(case):
    return (1.0 / 8.0 ** case.level[case.kinetic_leaves()].astype(np.float64))


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("nv,vlim", [(12, 4.5), (24, 5.0)])
def test_p1_uniform_maxwellian_is_steady(nv, vlim):
    """Every leaf of a periodic 2:1 tree holds the same Maxwellian; collisions on.  Steady to round-off
    (pins S2-S6 together, sub-face areas, and reading G7: only the *discrete* Maxwellian is a fixed point)."""
    c = inputs.config1(nv=nv)
    c.vmin, c.vmax = (-vlim,) * 3, (vlim,) * 3
    prim = np.tile(np.array([[1.3, 0.4, -0.2, 0.1, 0.9]]), (c.n_leaves, 1))
    f = inputs.maxwellian_canonical(c, prim)
    o = Oracle(c)
    f1 = o.step(f, c.dt, nsteps=3)
    assert rel_linf(f1, f) < 5e-14


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("which", ["config1", "multilevel"])
def test_p2_transport_conserves_mass_momentum_energy(which):
    """Periodic adaptive tree, noisy f: face fluxes telescope, also across 2:1 faces."""
    if which == "config1":
        c = inputs.config1()
    else:
        lv, ijk = random_tree(np.random.default_rng(3), 1, 4, P, 0.3)
        c = periodic_case(lv, ijk, nv=(6, 4, 8))
    f = _noisy(c, 11)
    o = Oracle(c, kn=math.inf)
    f1 = o.transport(f, c.dt)
    V = _volumes(c)
    for a in range(5):
        before = math.fsum((V * np_moments(c, f)[:, a]).tolist())
        after = math.fsum((V * np_moments(c, f1)[:, a]).tolist())
        scale = math.fsum((V * np.abs(np_moments(c, f)[:, a])).tolist())
        assert abs(after - before) <= 2e-14 * scale, (a, before, after)
    assert rel_linf(f1, f) > 1e-4  # something moved


# ---------------------------------------------------------------- P3
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p3_free_streaming_closed_form(axis):
    """Uniform periodic grid, Kn = inf, f0 = M_i (1 + eps sin 2 pi x_j): the upwind scheme multiplies the
    Fourier mode by g_i = 1 - c_i (1 - exp(-i s_i theta)) each step."""
    lv, ijk = inputs.build_tree(3, 3, {}, P)
    c = periodic_case(lv, ijk, nv=(6, 6, 6), vlim=4.0)
    eps, nsteps = 0.1, 7
    X = xi_grids(c)
    M = np.exp(-(X[0] ** 2 + X[1] ** 2 + X[2] ** 2) / 2) / (2 * np.pi) ** 1.5
    x = c.centres()[:, axis]
    f0 = M[None, :] * (1 + eps * np.sin(2 * np.pi * x))[:, None]
    o = Oracle(c, kn=math.inf)
    dt, h = c.dt, 1.0 / 8
    f = o.step(f0, dt, nsteps=nsteps)
    xi = X[axis]
    cfl = np.abs(xi) * dt / h
    g = 1 - cfl * (1 - np.exp(-1j * np.sign(xi) * 2 * np.pi * h))
    exact = M[None, :] * (1 + eps * np.imag(g[None, :] ** nsteps * np.exp(2j * np.pi * x)[:, None]))
    assert rel_linf(f, exact) < 1e-14
    # and the continuum solution f0(x - xi t) within the first-order bound n c (1-c) theta^2 / 2 * eps
    cont = M[None, :] * (1 + eps * np.sin(2 * np.pi * (x[:, None] - xi[None, :] * nsteps * dt)))
    bound = nsteps * cfl * (1 - cfl) * (2 * np.pi * h) ** 2 / 2 * eps * M
    assert np.all(np.abs(f - cont) <= bound[None, :] * 1.05 + 1e-15)


# ---------------------------------------------------------------- P4
def test_p4_faces_config1_counts_and_brute_force():
    c = inputs.config1()
    o = Oracle(c)
    ow, ng, ar, ax, ra = o.faces()
    assert (ra == 0).sum() == 1644 and (ra != 0).sum() == 96
    got = sorted(zip(ow.tolist(), ng.tolist(), ax.tolist(), ar.tolist()))
    assert got == brute_force_faces(c.level, c.ijk, P)


@pytest.mark.parametrize("seed,periodic", [(0, P), (1, (False, False, False)), (2, (True, False, True)), (5, P)])
def test_p4_faces_random_trees(seed, periodic):
    rng = np.random.default_rng(seed)
    lv, ijk = random_tree(rng, 1, 4, periodic, 0.12)
    assert 100 < lv.shape[0] <= 1500
    bc = tuple(inputs.BC_PERIODIC if periodic[s // 2] else inputs.BC_OUTFLOW for s in range(6))
    kind = np.zeros(lv.shape[0], np.uint8)
    kind[rng.uniform(size=lv.shape[0]) < 0.1] = inputs.CELL_SOLID   # faces of solids are not interior faces
    c = periodic_case(lv, ijk, bc=bc, kind=kind)
    o = Oracle(c)
    ow, ng, ar, ax, ra = o.faces()
    got = sorted(zip(ow.tolist(), ng.tolist(), ax.tolist(), ar.tolist()))
    assert got == brute_force_faces(lv, ijk, periodic, live=kind != inputs.CELL_SOLID)
    assert np.all(ra == (lv[ng].astype(int) - lv[ow].astype(int)))
    assert set(np.unique(ra)) <= {-1, 0, 1}


def test_p4_face_based_transport_matches_cell_based():
    """Independent numpy transport: loop over the brute-force FACE list and move A xi f_up dt from the
    upwind to the downwind cell.  Pins S2/S3 including 2:1 faces."""
    lv, ijk = random_tree(np.random.default_rng(7), 1, 3, P, 0.35)
    c = periodic_case(lv, ijk, nv=(4, 6, 4))
    f = _noisy(c, 5)
    dt = c.dt
    X = xi_grids(c)
    V = 1.0 / 8.0 ** lv.astype(np.float64)
    fs = f.copy()
    for p, q, a, area in brute_force_faces(lv, ijk, P):
        flux = area * X[a] * np.where(X[a] > 0, f[p], f[q])       # through the face, towards +axis
        fs[p] -= dt / V[p] * flux
        fs[q] += dt / V[q] * flux
    got = Oracle(c, kn=math.inf).transport(f, dt)
    assert rel_linf(got, fs) < 1e-14


def test_mesh_validation_rejects_bad_trees():
    from oracle.dvm_oracle import OracleError
    lv, ijk = inputs.build_tree(2, 2, {}, P)
    c = periodic_case(lv[:-1], ijk[:-1])                     # a gap
    with pytest.raises(OracleError):
        Oracle(c)
    # 2:1 violation: level-1 cube with one octant refined twice, without balancing
    oct_ = [(i, j, k) for k in range(2) for j in range(2) for i in range(2)]
    lv = [1] * 7 + [2] * 7 + [3] * 8
    ijk = oct_[1:]                                            # level 1, octant (0,0,0) split
    ijk += oct_[:-1]                                          # level 2, its child (1,1,1) split again:
    ijk += [(2 + i, 2 + j, 2 + k) for (i, j, k) in oct_]      # level-3 leaves that touch level-1 leaves
    c = periodic_case(np.array(lv, np.uint8), np.array(ijk, np.uint32), bc=(inputs.BC_OUTFLOW,) * 6)
    with pytest.raises(OracleError):
        Oracle(c)


# ---------------------------------------------------------------- P5
def test_p5_leaf_order_and_axis_permutation_and_mirror():
    lv, ijk = random_tree(np.random.default_rng(21), 1, 3, P, 0.3)
    nv = (4, 6, 8)
    c = periodic_case(lv, ijk, nv=nv, kn=0.05)
    f = _noisy(c, 9)
    ref = Oracle(c).step(f, c.dt, 2)
    # (a) shuffled leaf list
    perm = np.random.default_rng(1).permutation(lv.shape[0])
    c2 = periodic_case(lv[perm], ijk[perm], nv=nv, kn=0.05)
    out = Oracle(c2).step(f[perm], c.dt, 2)
    assert np.array_equal(out, ref[perm])
    # (b) cyclic axis permutation x->y->z->x of both the tree and the velocity axes
    ijk3 = ijk[:, [2, 0, 1]]
    nv3 = (nv[2], nv[0], nv[1])
    c3 = periodic_case(lv, ijk3, nv=nv3, kn=0.05)
    f3 = f.reshape(-1, nv[2], nv[1], nv[0]).transpose(0, 2, 1, 3)     # new (z,y,x) = old (y,x,z)
    f3 = np.ascontiguousarray(f.reshape(-1, nv[2], nv[1], nv[0]).transpose(0, 2, 3, 1)).reshape(f.shape[0], -1)
    out3 = Oracle(c3).step(f3, c.dt, 2)
    back = out3.reshape(-1, nv[1], nv[0], nv[2]).transpose(0, 3, 1, 2).reshape(f.shape[0], -1)
    assert rel_linf(back, ref) < 1e-14
    # (c) mirror image in x: i -> 2^l-1-i and kx -> nvx-1-kx
    ijkm = ijk.copy(); ijkm[:, 0] = (1 << lv.astype(np.int64)) - 1 - ijk[:, 0]
    cm = periodic_case(lv, ijkm, nv=nv, kn=0.05)
    fm = np.ascontiguousarray(f.reshape(-1, nv[2], nv[1], nv[0])[..., ::-1]).reshape(f.shape[0], -1)
    outm = Oracle(cm).step(fm, c.dt, 2)
    backm = outm.reshape(-1, nv[2], nv[1], nv[0])[..., ::-1].reshape(f.shape[0], -1)
    assert rel_linf(backm, ref) < 1e-14


def test_p5_uniform_refined_equals_direct():
    """A uniform level-2 tree given as (level-1 cells all split) is the level-2 grid; same numbers."""
    lv_a, ijk_a = inputs.build_tree(2, 2, {}, P)
    lv_b, ijk_b = inputs.build_tree(1, 2, {1: np.ones((2, 2, 2), bool)}, P)
    ka = {tuple(x): n for n, x in enumerate(ijk_a.tolist())}
    perm = np.array([ka[tuple(x)] for x in ijk_b.tolist()])
    ca, cb = periodic_case(lv_a, ijk_a), periodic_case(lv_b, ijk_b)
    f = _noisy(ca, 2)
    assert np.array_equal(Oracle(ca).step(f, ca.dt)[perm], Oracle(cb).step(f[perm], cb.dt))


# ---------------------------------------------------------------- P6, P7
def test_p6_transport_is_linear():
    c = inputs.small(4); c.nv = (4, 4, 4)
    o = Oracle(c, kn=math.inf)
    rng = np.random.default_rng(0)
    f = rng.uniform(0, 1, (o.n_kinetic, c.Nv)); g = rng.uniform(0, 1, f.shape)
    a, b = 0.7, -1.9
    lhs = o.transport(a * f + b * g, c.dt)
    rhs = a * o.transport(f, c.dt) + b * o.transport(g, c.dt)
    assert rel_linf(lhs, rhs) < 1e-14


def test_p7_positivity_and_maximum_principle_at_cfl_one():
    c = inputs.small(4); c.nv = (4, 4, 4); c.cfl = 1.0
    o = Oracle(c, kn=math.inf)
    rng = np.random.default_rng(4)
    f = rng.uniform(0, 1, (o.n_kinetic, c.Nv)) ** 8          # many values near zero
    f1 = o.transport(f, c.dt)
    assert f1.min() >= 0.0
    # convex combination of values at the same velocity node
    assert np.all(f1.max(axis=0) <= f.max(axis=0) * (1 + 1e-15))
    assert np.all(f1.min(axis=0) >= f.min(axis=0) * (1 - 1e-15))
    # with the 1-D-style dt (G11's rejected alternative) the own-cell coefficient can go negative
    c.cfl = 1.0 * 3.0
    f2 = Oracle(c, kn=math.inf).transport(f, c.dt)
    assert f2.min() < 0.0


# ---------------------------------------------------------------- P8, G7
def _discrete_maxwellian_scipy(case, rho):
    """Independent solve of w sum m exp(alpha.m) = rho with scipy's hybrid Powell solver."""
    X, Y, Z = xi_grids(case)
    m = np.stack([np.ones_like(X), X, Y, Z, X * X + Y * Y + Z * Z])
    w = np.prod([(case.vmax[a] - case.vmin[a]) / case.nv[a] for a in range(3)])
    n = rho[0]; u = rho[1:4] / n; T = (rho[4] - n * u @ u) / (3 * n)
    a0 = np.array([np.log(n / (2 * np.pi * T) ** 1.5) - u @ u / (2 * T), *(u / T), -1 / (2 * T)])
    sol = optimize.root(lambda a: w * (m @ np.exp(a @ m)) - rho, a0, jac=lambda a: w * (m * np.exp(a @ m)) @ m.T,
                        method="hybr", tol=1e-15)
    return sol.x, np.exp(sol.x @ m)


def test_p8_newton_matches_independent_root_and_analytic_family():
    lv, ijk = inputs.build_tree(1, 1, {}, P)
    c = periodic_case(lv, ijk, nv=(12, 12, 12), vlim=4.5)
    o = Oracle(c)
    X, Y, Z = xi_grids(c)
    # (a) a pointwise Maxwellian is in the exponential family: the root is its own parameters
    n, u, T = 1.7, np.array([0.3, -0.5, 0.2]), 0.8
    f = inputs.maxwellian_canonical(c, np.array([[n, *u, T]]))[0]
    rho = np_moments(c, f[None])[0]
    alpha, it = o.newton(rho)
    expect = np.array([np.log(n / (2 * np.pi * T) ** 1.5) - u @ u / (2 * T), *(u / T), -1 / (2 * T)])
    assert 0 <= it <= 4
    assert np.allclose(alpha, expect, rtol=0, atol=5e-12)
    # (b) a bimodal f: compare with scipy's root of the same five equations
    f = 0.6 * inputs.maxwellian_canonical(c, np.array([[1.0, 1.5, 0, 0, 0.6]]))[0] \
        + 0.4 * inputs.maxwellian_canonical(c, np.array([[2.0, -0.8, 0.3, 0, 1.2]]))[0]
    rho = np_moments(c, f[None])[0]
    alpha, it = o.newton(rho)
    a_ref, M_ref = _discrete_maxwellian_scipy(c, rho)
    assert it >= 1
    assert np.allclose(alpha, a_ref, rtol=0, atol=1e-10)
    assert np.allclose(np_moments(c, np.exp(alpha @ np.stack([np.ones_like(X), X, Y, Z, X * X + Y * Y + Z * Z]))[None])[0],
                       rho, rtol=1e-12)


def test_p8_relaxation_conserves_moments_and_fixes_maxwellians():
    c = inputs.config1()
    o = Oracle(c)
    f = _noisy(c, 3, amp=0.5)
    f1 = o.relax(f, 0.05)
    m0, m1 = np_moments(c, f), np_moments(c, f1)
    assert np.abs(m1 - m0).max() <= 2e-13 * np.abs(m0).max()
    assert rel_linf(f1, f) > 1e-4
    # discrete Maxwellians exp(alpha.m) are fixed points
    X, Y, Z = xi_grids(c)
    rng = np.random.default_rng(8)
    al = np.stack([rng.uniform(-3, -1, 568), rng.uniform(-.5, .5, 568), rng.uniform(-.5, .5, 568),
                   rng.uniform(-.5, .5, 568), rng.uniform(-0.7, -0.4, 568)], axis=1)
    M = np.exp(al @ np.stack([np.ones_like(X), X, Y, Z, X * X + Y * Y + Z * Z]))
    assert rel_linf(o.relax(M, 0.002), M) < 2e-14


# ---------------------------------------------------------------- P9, P10
def test_p9_homogeneous_relaxation_closed_form_and_p10_entropy():
    lv, ijk = inputs.build_tree(1, 1, {}, P)
    c = periodic_case(lv, ijk, nv=(10, 10, 10), vlim=5.0, kn=0.2)
    f0 = 0.5 * inputs.maxwellian_canonical(c, np.array([[1.0, 1.2, 0, 0, 0.7]])) \
        + 0.5 * inputs.maxwellian_canonical(c, np.array([[1.0, -1.2, 0.4, 0, 1.1]]))
    f0 = np.tile(f0, (8, 1))
    rho = np_moments(c, f0)[0]
    _, M = _discrete_maxwellian_scipy(c, rho)
    n = rho[0]; T = (rho[4] - (rho[1:4] @ rho[1:4]) / n) / (3 * n)
    nu = 1.0 * n * np.sqrt(T) / 0.2                                   # G9 with c_nu = 1, omega = 1/2
    dt, nsteps = 0.01, 6
    o = Oracle(c)
    w = np.prod([(c.vmax[a] - c.vmin[a]) / c.nv[a] for a in range(3)])
    f, H = f0, [w * np.sum(f0[0] * np.log(f0[0]))]
    for _ in range(nsteps):
        f = o.step(f, dt)
        H.append(w * np.sum(f[0] * np.log(f[0])))
    exact = M[None, :] + (1 - dt * nu) ** nsteps * (f0 - M[None, :])
    assert rel_linf(f, exact) < 1e-12
    assert np.all(np.diff(H) < 0)                                      # P10: entropy decreases


# ---------------------------------------------------------------- P11 and the ghost states
def _replicate(f_small, cs, cb, mirror_axis=None):
    """State on the big periodic cube `cb` that repeats the small cube `cs` (h ratio 2), mirrored
    (cell and velocity) in `mirror_axis` for the second copy."""
    ns = 1 << int(cs.level[0])
    key = {tuple(x): r for r, x in enumerate(cs.ijk.tolist())}
    nvx, nvy, nvz = cs.nv
    out = np.empty((cb.n_leaves, cs.Nv))
    for r, x in enumerate(cb.ijk.tolist()):
        x = list(x); flip = False
        if mirror_axis is not None and x[mirror_axis] >= ns:
            x[mirror_axis] = 2 * ns - 1 - x[mirror_axis]; flip = True
        row = f_small[key[tuple(v % ns for v in x)]].reshape(nvz, nvy, nvx)
        if flip:
            row = np.flip(row, axis=2 - mirror_axis)
        out[r] = row.reshape(-1)
    return out


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p11_specular_box_equals_mirrored_periodic_domain(axis):
    """A box with specular walls on one axis is the half of a periodic domain twice as long whose
    state is mirror-symmetric (cells and velocities).  Pins the specular ghost (a1b)."""
    lv, ijk = inputs.build_tree(2, 2, {}, P)
    bc = [inputs.BC_PERIODIC] * 6; bc[2 * axis] = bc[2 * axis + 1] = inputs.BC_SPECULAR
    cs = periodic_case(lv, ijk, nv=(4, 6, 4), bc=tuple(bc), kn=0.3)
    lvb, ijkb = inputs.build_tree(3, 3, {}, P)
    cb = periodic_case(lvb, ijkb, nv=(4, 6, 4), kn=0.15)          # dt halves, so nu doubles: same dt*nu
    fs = _noisy(cs, 13)
    fb = _replicate(fs, cs, cb, mirror_axis=axis)
    dts = 0.01
    outs = Oracle(cs).step(fs, dts, 3)
    outb = Oracle(cb).step(fb, dts / 2, 3)                          # h is half as large
    assert rel_linf(outb, _replicate(outs, cs, cb, mirror_axis=axis)) < 1e-14
    # mass and energy conserved by transport in a fully closed box; wall-normal momentum is not
    cs2 = periodic_case(lv, ijk, nv=(4, 6, 4), bc=(inputs.BC_SPECULAR,) * 6)
    f1 = Oracle(cs2, kn=math.inf).transport(fs, dts)
    m0, m1 = np_moments(cs2, fs).sum(0), np_moments(cs2, f1).sum(0)
    assert abs(m1[0] - m0[0]) < 1e-14 * m0[0] and abs(m1[4] - m0[4]) < 1e-14 * m0[4]


def test_solid_leaves_act_as_specular_walls():
    """x in [0.5,1) SOLID in a periodic level-2 cube: the live half sees walls on both sides and equals
    a level-1 ... no: a level-2 box half as wide.  Compare with a specular box built as its own cube."""
    lv, ijk = inputs.build_tree(2, 2, {}, P)
    kind = np.where(ijk[:, 0] >= 2, inputs.CELL_SOLID, inputs.CELL_KINETIC).astype(np.uint8)
    c_solid = periodic_case(lv, ijk, nv=(4, 4, 4), kind=kind, kn=0.3)
    lv1, ijk1 = inputs.build_tree(1, 1, {}, P)
    bc = (inputs.BC_SPECULAR, inputs.BC_SPECULAR) + (inputs.BC_PERIODIC,) * 4
    c_box = periodic_case(lv1, ijk1, nv=(4, 4, 4), bc=bc, kn=0.6)   # dt doubles: keep dt*nu
    f_box = _noisy(c_box, 17)
    kin = c_solid.kinetic_leaves()
    key = {tuple(x): r for r, x in enumerate(ijk1.tolist())}
    rows = np.array([key[(x[0] % 2, x[1] % 2, x[2] % 2)] for x in ijk[kin].tolist()])
    out_solid = Oracle(c_solid).step(f_box[rows], 0.01, 3)
    out_box = Oracle(c_box).step(f_box, 0.02, 3)
    assert rel_linf(out_solid, out_box[rows]) < 1e-14


@pytest.mark.parametrize("ghost", ["inflow", "fluid"])
def test_matching_inflow_and_fluid_ghosts_keep_a_uniform_state(ghost):
    """Inflow (a1b) and fluid-leaf (G13) ghosts are pointwise Maxwellians: when their
    state equals the uniform interior Maxwellian nothing changes (transport only, so the discrete
    Maxwellian plays no role).  A wrong normalisation, sign or temperature convention fails here."""
    state = np.array([0.9, 0.7, -0.3, 0.2, 1.3])
    lv, ijk = random_tree(np.random.default_rng(2), 2, 3, (False,) * 3, 0.2)
    n = lv.shape[0]
    kind = np.zeros(n, np.uint8)
    bc = (inputs.BC_INFLOW, inputs.BC_OUTFLOW, inputs.BC_INFLOW, inputs.BC_INFLOW, inputs.BC_OUTFLOW, inputs.BC_INFLOW)
    inflow = np.tile(state, (6, 1))
    fm = None
    if ghost == "fluid":
        kind[np.random.default_rng(3).uniform(size=n) < 0.4] = inputs.CELL_FLUID
        fm = np.tile(state, (n, 1))
    c = periodic_case(lv, ijk, nv=(6, 6, 6), vlim=6.0, bc=bc, kind=kind, inflow=inflow, fluid_moments=fm)
    f = inputs.maxwellian_canonical(c, np.tile(state, (len(c.kinetic_leaves()), 1)))
    f1 = Oracle(c, kn=math.inf).step(f, c.dt, 2)
    assert rel_linf(f1, f) < 1e-14
    # and a different ghost state does change the cells that touch it
    c.inflow[:, 0] = 2.0
    if fm is not None:
        c.fluid_moments[:, 0] = 2.0
    assert rel_linf(Oracle(c, kn=math.inf).step(f, c.dt, 1), f) > 1e-3


def test_outflow_is_zero_gradient():
    """1-D check: uniform state, outflow at both x ends -> steady; with a gradient, the boundary cell's
    update equals the upwind formula with ghost = own."""
    lv, ijk = inputs.build_tree(2, 2, {}, P)
    bc = (inputs.BC_OUTFLOW, inputs.BC_OUTFLOW) + (inputs.BC_PERIODIC,) * 4
    c = periodic_case(lv, ijk, nv=(4, 2, 2), bc=bc)
    f = _noisy(c, 23, amp=0.0) * (1 + 0.2 * c.centres()[:, 0])[:, None]
    X = xi_grids(c)[0]
    dt, h = c.dt, 0.25
    f1 = Oracle(c, kn=math.inf).transport(f, dt)
    row = {tuple(x): r for r, x in enumerate(ijk.tolist())}
    for j in range(2):
        for k in range(2):
            cells = [row[(i, j, k)] for i in range(4)]
            for pos, r in enumerate(cells):
                left = f[cells[pos - 1]] if pos > 0 else f[r]
                right = f[cells[pos + 1]] if pos < 3 else f[r]
                expect = f[r] - dt / h * np.where(X > 0, X * (f[r] - left), X * (right - f[r]))
                assert np.allclose(f1[r], expect, rtol=1e-14, atol=0)


def test_moments_report_half_energy():
    c = inputs.config1()
    f = _noisy(c, 1)
    mom = Oracle(c).moments(f)
    ref = np_moments(c, f).T
    ref[4] *= 0.5
    assert rel_linf(mom, ref) < 1e-14
