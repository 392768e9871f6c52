"""lbm_oracle.py -- TEST INFRASTRUCTURE ONLY.  Plain fp64 CPU statement of one step of the lattice-Boltzmann variant of
the UFS kinetic module, written from the paper.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may use it; it shares nothing with paper_1503_00707_b200/csrc.

What is computed, per step:
  L1  "The LBM Module in UFS is designed as a subset of the DVM kinetic solvers ... uses 3x3 (D2Q9), 19 (D3Q19), and 3x3x3
      (D3Q27) velocity lattices": the velocity nodes are those of the 3x3x3 DVM grid with nodes -1, 0, 1;
      D3Q19 leaves the eight corners out.
  L2  transport: the finite-volume scheme of the DVM solver ("The finite volume LBM implementation", PAPER.md:227;
      "summations over neighboring cells ... from 6 to 6x4 on an Octree mesh"): f* = f - dt sum_F (A_F/V)
      (c_i . n_F) f_up -- oracle/dvm_oracle.c, steps S2/S3, called as a library step on the 27-node grid with
      collisions off (pinned in tests/test_oracle_pins.py; a velocity that is left out stays zero: S2 is linear and
      acts on every velocity by itself).
  L3  rho = sum_i f*_i,  rho u = sum_i c_i f*_i
  L4  f_eq_i = w_i rho (1 + c_i.u / cs^2 + (c_i.u)^2 / (2 cs^4) - u^2 / (2 cs^2)),  cs = 1/sqrt(3)
  L5  f' = f* + (dt / tau) (f_eq - f*)        (BGK term -(f - f_eq)/tau; forward Euler like S6, reading G4/G5)
Ghost states: periodic, specular walls and SOLID leaves, outflow as in the DVM step; INFLOW: f_eq of the side's (rho, u)
("equilibrium distribution function for initial and boundary conditions").

Readings: the lattice weights w_i are the standard ones the paper's Ref. [44] uses and PAPER.md does not
print: D3Q19 1/3, 1/18, 1/36; D3Q27 8/27, 2/27, 1/54, 1/216 for |c|^2 = 0, 1, 2, 3 -- pinned by the isotropy
conditions they are the unique solution of (tests/test_lbm_oracle_pins.py).

Pins: sum w = 1, sum w c_a c_b = cs^2 delta_ab, sum w c_a c_b c_g c_d = cs^4 (3 delta-pair terms); moments of f_eq:
sum f_eq = rho, sum c f_eq = rho u, sum c_a c_b f_eq = rho (cs^2 delta_ab + u_a u_b); relaxation conserves rho and rho u;
a uniform equilibrium is steady on a 2:1 periodic tree; mass is conserved by the whole step on a periodic tree.
"""
import numpy as np

from oracle.dvm_oracle import Oracle

CS2 = 1.0 / 3.0


def lattice(q):
    """(c [Q,3] integers, w [Q], active [Q] indices into the 27-node canonical order (kz*3+ky)*3+kx, c = k - 1)."""
    assert q in (19, 27)
    idx, cs, ws = [], [], []
    w19 = {0: 1.0 / 3.0, 1: 1.0 / 18.0, 2: 1.0 / 36.0}
    w27 = {0: 8.0 / 27.0, 1: 2.0 / 27.0, 2: 1.0 / 54.0, 3: 1.0 / 216.0}
    for kz in range(3):
        for ky in range(3):
            for kx in range(3):
                c = (kx - 1, ky - 1, kz - 1)
                n2 = c[0] ** 2 + c[1] ** 2 + c[2] ** 2
                if q == 19 and n2 > 2:
                    continue
                idx.append((kz * 3 + ky) * 3 + kx)
                cs.append(c)
                ws.append((w19 if q == 19 else w27)[n2])
    return np.array(cs, np.float64), np.array(ws), np.array(idx, np.int64)


def equilibrium(q, rho, u):
    """L4 for arrays rho [n], u [n,3] -> [n,Q]."""
    c, w, _ = lattice(q)
    out = np.empty((rho.shape[0], c.shape[0]))
    for i in range(c.shape[0]):
        cu = c[i, 0] * u[:, 0] + c[i, 1] * u[:, 1] + c[i, 2] * u[:, 2]
        uu = u[:, 0] ** 2 + u[:, 1] ** 2 + u[:, 2] ** 2
        out[:, i] = w[i] * rho * (1.0 + cu / CS2 + cu * cu / (2.0 * CS2 * CS2) - uu / (2.0 * CS2))
    return out


def moments(q, f):
    """L3: rho [n], rho u [n,3]."""
    c, _, _ = lattice(q)
    rho = np.zeros(f.shape[0])
    mom = np.zeros((f.shape[0], 3))
    for i in range(c.shape[0]):
        rho += f[:, i]
        for a in range(3):
            mom[:, a] += c[i, a] * f[:, i]
    return rho, mom


class LbmOracle:
    """case: a Case made by inputs.lbm_case (3x3x3 grid on [-1.5,1.5]^3, meta['lattice'], meta['omega'])."""

    def __init__(self, case, tau, window=False):
        assert tuple(case.nv) == (3, 3, 3) and tuple(case.vmin) == (-1.5,) * 3 and tuple(case.vmax) == (1.5,) * 3
        self.q = int(case.meta["lattice"])
        self.tau = float(tau)
        self.c, self.w, self.active = lattice(self.q)
        self.dvm = Oracle(case, kn=float("inf"), window=window)   # L2: transport only (window: a part of a mesh, bench sample)
        self.n = self.dvm.n_kinetic
        for s in range(6):
            if case.bc[s] == 2:                                 # INFLOW: equilibrium of the side's (rho, u)
                t = np.zeros(27)
                t[self.active] = equilibrium(self.q, np.array([case.inflow[s][0]]), np.array([case.inflow[s][1:4]]))[0]
                self.dvm.set_inflow_table(s, t)

    def transport(self, f, dt):
        f27 = np.zeros((self.n, 27))
        f27[:, self.active] = f
        return self.dvm.transport(f27, dt)[:, self.active]

    def collide(self, fstar, dt):
        rho, mom = moments(self.q, fstar)
        feq = equilibrium(self.q, rho, mom / rho[:, None])
        return fstar + (dt / self.tau) * (feq - fstar)

    def step(self, f, dt, nsteps=1):
        for _ in range(nsteps):
            f = self.collide(self.transport(f, dt), dt)
        return f

    def moments(self, f):
        """[4, n]: rho, rho ux, rho uy, rho uz."""
        rho, mom = moments(self.q, f)
        return np.vstack([rho[None, :], mom.T])


def initial_f(case):
    """f(t=0) = f_eq of case.prim0 (rho, u) on the kinetic leaves, times the case's seeded relative noise."""
    kin = case.kinetic_leaves()
    q = int(case.meta["lattice"])
    f = equilibrium(q, case.prim0[kin, 0], case.prim0[kin, 1:4])
    if case.noise_rel:
        rng = np.random.default_rng(150300707 + 900 + case.noise_seed)
        f = f * (1.0 + case.noise_rel * rng.uniform(-1, 1, f.shape))
    return f
