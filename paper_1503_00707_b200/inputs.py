"""Seeded synthetic inputs for the DVM step: octree leaf lists, velocity grids, initial states, masks.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic (no flux, no moments of f, no Newton, no relaxation).  It only *describes problems*:
which leaves exist, what the boundary codes are, which macroscopic state each leaf starts from and
the distribution function that state implies at t = 0.  The recipes are the five configurations of
BASELINE.json as made concrete in SURVEY.md section 8(d); they stand
in for the paper's own workloads (sphere flow and X-51A waverider: PAPER.md:193, 207-209), whose
geometry is not public.

Conventions (section 2.1 for the tree, PAPER.md:93 for the velocity grid):
  * a leaf is (level l, integer coordinates (i, j, k) at its own level), edge h = L / 2**l;
  * velocity node k on axis b is xi = vmin_b + (k + 1/2) dv_b, canonical index (kz*nvy + ky)*nvx + kx;
  * boundary sides are ordered -x, +x, -y, +y, -z, +z.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# codes shared with include/ufs_dvm.h (plain integers; the header is the authority for the C side)
BC_PERIODIC, BC_SPECULAR, BC_INFLOW, BC_OUTFLOW = 0, 1, 2, 3
CELL_KINETIC, CELL_FLUID, CELL_SOLID = 0, 1, 2
STORE_F64, STORE_F32 = 0, 1

SEED_BASE = 150300707  # numpy.random.default_rng(SEED_BASE + config number)


@dataclass
class Case:
    """One problem statement: mesh + velocity grid + gas model + initial state + run length."""
    name: str
    level: np.ndarray            # [n] uint8
    ijk: np.ndarray              # [n,3] uint32, coordinates at the leaf's own level
    kind: np.ndarray             # [n] uint8 CELL_*
    domain_len: float
    bc: tuple                    # 6 x BC_*
    inflow: np.ndarray           # [6,5] (n,ux,uy,uz,T) for INFLOW sides
    fluid_moments: Optional[np.ndarray]  # [n,5] primitive (n,ux,uy,uz,T); used for FLUID leaves
    nv: tuple
    vmin: tuple
    vmax: tuple
    kn: float
    visc_exp: float
    nu_prefactor: float
    storage: int
    cfl: float
    nsteps: int
    prim0: np.ndarray            # [n,5] primitive state (n,ux,uy,uz,T) of every leaf at t=0
    noise_rel: float = 0.0       # relative uniform noise per phase cell (config 1)
    noise_seed: int = 0
    meta: dict = field(default_factory=dict)

    # ---- derived quantities that are part of the problem statement, not of the method ----
    @property
    def n_leaves(self) -> int:
        return int(self.level.shape[0])

    @property
    def Nv(self) -> int:
        return int(self.nv[0] * self.nv[1] * self.nv[2])

    def kinetic_leaves(self) -> np.ndarray:
        """Indices (into the leaf list, ascending) of the KINETIC leaves; this is the oracle's cell order."""
        return np.nonzero(self.kind == CELL_KINETIC)[0]

    def xi_nodes(self, axis: int) -> np.ndarray:
        dv = (self.vmax[axis] - self.vmin[axis]) / self.nv[axis]
        return self.vmin[axis] + (np.arange(self.nv[axis]) + 0.5) * dv

    def centres(self, idx=None) -> np.ndarray:
        lv = self.level if idx is None else self.level[idx]
        ij = self.ijk if idx is None else self.ijk[idx]
        h = self.domain_len / (2.0 ** lv.astype(np.float64))
        return (ij.astype(np.float64) + 0.5) * h[:, None]

    @property
    def dt(self) -> float:
        """dt = CFL * h_min / (xi_max_x + xi_max_y + xi_max_z) over non-solid leaves."""
        live = self.kind != CELL_SOLID
        hmin = self.domain_len / 2.0 ** int(self.level[live].max())
        s = sum(float(np.abs(self.xi_nodes(a)).max()) for a in range(3))
        return self.cfl * hmin / s


# ----------------------------------------------------------------------------------------------
# initial distribution function (an input: the state the run starts from)
# ----------------------------------------------------------------------------------------------
def maxwellian_canonical(case: Case, prim: np.ndarray) -> np.ndarray:
    """Pointwise Maxwellian n/(2 pi T)^{3/2} exp(-|xi-u|^2/(2T)) at every velocity node, canonical order.

    prim: [m,5] -> returns [m, Nv] float64.  Used only to write the initial condition."""
    xs, ys, zs = (case.xi_nodes(a) for a in range(3))
    n, ux, uy, uz, T = (prim[:, c][:, None] for c in range(5))
    ex = np.exp(-(xs[None, :] - ux) ** 2 / (2 * T))           # [m,nvx]
    ey = np.exp(-(ys[None, :] - uy) ** 2 / (2 * T))
    ez = np.exp(-(zs[None, :] - uz) ** 2 / (2 * T))
    a = n / (2 * np.pi * T) ** 1.5
    f = a[:, :, None, None] * ez[:, :, None, None] * ey[:, None, :, None] * ex[:, None, None, :]
    return f.reshape(prim.shape[0], -1)


def initial_f(case: Case, rows: Optional[np.ndarray] = None) -> np.ndarray:
    """f at t=0 for the kinetic leaves, [n_kinetic, Nv] float64, rows in kinetic_leaves() order,
    velocities in canonical order.  `rows` selects a subset of kinetic rows (positions in that order)."""
    kin = case.kinetic_leaves()
    sel = np.arange(kin.size) if rows is None else np.asarray(rows)
    f = maxwellian_canonical(case, case.prim0[kin[sel]])
    if case.noise_rel:
        # one Generator per kinetic row so any subset reproduces the same bits
        for r, row in enumerate(sel):
            rng = np.random.default_rng([case.noise_seed, int(row)])
            f[r] *= 1.0 + case.noise_rel * rng.uniform(-1.0, 1.0, f.shape[1])
    if case.storage == STORE_F32:
        f = f.astype(np.float32).astype(np.float64)   # both sides start from the same fp32 bits
    return f


# ----------------------------------------------------------------------------------------------
# octree construction on dense per-level boolean grids (vectorised; up to level 8 = 256^3)
# ----------------------------------------------------------------------------------------------
def _pool2(a):
    n = a.shape[0] // 2
    return a.reshape(n, 2, n, 2, n, 2).any(axis=(1, 3, 5))


def _up2(a):
    return a.repeat(2, 0).repeat(2, 1).repeat(2, 2)


def _dilate26(a, periodic):
    out = a.copy()
    for ax in range(3):
        b = out.copy()
        for s in (1, -1):
            r = np.roll(out, s, axis=ax)
            if not periodic[ax]:
                sl = [slice(None)] * 3
                sl[ax] = 0 if s == 1 else -1
                r[tuple(sl)] = False
            b |= r
        out = b
    return out


def build_tree(base: int, lmax: int, split: dict, periodic) -> tuple:
    """split[l] (bool [2^l]^3, for base <= l < lmax) marks level-l cells that must be divided.
    Cells below `base` are always divided.  Then 2:1 balance over all 26 neighbours (PAPER.md:45,
    both constraints), with wrap on periodic axes.  Returns (level u8 [n], ijk u32 [n,3]) with leaves
    listed level by level in raster order (deliberately NOT Morton order)."""
    periodic = tuple(bool(p) for p in periodic)
    sp = {}
    for l in range(lmax):
        if l < base:
            sp[l] = np.ones((2 ** l,) * 3, bool)
        else:
            sp[l] = np.array(split.get(l, np.zeros((2 ** l,) * 3, bool)), dtype=bool)
    # a split cell's ancestors must be split too
    for l in range(lmax - 1, 0, -1):
        sp[l - 1] |= _pool2(sp[l])
    # balance, fine to coarse: every cell adjacent (26-neighbourhood) to a split cell must exist
    for l in range(lmax - 1, 0, -1):
        must_exist = _dilate26(sp[l], periodic)
        sp[l - 1] |= _pool2(must_exist)
    exists = {0: np.ones((1, 1, 1), bool)}
    for l in range(1, lmax + 1):
        exists[l] = _up2(sp[l - 1])
    sp[lmax] = np.zeros((2 ** lmax,) * 3, bool)
    levels, coords = [], []
    for l in range(lmax + 1):
        leaf = exists[l] & ~sp[l]
        if leaf.any():
            c = np.argwhere(leaf).astype(np.uint32)
            coords.append(c)
            levels.append(np.full(c.shape[0], l, np.uint8))
    return np.concatenate(levels), np.concatenate(coords)


def _descendant_pred_to_splits(base, lmax, pred_lmax):
    """SURVEY.md 8(d) tree rule: a cell at level l<lmax is split iff at least one of its level-lmax
    descendant centres satisfies the predicate."""
    split, p = {}, pred_lmax
    for l in range(lmax - 1, base - 1, -1):
        p = _pool2(p)
        split[l] = p.copy()
    return split


def _centres_grid(l):
    c = (np.arange(2 ** l) + 0.5) / 2 ** l
    return np.meshgrid(c, c, c, indexing="ij")


def _fourier_field(rng, x, nmodes=8):
    """g(x) = sum_m a_m sin(2 pi k_m.x + phi_m) / sum|a_m|, integer k_m in {-2..2}^3 \\ 0.  |g| <= 1."""
    ks = []
    while len(ks) < nmodes:
        k = rng.integers(-2, 3, 3)
        if np.any(k != 0):
            ks.append(k)
    ks = np.array(ks, dtype=np.float64)
    a = rng.uniform(0.2, 1.0, nmodes)
    ph = rng.uniform(0, 2 * np.pi, nmodes)
    g = np.zeros(x.shape[0])
    for m in range(nmodes):
        g += a[m] * np.sin(2 * np.pi * (x @ ks[m]) + ph[m])
    return g / np.abs(a).sum()


def _case(name, level, ijk, kind, bc, nv, vlim, kn, storage, cfl, nsteps, prim0,
          inflow=None, fluid_moments=None, noise_rel=0.0, noise_seed=0, meta=None):
    return Case(name=name, level=np.ascontiguousarray(level, np.uint8),
                ijk=np.ascontiguousarray(ijk, np.uint32), kind=np.ascontiguousarray(kind, np.uint8),
                domain_len=1.0, bc=tuple(bc),
                inflow=np.zeros((6, 5)) if inflow is None else np.ascontiguousarray(inflow, np.float64),
                fluid_moments=None if fluid_moments is None else np.ascontiguousarray(fluid_moments, np.float64),
                nv=(nv,) * 3, vmin=(-vlim,) * 3, vmax=(vlim,) * 3, kn=kn, visc_exp=0.5, nu_prefactor=1.0,
                storage=storage, cfl=cfl, nsteps=nsteps, prim0=np.ascontiguousarray(prim0, np.float64),
                noise_rel=noise_rel, noise_seed=noise_seed, meta=meta or {})


# ----------------------------------------------------------------------------------------------
# the five configurations (BASELINE.json "configs", SURVEY.md 8(d) rows 1, 2, 3/3', 4-lit/4, 5)
# `scale="small"` gives a reduced version of the same recipe that the oracle steps in seconds.
# ----------------------------------------------------------------------------------------------
def config1(nv: int = 12, base: int = 3) -> Case:
    """Tiny periodic 2:1 tree: base-3 cube, the level-3 leaves with centre within 0.2 of the cube
    centre refined once.  568 leaves (504 L3 + 64 L4) for base=3."""
    X, Y, Z = _centres_grid(base)
    s = ((X - .5) ** 2 + (Y - .5) ** 2 + (Z - .5) ** 2) < 0.2 ** 2
    level, ijk = build_tree(base, base + 1, {base: s}, (True,) * 3)
    n = level.shape[0]
    c = (ijk + 0.5) / (2.0 ** level)[:, None]
    prim = np.zeros((n, 5))
    prim[:, 0] = 1 + 0.05 * np.sin(2 * np.pi * c[:, 0])
    prim[:, 4] = 1.0
    return _case("config1", level, ijk, np.zeros(n, np.uint8), (BC_PERIODIC,) * 6, nv, 4.5, 0.1,
                 STORE_F64, 0.4, 10, prim, noise_rel=1e-3, noise_seed=SEED_BASE + 1)


def config2(level_: int = 6, nv: int = 24, nsteps: int = 50) -> Case:
    """Sod tube on a uniform grid: specular y/z walls, zero-gradient x ends."""
    level, ijk = build_tree(level_, level_, {}, (False,) * 3)
    n = level.shape[0]
    c = (ijk + 0.5) / (2.0 ** level)[:, None]
    left = c[:, 0] < 0.5
    prim = np.zeros((n, 5))
    prim[:, 0] = np.where(left, 1.0, 0.125)
    prim[:, 4] = np.where(left, 1.0, 0.8)
    bc = (BC_OUTFLOW, BC_OUTFLOW, BC_SPECULAR, BC_SPECULAR, BC_SPECULAR, BC_SPECULAR)
    return _case("config2", level, ijk, np.zeros(n, np.uint8), bc, nv, 5.0, 0.01, STORE_F64, 0.4, nsteps, prim)


MACH2_INFLOW = (1.0, 2.0 * np.sqrt(5.0 / 3.0), 0.0, 0.0, 1.0)   # Mach 2, gamma = 5/3, T = 1


def _sphere_tree(base, lmax):
    X, Y, Z = _centres_grid(lmax)
    r = np.sqrt((X - .3) ** 2 + (Y - .5) ** 2 + (Z - .5) ** 2)
    split = _descendant_pred_to_splits(base, lmax, (r > 0.08) & (r < 0.14))
    level, ijk = build_tree(base, lmax, split, (False,) * 3)
    c = (ijk + 0.5) / (2.0 ** level)[:, None]
    rc = np.sqrt((c[:, 0] - .3) ** 2 + (c[:, 1] - .5) ** 2 + (c[:, 2] - .5) ** 2)
    kind = np.where(rc < 0.1, CELL_SOLID, CELL_KINETIC).astype(np.uint8)
    return level, ijk, kind, c


_SPHERE_BC = (BC_INFLOW, BC_OUTFLOW, BC_SPECULAR, BC_SPECULAR, BC_SPECULAR, BC_SPECULAR)


def config3(base: int = 4, lmax: int = 7, nv: int = 24, nsteps: int = 20) -> Case:
    """Mach-2 flow past a staircase sphere (solid leaves removed, specular at their faces).
    lmax=7 is the literal reading (26 312 live leaves), lmax=8 is 3' (154 188)."""
    level, ijk, kind, c = _sphere_tree(base, lmax)
    n = level.shape[0]
    prim = np.tile(np.array(MACH2_INFLOW), (n, 1))
    inflow = np.zeros((6, 5)); inflow[0] = MACH2_INFLOW
    return _case(f"config3_l{lmax}", level, ijk, kind, _SPHERE_BC, nv, 6.0, 0.05, STORE_F64, 0.4, nsteps,
                 prim, inflow=inflow)


def _boxes_pred(rng, nboxes, lmax, pred=None, side_scale=1.0):
    n = 2 ** lmax
    c = (np.arange(n) + 0.5) / n
    if pred is None:
        pred = np.zeros((n,) * 3, bool)
    for _ in range(nboxes):
        s = rng.uniform(0.02, 0.1) * side_scale
        lo = rng.uniform(0, 1, 3)
        m = [((c - lo[a]) % 1.0) < s for a in range(3)]
        pred |= m[0][:, None, None] & m[1][None, :, None] & m[2][None, None, :]
    return pred


def config4_tree(base=6, lmax=8, target_leaves: Optional[int] = None, nboxes=32, side_scale=1.0):
    """Periodic tree refined to lmax inside random axis-aligned periodic cubes.  With target_leaves the
    box stream is extended (same Generator) until the balanced leaf count first reaches the target."""
    rng = np.random.default_rng(SEED_BASE + 4)
    pred = _boxes_pred(rng, nboxes, lmax, side_scale=side_scale)
    used = nboxes
    while True:
        level, ijk = build_tree(base, lmax, _descendant_pred_to_splits(base, lmax, pred), (True,) * 3)
        if target_leaves is None or level.shape[0] >= target_leaves:
            return level, ijk, used
        # add boxes in batches proportional to the shortfall, then single steps near the target
        short = target_leaves - level.shape[0]
        step = max(1, int(0.5 * short / max(1.0, level.shape[0] / used)))
        pred = _boxes_pred(rng, step, lmax, pred, side_scale=side_scale)
        used += step


def config4(base: int = 6, lmax: int = 8, nv: int = 24, nsteps: int = 10,
            target_leaves: Optional[int] = 1_000_000, nboxes: int = 32, side_scale: float = 1.0) -> Case:
    """Paper-scale periodic kinetic octree, fp32 storage.  target_leaves=None gives "4-lit" (32 boxes)."""
    level, ijk, used = config4_tree(base, lmax, target_leaves, nboxes, side_scale)
    n = level.shape[0]
    c = (ijk + 0.5) / (2.0 ** level)[:, None]
    rng = np.random.default_rng(SEED_BASE + 40)
    g = [_fourier_field(rng, c) for _ in range(5)]
    prim = np.zeros((n, 5))
    prim[:, 0] = 1.25 + 0.75 * g[0]
    prim[:, 1:4] = 0.5 * np.stack(g[1:4], axis=1)
    prim[:, 4] = 1.1 + 0.4 * g[4]
    return _case("config4" if target_leaves else "config4_lit", level, ijk, np.zeros(n, np.uint8),
                 (BC_PERIODIC,) * 6, nv, 6.0, 0.02, STORE_F32, 0.4, nsteps, prim, meta={"boxes": used})


def config5(base: int = 4, lmax: int = 7, nv: int = 24, nsteps: int = 20, kinetic_fraction: float = 0.3) -> Case:
    """Hybrid mask on the sphere tree: the 30 % of live leaves with the largest |grad n| h / n of an
    analytic seeded density field are KINETIC, the rest FLUID with frozen moments."""
    level, ijk, kind, c = _sphere_tree(base, lmax)
    n = level.shape[0]
    rng = np.random.default_rng(SEED_BASE + 5)
    cen = np.array([.3, .5, .5])
    d = c - cen
    r = np.sqrt((d ** 2).sum(1))
    g = _fourier_field(rng, c)
    bump = np.exp(-(r - 0.12) ** 2 / (2 * 0.03 ** 2))
    dens = 1 + 1.3 * bump + 0.05 * g
    # gradient of the radial part analytically, of g by centred differences of the analytic field
    eps = 1e-6
    rng2 = np.random.default_rng(SEED_BASE + 5)
    gg = np.stack([(_fourier_field(np.random.default_rng(SEED_BASE + 5), c + eps * e)
                    - _fourier_field(np.random.default_rng(SEED_BASE + 5), c - eps * e)) / (2 * eps)
                   for e in np.eye(3)], axis=1)
    del rng2
    grad = (1.3 * bump * (-(r - 0.12) / 0.03 ** 2))[:, None] * d / np.maximum(r, 1e-300)[:, None] + 0.05 * gg
    h = 1.0 / 2.0 ** level
    ind = np.sqrt((grad ** 2).sum(1)) * h / dens
    live = np.nonzero(kind != CELL_SOLID)[0]
    nk = int(np.floor(kinetic_fraction * live.size))
    # largest indicator first; ties broken by position in the leaf list (stable sort)
    order = live[np.argsort(-ind[live], kind="stable")]
    kind = kind.copy()
    kind[live] = CELL_FLUID
    kind[order[:nk]] = CELL_KINETIC
    prim = np.zeros((n, 5))
    prim[:, 0] = dens
    prim[:, 1] = MACH2_INFLOW[1] * (1 - 0.5 * np.exp(-(r - 0.12) ** 2 / (2 * 0.05 ** 2)))
    prim[:, 4] = 1 + 0.5 * (dens - 1)
    inflow = np.zeros((6, 5)); inflow[0] = MACH2_INFLOW
    return _case(f"config5_l{lmax}", level, ijk, kind, _SPHERE_BC, nv, 6.0, 0.05, STORE_F64, 0.4, nsteps,
                 prim, inflow=inflow, fluid_moments=prim.copy())


def small(config: int) -> Case:
    """Reduced versions of the five recipes: same structure (level jumps, boundary kinds, mask, storage),
    a few hundred leaves, so the oracle steps them in seconds while a slab still spans several tiles."""
    if config == 1:
        return config1()
    if config == 2:
        return config2(level_=3, nv=24, nsteps=4)
    if config == 3:
        return config3(base=3, lmax=5, nv=24, nsteps=3)
    if config == 4:
        c = config4(base=3, lmax=5, nv=24, nsteps=3, target_leaves=None, nboxes=6, side_scale=3.0)
        return c
    if config == 5:
        return config5(base=3, lmax=5, nv=24, nsteps=3)
    raise ValueError(config)


def window_leaves(case: Case, centre_leaf: int, rings: int, neighbours_of) -> np.ndarray:
    """Leaf ids within `rings` face-rings of `centre_leaf` (breadth-first over face neighbours)."""
    keep = {int(centre_leaf)}
    front = [int(centre_leaf)]
    for _ in range(rings):
        nxt = []
        for j in neighbours_of(front).tolist():
            if j not in keep:
                keep.add(j); nxt.append(j)
        front = nxt
        if not front:
            break
    return np.array(sorted(keep), dtype=np.int64)


def sub_case(case: Case, leaf_ids: np.ndarray, name: Optional[str] = None) -> Case:
    """The Case restricted to some leaves (a window of the mesh; the oracle takes it with window=True)."""
    import copy
    sub = copy.copy(case)
    sub.level, sub.ijk, sub.kind = case.level[leaf_ids].copy(), case.ijk[leaf_ids].copy(), case.kind[leaf_ids].copy()
    sub.prim0 = case.prim0[leaf_ids].copy()
    sub.fluid_moments = None if case.fluid_moments is None else case.fluid_moments[leaf_ids].copy()
    sub.name = name or (case.name + "_window")
    return sub


def morton_order(level: np.ndarray, ijk: np.ndarray) -> np.ndarray:
    """Leaf ids in N-order (Morton; reading G15: depth-first, child index x + 2y + 4z)."""
    level = np.asarray(level).astype(np.int64)
    lmax = int(level.max())
    xyz = np.asarray(ijk).astype(np.int64) << (lmax - level)[:, None]
    key = np.zeros(level.shape[0], np.int64)
    for b in range(lmax):
        for a in range(3):
            key |= ((xyz[:, a] >> b) & 1) << (3 * b + a)
    return np.argsort(key * 32 + level, kind="stable")


def with_body_of(old: Case, new: Case, name: Optional[str] = None) -> Case:
    """`new` with the solid body of `old`: every leaf of `new` that lies inside a SOLID leaf of `old` is SOLID (a mesh
    change does not move the body; a staircase body re-sampled on a finer mesh would otherwise uncover KINETIC leaves
    that have no old state to take over).  New SOLID leaves outside the old body are kept."""
    import copy
    solid = old.kind == CELL_SOLID
    keys = {(int(l), int(i), int(j), int(k)) for l, (i, j, k) in zip(old.level[solid], old.ijk[solid])}
    levels = sorted({k[0] for k in keys})
    out = copy.copy(new)
    out.kind = new.kind.copy()
    for lo in levels:
        m = new.level >= lo
        sh = (new.level[m].astype(np.int64) - lo)[:, None]
        anc = new.ijk[m].astype(np.int64) >> sh
        hit = np.fromiter(((lo, int(a), int(b), int(c)) in keys for a, b, c in anc), bool, count=anc.shape[0])
        idx = np.nonzero(m)[0][hit]
        out.kind[idx] = CELL_SOLID
    out.name = name or (new.name + "_body_of_" + old.name)
    return out


# ----------------------------------------------------------------------------------------------
# lattice-Boltzmann variant: problem statements only.  The lattice itself (velocities, weights) is
# textbook data both sides need to agree on what an index means; the equilibrium formula is NOT here (each side has its own).
# ----------------------------------------------------------------------------------------------
def lattice_velocities(q: int) -> np.ndarray:
    """c_i [Q,3] in {-1,0,1}^3 for D3Q27 (all 27) or D3Q19 (|c|^2 <= 2), in ascending canonical index
    (kz*3 + ky)*3 + kx with c = k - 1 -- the 3x3x3 velocity grid of the DVM solver."""
    assert q in (19, 27)
    k = np.arange(27)
    c = np.stack([k % 3 - 1, (k // 3) % 3 - 1, k // 9 - 1], axis=1)
    keep = (c ** 2).sum(axis=1) <= (2 if q == 19 else 3)
    return c[keep].astype(np.int64)


def lbm_case(tree: Case, lattice: int = 19, omega: float = 0.7, cfl: float = 0.4, nsteps: int = 5, mach: float = 0.1,
             storage: int = STORE_F64, noise_rel: float = 1e-3, seed: int = 0) -> Case:
    """An LBM problem on the mesh, boundary codes and solid leaves of `tree`: 3x3x3 velocity grid on [-1.5,1.5]^3 (nodes
    -1, 0, 1: lattice units, c_s^2 = 1/3), D3Q19 or D3Q27, relaxation time tau = dt / omega, initial state
    rho = 1 + 0.05 sin(2 pi x) cos(2 pi y), u = Ma c_s (cos 2 pi z, 0.5 sin 2 pi x, -0.3) (smooth, all components alive);
    INFLOW sides carry (rho, u) = (1, Ma c_s e_x).  FLUID leaves of the tree become KINETIC (the LBM has no mask)."""
    import copy
    c = copy.copy(tree)
    c.name = f"lbm_d3q{lattice}_{tree.name}"
    c.kind = np.where(tree.kind == CELL_SOLID, CELL_SOLID, CELL_KINETIC).astype(np.uint8)
    c.fluid_moments = None
    c.nv, c.vmin, c.vmax = (3, 3, 3), (-1.5,) * 3, (1.5,) * 3
    c.kn = float("inf")
    c.storage, c.cfl, c.nsteps = storage, cfl, nsteps
    x = c.centres()
    cs = 1.0 / np.sqrt(3.0)
    prim = np.zeros((c.n_leaves, 5))
    prim[:, 0] = 1 + 0.05 * np.sin(2 * np.pi * x[:, 0]) * np.cos(2 * np.pi * x[:, 1])
    prim[:, 1] = mach * cs * np.cos(2 * np.pi * x[:, 2])
    prim[:, 2] = 0.5 * mach * cs * np.sin(2 * np.pi * x[:, 0])
    prim[:, 3] = -0.3 * mach * cs
    prim[:, 4] = 1.0 / 3.0
    c.prim0 = prim
    c.inflow = np.zeros((6, 5)); c.inflow[:, 0] = 1.0; c.inflow[:, 1] = mach * cs; c.inflow[:, 4] = 1.0 / 3.0
    c.noise_rel, c.noise_seed = noise_rel, seed
    c.meta = dict(tree.meta, lattice=lattice, omega=omega)
    return c


def lbm_tau(case: Case) -> float:
    """Relaxation time of an lbm_case: dt / omega."""
    return case.dt / case.meta["omega"]
