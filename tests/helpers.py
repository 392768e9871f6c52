"""Test-side helpers that are independent of both the oracle and the CUDA path."""
import numpy as np

from paper_1503_00707_b200 import inputs


def brute_force_faces(level, ijk, periodic, live=None):
    """All leaf pairs whose boxes touch on one axis with positive overlap on the other two
    (periodic images included).  Returns a sorted list of (low cell, high cell, axis, area) with
    area in units of the cube face (L = 1).  O(n^2), tiny trees only."""
    level = np.asarray(level).astype(np.int64); ijk = np.asarray(ijk).astype(np.int64)
    lmax = int(level.max()); N = 1 << lmax
    size = (1 << (lmax - level))
    lo = ijk * size[:, None]; hi = lo + size[:, None]
    n = level.shape[0]
    out = []
    for a in range(3):
        b1, b2 = (a + 1) % 3, (a + 2) % 3
        touch = hi[:, None, a] == lo[None, :, a]
        if periodic[a]:
            touch |= (hi[:, None, a] == N) & (lo[None, :, a] == 0)
        o1 = np.minimum(hi[:, None, b1], hi[None, :, b1]) - np.maximum(lo[:, None, b1], lo[None, :, b1])
        o2 = np.minimum(hi[:, None, b2], hi[None, :, b2]) - np.maximum(lo[:, None, b2], lo[None, :, b2])
        ok = touch & (o1 > 0) & (o2 > 0)
        if live is not None:
            ok &= live[:, None] & live[None, :]
        p, q = np.nonzero(ok)
        area = (o1[p, q] * o2[p, q]).astype(np.float64) / float(N) ** 2
        out += [(int(pp), int(qq), a, float(ar)) for pp, qq, ar in zip(p, q, area)]
    return sorted(out)


def random_tree(rng, base, lmax, periodic, p_split=0.25):
    split = {}
    for l in range(base, lmax):
        split[l] = rng.uniform(size=(2 ** l,) * 3) < p_split
    return inputs.build_tree(base, lmax, split, periodic)


def periodic_case(level, ijk, nv=(6, 6, 6), vlim=4.0, kn=0.1, bc=None, kind=None, **kw):
    n = level.shape[0]
    prim = np.zeros((n, 5)); prim[:, 0] = 1; prim[:, 4] = 1
    c = inputs._case("t", level, ijk, np.zeros(n, np.uint8) if kind is None else kind,
                     bc or (inputs.BC_PERIODIC,) * 6, nv[0], vlim, kn, inputs.STORE_F64, 0.4, 1, prim, **kw)
    c.nv = tuple(nv)
    return c


def rel_linf(a, b):
    """max|a-b| / max|b|."""
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / np.abs(np.asarray(b)).max())


def xi_grids(case):
    xs, ys, zs = (case.xi_nodes(a) for a in range(3))
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    return X.ravel(), Y.ravel(), Z.ravel()


def np_moments(case, f):
    """w * sum m f, rows x (n, n ux, n uy, n uz, sum xi^2 f) -- numpy re-statement for the tests."""
    X, Y, Z = xi_grids(case)
    w = np.prod([(case.vmax[a] - case.vmin[a]) / case.nv[a] for a in range(3)])
    m = np.stack([np.ones_like(X), X, Y, Z, X * X + Y * Y + Z * Z])
    return w * (f @ m.T)


def moment_scales(m_ref, eps_storage=2.3e-16):
    """Denominators of the relative L-infinity error (G17) of the five moment fields [5, n].  The three momentum
    components are one vector field: they are scaled by the largest norm of the momentum vector.  Only a momentum
    field that is zero to round-off (no larger than 1e3 storage roundings of n * sqrt(R T0)) falls back to max n."""
    m_ref = np.asarray(m_ref)
    n_max = float(np.abs(m_ref[0]).max())
    p_max = float(np.sqrt((m_ref[1:4] ** 2).sum(axis=0)).max())
    if p_max <= 1e3 * eps_storage * n_max:
        p_max = n_max
    return [n_max, p_max, p_max, p_max, float(np.abs(m_ref[4]).max())]


def assert_moments_close(m_gpu, m_ref, tol, eps_storage=2.3e-16, what=""):
    scales = moment_scales(m_ref, eps_storage)
    for a in range(5):
        err = float(np.abs(np.asarray(m_gpu[a]) - np.asarray(m_ref[a])).max()) / scales[a]
        assert err <= tol, f"{what} moment {a}: {err:.3e} > {tol:g}"


def gpu_field_error(st, f_ref, chunk_slabs=2048):
    """max|f_gpu - f_ref| and max|f_ref| over the whole field, read from the device slab chunk by slab chunk
    (f_ref rows are Case kinetic rows, canonical velocity order)."""
    dmax = rmax = 0.0
    for s0 in range(0, st.n_kinetic, chunk_slabs):
        slabs = np.arange(s0, min(s0 + chunk_slabs, st.n_kinetic))
        got = st.read_canonical(slabs)
        ref = f_ref[st.row_of_slab[slabs]]
        assert np.all(np.isfinite(got))
        dmax = max(dmax, float(np.abs(got - ref).max()))
        rmax = max(rmax, float(np.abs(ref).max()))
    return dmax, rmax
