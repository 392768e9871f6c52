"""ctypes wrapper of oracle/dvm_oracle.c.  TEST INFRASTRUCTURE ONLY (see the header of the C file).

Rows of every f / moments array are the KINETIC leaves in leaf-list order; velocities are in
canonical order (kz*nvy + ky)*nvx + kx.  Nothing here imports the CUDA package except the shared,
arithmetic-free input description (`Case`)."""
import ctypes as C

import numpy as np

from . import build as _build


class _Desc(C.Structure):
    _fields_ = [("n_leaves", C.c_int64), ("level", C.c_void_p), ("ijk", C.c_void_p), ("kind", C.c_void_p),
                ("domain_len", C.c_double), ("bc", C.c_int32 * 6), ("inflow", (C.c_double * 5) * 6),
                ("fluid_moments", C.c_void_p), ("nv", C.c_int32 * 3), ("vmin", C.c_double * 3),
                ("vmax", C.c_double * 3), ("kn", C.c_double), ("visc_exp", C.c_double),
                ("nu_prefactor", C.c_double), ("window", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_dvm_create.argtypes = [C.POINTER(_Desc), C.POINTER(C.c_void_p)]
        L.oracle_dvm_destroy.argtypes = [C.c_void_p]
        L.oracle_dvm_error.argtypes = [C.c_void_p]; L.oracle_dvm_error.restype = C.c_char_p
        L.oracle_dvm_n_kinetic.argtypes = [C.c_void_p]; L.oracle_dvm_n_kinetic.restype = C.c_int64
        for name in ("oracle_dvm_transport", "oracle_dvm_relax", "oracle_dvm_step"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
        L.oracle_dvm_moments.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_dvm_newton.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_dvm_newton_max_iters.argtypes = [C.c_void_p]
        L.oracle_dvm_faces.argtypes = [C.c_void_p] + [C.c_void_p] * 5; L.oracle_dvm_faces.restype = C.c_int64
        L.oracle_dvm_boundary_counts.argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_dvm_leaf_neighbours.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        L.oracle_dvm_kinetic_leaves.argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_dvm_remap.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_dvm_set_threads.argtypes = [C.c_int]
        L.oracle_dvm_set_inflow_table.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"oracle error {code}: {msg}")
        self.code = code


class Oracle:
    """One mesh + velocity grid + gas model; steps f on the host in fp64."""

    def __init__(self, case, kn=None, window=False):
        L = lib()
        d = _Desc()
        self._keep = [np.ascontiguousarray(case.level, np.uint8), np.ascontiguousarray(case.ijk, np.uint32),
                      np.ascontiguousarray(case.kind, np.uint8)]
        d.n_leaves = case.n_leaves
        d.level, d.ijk, d.kind = (a.ctypes.data for a in self._keep)
        d.domain_len = case.domain_len
        d.bc[:] = list(case.bc)
        for s in range(6):
            d.inflow[s][:] = [float(x) for x in case.inflow[s]]
        if case.fluid_moments is not None:
            fm = np.ascontiguousarray(case.fluid_moments, np.float64); self._keep.append(fm)
            d.fluid_moments = fm.ctypes.data
        d.nv[:] = list(case.nv); d.vmin[:] = list(case.vmin); d.vmax[:] = list(case.vmax)
        d.kn = case.kn if kn is None else kn
        d.visc_exp, d.nu_prefactor = case.visc_exp, case.nu_prefactor
        d.window = 1 if window else 0
        self._h = C.c_void_p()
        rc = L.oracle_dvm_create(C.byref(d), C.byref(self._h))
        if rc != 0:
            msg = L.oracle_dvm_error(self._h).decode() if self._h else ""
            L.oracle_dvm_destroy(self._h); self._h = None
            raise OracleError(rc, msg)
        self.n_kinetic = int(L.oracle_dvm_n_kinetic(self._h))
        self.Nv = case.Nv

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle_dvm_destroy(self._h); self._h = None

    def _run(self, fn, f, dt):
        f = np.ascontiguousarray(f, np.float64)
        assert f.shape == (self.n_kinetic, self.Nv), f.shape
        out = np.empty_like(f)
        rc = fn(self._h, f.ctypes.data, out.ctypes.data, float(dt))
        if rc != 0:
            raise OracleError(rc, "Newton failed" if rc == -5 else "")
        return out

    def set_inflow_table(self, side, values):
        """Ghost state of INFLOW side `side` given as a table [Nv] (canonical velocity order) instead of a Maxwellian."""
        v = np.ascontiguousarray(values, np.float64)
        assert v.shape == (self.Nv,)
        rc = lib().oracle_dvm_set_inflow_table(self._h, int(side), v.ctypes.data)
        assert rc == 0

    def transport(self, f, dt):
        return self._run(lib().oracle_dvm_transport, f, dt)

    def relax(self, fstar, dt):
        return self._run(lib().oracle_dvm_relax, fstar, dt)

    def step(self, f, dt, nsteps=1):
        for _ in range(nsteps):
            f = self._run(lib().oracle_dvm_step, f, dt)
        return f

    def moments(self, f):
        f = np.ascontiguousarray(f, np.float64)
        mom = np.empty((5, self.n_kinetic))
        lib().oracle_dvm_moments(self._h, f.ctypes.data, mom.ctypes.data)
        return mom

    def newton(self, rho):
        rho = np.ascontiguousarray(rho, np.float64); alpha = np.empty(5)
        it = lib().oracle_dvm_newton(self._h, rho.ctypes.data, alpha.ctypes.data)
        return alpha, it

    @property
    def newton_max_iters(self):
        return int(lib().oracle_dvm_newton_max_iters(self._h))

    def faces(self):
        L = lib()
        n = int(L.oracle_dvm_faces(self._h, None, None, None, None, None))
        owner = np.empty(n, np.int64); neigh = np.empty(n, np.int64); area = np.empty(n)
        axis = np.empty(n, np.int8); ratio = np.empty(n, np.int8)
        L.oracle_dvm_faces(self._h, owner.ctypes.data, neigh.ctypes.data, area.ctypes.data, axis.ctypes.data, ratio.ctypes.data)
        return owner, neigh, area, axis, ratio

    def boundary_counts(self):
        c = np.zeros(5, np.int64)
        lib().oracle_dvm_boundary_counts(self._h, c.ctypes.data)
        return {"specular": int(c[1]), "inflow": int(c[2]), "outflow": int(c[3]), "solid": int(c[4])}

    def leaf_neighbours(self, leaves):
        out = []
        buf = np.empty(24, np.int64)
        for j in np.asarray(leaves).ravel().tolist():
            k = lib().oracle_dvm_leaf_neighbours(self._h, int(j), buf.ctypes.data)
            out.extend(buf[:k].tolist())
        return np.array(out, dtype=np.int64)

    def remap_from(self, old: "Oracle", f_old):
        """f on this mesh from f on `old` (volume average of the old piecewise-constant field, reading G20)."""
        f_old = np.ascontiguousarray(f_old, np.float64)
        assert f_old.shape == (old.n_kinetic, old.Nv)
        out = np.empty((self.n_kinetic, self.Nv))
        rc = lib().oracle_dvm_remap(old._h, self._h, f_old.ctypes.data, out.ctypes.data)
        if rc != 0:
            raise OracleError(rc, "remap: a new kinetic leaf lies over a SOLID leaf or outside the old mesh")
        return out

    def kinetic_leaves(self):
        a = np.empty(self.n_kinetic, np.int64)
        lib().oracle_dvm_kinetic_leaves(self._h, a.ctypes.data)
        return a


def threads():
    return int(lib().oracle_dvm_threads())


def set_threads(n: int):
    """OpenMP threads of the following oracle calls (bench.py times the oracle with 1 thread and with all cores)."""
    lib().oracle_dvm_set_threads(int(n))
