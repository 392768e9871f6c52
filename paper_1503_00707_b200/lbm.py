"""ctypes binding of include/ufs_lbm.h (same names, argument marshalling only) and a small holder of the device tensors.
The lattice-Boltzmann variant of the kinetic step; no CPU fallback."""
import ctypes as C
from typing import Optional

import numpy as np

from . import binding as B
from .inputs import STORE_F32, Case, lbm_tau

EXPORTS = ["ufs_lbm_create", "ufs_lbm_create_host", "ufs_lbm_step", "ufs_lbm_moments", "ufs_lbm_sync", "ufs_lbm_destroy",
           "ufs_lbm_current", "ufs_lbm_layout", "ufs_lbm_launch_count", "ufs_lbm_last_error"]


class ufs_lbm_desc(C.Structure):
    _fields_ = [("n_leaves", C.c_int64), ("level", C.c_void_p), ("ijk", C.c_void_p), ("kind", C.c_void_p),
                ("domain_len", C.c_double), ("bc", C.c_int32 * 6), ("inflow", (C.c_double * 4) * 6),
                ("lattice", C.c_int32), ("tau", C.c_double), ("storage", C.c_int32)]


_ready = False


def lib() -> C.CDLL:
    global _ready
    L = B.lib()
    if not _ready:
        vp = C.c_void_p
        L.ufs_lbm_create.argtypes = [C.POINTER(ufs_lbm_desc), C.POINTER(C.c_void_p), vp, C.POINTER(C.c_void_p)]
        L.ufs_lbm_create_host.argtypes = [C.POINTER(ufs_lbm_desc), C.POINTER(C.c_void_p)]
        L.ufs_lbm_step.argtypes = [vp, C.c_double, C.c_int]
        L.ufs_lbm_moments.argtypes = [vp, vp]
        for name in ("ufs_lbm_sync", "ufs_lbm_destroy", "ufs_lbm_current"):
            getattr(L, name).argtypes = [vp]
        L.ufs_lbm_layout.argtypes = [vp, C.POINTER(C.c_int64), vp, C.POINTER(C.c_int32), vp, vp]
        L.ufs_lbm_launch_count.argtypes = [vp]; L.ufs_lbm_launch_count.restype = C.c_int64
        L.ufs_lbm_last_error.argtypes = [vp]; L.ufs_lbm_last_error.restype = C.c_char_p
        _ready = True
    return L


def make_desc(case: Case, tau: Optional[float] = None, storage: Optional[int] = None):
    keep = [np.ascontiguousarray(case.level, np.uint8), np.ascontiguousarray(case.ijk, np.uint32),
            np.ascontiguousarray(case.kind, np.uint8)]
    d = ufs_lbm_desc()
    d.n_leaves = case.n_leaves
    d.level, d.ijk, d.kind = (a.ctypes.data for a in keep)
    d.domain_len = case.domain_len
    d.bc[:] = list(case.bc)
    for s in range(6):
        d.inflow[s][:] = [float(x) for x in case.inflow[s][:4]]
    d.lattice = int(case.meta["lattice"])
    d.tau = lbm_tau(case) if tau is None else tau
    d.storage = case.storage if storage is None else storage
    return d, keep


def _check(h, rc):
    if rc != B.OK:
        raise B.UfsDvmError(rc, lib().ufs_lbm_last_error(h).decode() if h else "")


def _created(rc, h):
    if rc != B.OK:
        msg = lib().ufs_lbm_last_error(h).decode() if h else ""
        lib().ufs_lbm_destroy(h)
        raise B.UfsDvmError(rc, msg)
    return h


def ufs_lbm_create_host(desc):
    h = C.c_void_p()
    return _created(lib().ufs_lbm_create_host(C.byref(desc), C.byref(h)), h)


def ufs_lbm_create(desc, f_dev_ptrs, cuda_stream: int = 0):
    h = C.c_void_p()
    arr = (C.c_void_p * 2)(f_dev_ptrs[0], f_dev_ptrs[1])
    return _created(lib().ufs_lbm_create(C.byref(desc), arr, C.c_void_p(cuda_stream), C.byref(h)), h)


def ufs_lbm_step(h, dt, nsteps=1):
    _check(h, lib().ufs_lbm_step(h, float(dt), int(nsteps)))


def ufs_lbm_moments(h, mom_dev_ptr):
    _check(h, lib().ufs_lbm_moments(h, C.c_void_p(mom_dev_ptr)))


def ufs_lbm_sync(h):
    _check(h, lib().ufs_lbm_sync(h))


def ufs_lbm_destroy(h):
    lib().ufs_lbm_destroy(h)


def ufs_lbm_current(h) -> int:
    return int(lib().ufs_lbm_current(h))


def ufs_lbm_launch_count(h) -> int:
    return int(lib().ufs_lbm_launch_count(h))


def ufs_lbm_layout(h):
    n, q = C.c_int64(), C.c_int32()
    _check(h, lib().ufs_lbm_layout(h, C.byref(n), None, C.byref(q), None, None))
    cell = np.empty(n.value, np.int64); c = np.empty((q.value, 3), np.int8); w = np.empty(q.value)
    _check(h, lib().ufs_lbm_layout(h, None, cell.ctypes.data, None, c.ctypes.data, w.ctypes.data))
    return int(n.value), cell, int(q.value), c, w


class LbmStepper:
    """Owns the two f tensors [Q, n_cells] (velocity-major, the library's layout) and the moments tensor (PyTorch, on `device`) and the library handle.
    Canonical rows are the case's non-SOLID leaves in ascending leaf order, columns the lattice velocities in the
    library's column order (= inputs.lattice_velocities)."""

    def __init__(self, case: Case, device="cuda:0", tau: Optional[float] = None, storage: Optional[int] = None, stream=None):
        import torch
        self.torch = torch
        self.storage = case.storage if storage is None else storage
        self.dtype = torch.float32 if self.storage == STORE_F32 else torch.float64
        self.device = torch.device(device)
        desc, self._keep = make_desc(case, tau=tau, storage=self.storage)
        self.q = int(case.meta["lattice"])
        kin = case.kinetic_leaves()
        with torch.cuda.device(self.device):
            self.f = [torch.empty((self.q, kin.size), dtype=self.dtype, device=self.device) for _ in range(2)]
            self.mom = torch.empty((4, max(kin.size, 1)), dtype=torch.float64, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.h = ufs_lbm_create(desc, [t.data_ptr() for t in self.f], self.stream.cuda_stream)
        self.n_cells, self.cell_of_row, q, self.c, self.w = ufs_lbm_layout(self.h)
        assert self.n_cells == kin.size and q == self.q
        row_of_leaf = np.full(case.n_leaves, -1, np.int64); row_of_leaf[kin] = np.arange(kin.size)
        self.case_row = row_of_leaf[self.cell_of_row]          # library row -> canonical row

    def load_canonical(self, f_rows: np.ndarray):
        torch = self.torch
        assert f_rows.shape == (self.n_cells, self.q)
        with torch.cuda.stream(self.stream):
            self.f[ufs_lbm_current(self.h)].copy_(torch.from_numpy(np.ascontiguousarray(f_rows[self.case_row].T)).to(self.device).to(self.dtype))

    def read_canonical(self) -> np.ndarray:
        with self.torch.cuda.stream(self.stream):
            got = self.f[ufs_lbm_current(self.h)].double().cpu().numpy().T
        out = np.empty_like(got)
        out[self.case_row] = got
        return out

    def step(self, dt, nsteps=1):
        ufs_lbm_step(self.h, dt, nsteps)

    def moments(self) -> np.ndarray:
        ufs_lbm_moments(self.h, self.mom.data_ptr())
        ufs_lbm_sync(self.h)
        m = self.mom.cpu().numpy()[:, :self.n_cells]
        out = np.empty_like(m)
        out[:, self.case_row] = m
        return out

    def sync(self):
        ufs_lbm_sync(self.h)

    def close(self):
        if getattr(self, "h", None) is not None:
            ufs_lbm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
