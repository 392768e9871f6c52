"""Thin Python binding of libufs_dvm.so (include/ufs_dvm.h): same names, argument marshalling only.

Every step of the DVM path runs in the library's CUDA kernels; PyTorch is used here for device
memory and streams.  There is no CPU fallback: if the library cannot be built or loaded, importing
this module's functions raises.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build
from .inputs import STORE_F32, Case

OK, EINVAL, EMESH, ECUDA, ENOMEM, ENEWTON = 0, -1, -2, -3, -4, -5
_CODES = {EINVAL: "EINVAL", EMESH: "EMESH", ECUDA: "ECUDA", ENOMEM: "ENOMEM", ENEWTON: "ENEWTON"}

EXPORTS = ["ufs_dvm_create", "ufs_dvm_create_host", "ufs_dvm_step", "ufs_dvm_moments", "ufs_dvm_sync",
           "ufs_dvm_destroy", "ufs_dvm_current", "ufs_dvm_layout", "ufs_dvm_faces", "ufs_dvm_boundary_faces",
           "ufs_dvm_run_host", "ufs_dvm_launch_count", "ufs_dvm_kernel_info", "ufs_dvm_kernel_name",
           "ufs_dvm_last_error", "ufs_dvm_f_changed", "ufs_dvm_profile", "ufs_dvm_kernel_ms", "ufs_dvm_tiles", "ufs_dvm_remesh", "ufs_dvm_remap_plan",
           "ufs_dvm_partition", "ufs_dvm_create_part", "ufs_dvm_create_part_host", "ufs_dvm_part_layout", "ufs_dvm_halo",
           "ufs_dvm_halo_bytes", "ufs_dvm_halo_pack", "ufs_dvm_halo_unpack", "ufs_dvm_halo_done", "ufs_dvm_moments_static",
           "ufs_dvm_halo_push_setup", "ufs_dvm_push_entries", "ufs_dvm_sums_dev", "ufs_dvm_sums_use"]

STATIC_MAX_CELLS = 8192   # UFS_DVM_STATIC_MAX_CELLS of include/ufs_dvm.h


class ufs_dvm_desc(C.Structure):
    _fields_ = [("n_leaves", C.c_int64), ("level", C.c_void_p), ("ijk", C.c_void_p), ("kind", C.c_void_p),
                ("domain_len", C.c_double), ("bc", C.c_int32 * 6), ("inflow", (C.c_double * 5) * 6),
                ("fluid_moments", C.c_void_p), ("nv", C.c_int32 * 3), ("vmin", C.c_double * 3),
                ("vmax", C.c_double * 3), ("kn", C.c_double), ("visc_exp", C.c_double),
                ("nu_prefactor", C.c_double), ("storage", C.c_int32)]


class UfsDvmError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ufs_dvm {_CODES.get(code, code)}: {msg}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Loads (building first if stale) the C-ABI library.  Fails loudly; nothing stands in for it."""
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, i64p = C.c_void_p, C.c_void_p
        L.ufs_dvm_create.argtypes = [C.POINTER(ufs_dvm_desc), C.POINTER(C.c_void_p), vp, C.POINTER(C.c_void_p)]
        L.ufs_dvm_create_host.argtypes = [C.POINTER(ufs_dvm_desc), C.POINTER(C.c_void_p)]
        L.ufs_dvm_step.argtypes = [vp, C.c_double, C.c_int]
        L.ufs_dvm_moments.argtypes = [vp, vp]
        L.ufs_dvm_moments_static.argtypes = [vp, vp, vp]
        L.ufs_dvm_sync.argtypes = [vp]
        L.ufs_dvm_destroy.argtypes = [vp]
        L.ufs_dvm_current.argtypes = [vp]
        L.ufs_dvm_f_changed.argtypes = [vp]
        L.ufs_dvm_profile.argtypes = [vp, C.c_int]
        L.ufs_dvm_kernel_ms.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        L.ufs_dvm_layout.argtypes = [vp, C.POINTER(C.c_int64), i64p, vp]
        L.ufs_dvm_faces.argtypes = [vp, C.POINTER(C.c_int64), vp, vp, vp, vp, vp]
        L.ufs_dvm_boundary_faces.argtypes = [vp, C.POINTER(C.c_int64), vp, vp, vp, vp, vp, vp]
        L.ufs_dvm_run_host.argtypes = [vp, vp, vp, vp, vp, C.c_double, C.c_int]
        L.ufs_dvm_remesh.argtypes = [vp, C.POINTER(ufs_dvm_desc), C.POINTER(C.c_void_p), vp, C.POINTER(C.c_void_p), vp]
        L.ufs_dvm_remap_plan.argtypes = [vp, vp, C.POINTER(C.c_int64), vp, vp, vp, C.POINTER(C.c_int64), vp]
        L.ufs_dvm_tiles.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int32), vp, vp, vp, C.POINTER(C.c_int64), vp]
        i32p = C.c_void_p
        L.ufs_dvm_partition.argtypes = [C.POINTER(ufs_dvm_desc), C.c_int32, C.c_double, C.c_double, i32p]
        L.ufs_dvm_create_part.argtypes = [C.POINTER(ufs_dvm_desc), i32p, C.c_int32, C.c_int32, C.POINTER(C.c_void_p), vp, C.POINTER(C.c_void_p)]
        L.ufs_dvm_create_part_host.argtypes = [C.POINTER(ufs_dvm_desc), i32p, C.c_int32, C.c_int32, C.POINTER(C.c_void_p)]
        L.ufs_dvm_part_layout.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64), vp, vp]
        L.ufs_dvm_halo.argtypes = [vp, C.c_int32, C.POINTER(C.c_int64), vp, vp, C.POINTER(C.c_int64), vp, vp]
        L.ufs_dvm_halo_bytes.argtypes = [vp, C.c_int32, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.ufs_dvm_halo_pack.argtypes = [vp, C.c_int32, vp]
        L.ufs_dvm_halo_unpack.argtypes = [vp, C.c_int32, vp]
        L.ufs_dvm_halo_done.argtypes = [vp]
        L.ufs_dvm_halo_push_setup.argtypes = [vp, vp, vp, vp, vp, vp]
        L.ufs_dvm_sums_dev.argtypes = [vp, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]
        L.ufs_dvm_sums_use.argtypes = [vp, vp, vp]
        L.ufs_dvm_push_entries.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), vp, vp, vp, vp, vp, vp]
        L.ufs_dvm_launch_count.argtypes = [vp]; L.ufs_dvm_launch_count.restype = C.c_int64
        L.ufs_dvm_kernel_info.argtypes = [vp] + [C.POINTER(C.c_int32)] * 4
        L.ufs_dvm_last_error.argtypes = [vp]; L.ufs_dvm_last_error.restype = C.c_char_p
        L.ufs_dvm_kernel_name.argtypes = [vp]; L.ufs_dvm_kernel_name.restype = C.c_char_p
        _lib = L
    return _lib


def make_desc(case: Case, kn: Optional[float] = None, storage: Optional[int] = None):
    """ufs_dvm_desc for a Case.  Returns (desc, keepalive list of the host arrays it points to)."""
    keep = [np.ascontiguousarray(case.level, np.uint8), np.ascontiguousarray(case.ijk, np.uint32),
            np.ascontiguousarray(case.kind, np.uint8)]
    d = ufs_dvm_desc()
    d.n_leaves = case.n_leaves
    d.level, d.ijk, d.kind = (a.ctypes.data for a in keep)
    d.domain_len = case.domain_len
    d.bc[:] = list(case.bc)
    for s in range(6):
        d.inflow[s][:] = [float(x) for x in case.inflow[s]]
    if case.fluid_moments is not None:
        fm = np.ascontiguousarray(case.fluid_moments, np.float64)
        keep.append(fm)
        d.fluid_moments = fm.ctypes.data
    d.nv[:] = list(case.nv); d.vmin[:] = list(case.vmin); d.vmax[:] = list(case.vmax)
    d.kn = case.kn if kn is None else kn
    d.visc_exp, d.nu_prefactor = case.visc_exp, case.nu_prefactor
    d.storage = case.storage if storage is None else storage
    return d, keep


def _check(h, rc):
    if rc != OK:
        msg = lib().ufs_dvm_last_error(h).decode() if h else ""
        raise UfsDvmError(rc, msg)


# ---- the C calls, same names ---------------------------------------------------------------------
def ufs_dvm_create_host(desc: ufs_dvm_desc) -> C.c_void_p:
    h = C.c_void_p()
    rc = lib().ufs_dvm_create_host(C.byref(desc), C.byref(h))
    if rc != OK:
        msg = lib().ufs_dvm_last_error(h).decode() if h else ""
        lib().ufs_dvm_destroy(h)
        raise UfsDvmError(rc, msg)
    return h


def ufs_dvm_create(desc: ufs_dvm_desc, f_dev_ptrs, cuda_stream: int = 0) -> C.c_void_p:
    h = C.c_void_p()
    arr = (C.c_void_p * 2)(f_dev_ptrs[0], f_dev_ptrs[1])
    rc = lib().ufs_dvm_create(C.byref(desc), arr, C.c_void_p(cuda_stream), C.byref(h))
    if rc != OK:
        msg = lib().ufs_dvm_last_error(h).decode() if h else ""
        lib().ufs_dvm_destroy(h)
        raise UfsDvmError(rc, msg)
    return h


def ufs_dvm_step(h, dt: float, nsteps: int = 1):
    _check(h, lib().ufs_dvm_step(h, float(dt), int(nsteps)))


def ufs_dvm_moments(h, mom_dev_ptr: int):
    _check(h, lib().ufs_dvm_moments(h, C.c_void_p(mom_dev_ptr)))


def ufs_dvm_moments_static(h, f_dev_ptr: Optional[int], mom_dev_ptr: int):
    _check(h, lib().ufs_dvm_moments_static(h, C.c_void_p(f_dev_ptr), C.c_void_p(mom_dev_ptr)))


def ufs_dvm_sync(h):
    _check(h, lib().ufs_dvm_sync(h))


def ufs_dvm_destroy(h):
    return lib().ufs_dvm_destroy(h)


def ufs_dvm_current(h) -> int:
    return int(lib().ufs_dvm_current(h))


def ufs_dvm_f_changed(h):
    _check(h, lib().ufs_dvm_f_changed(h))


def ufs_dvm_profile(h, enable: bool):
    _check(h, lib().ufs_dvm_profile(h, int(bool(enable))))


def ufs_dvm_kernel_ms(h):
    ms, n = C.c_double(0.0), C.c_int32(0)
    _check(h, lib().ufs_dvm_kernel_ms(h, C.byref(ms), C.byref(n)))
    return float(ms.value), int(n.value)


def ufs_dvm_layout(h, Nv: int):
    """(n_kinetic, cell_of_slab, vel_of_slot); Nv = nv[0]*nv[1]*nv[2] sizes the slot array."""
    n = C.c_int64()
    _check(h, lib().ufs_dvm_layout(h, C.byref(n), None, None))
    cell = np.empty(n.value, np.int64)
    vel = np.empty(int(Nv), np.int32)
    _check(h, lib().ufs_dvm_layout(h, C.byref(n), cell.ctypes.data, vel.ctypes.data))
    return int(n.value), cell, vel


def ufs_dvm_faces(h):
    n = C.c_int64()
    _check(h, lib().ufs_dvm_faces(h, C.byref(n), None, None, None, None, None))
    owner = np.empty(n.value, np.int64); neigh = np.empty(n.value, np.int64); area = np.empty(n.value)
    axis = np.empty(n.value, np.int8); ratio = np.empty(n.value, np.int8)
    _check(h, lib().ufs_dvm_faces(h, C.byref(n), owner.ctypes.data, neigh.ctypes.data, area.ctypes.data,
                                  axis.ctypes.data, ratio.ctypes.data))
    return owner, neigh, area, axis, ratio


def ufs_dvm_boundary_faces(h):
    n = C.c_int64()
    _check(h, lib().ufs_dvm_boundary_faces(h, C.byref(n), None, None, None, None, None, None))
    cell = np.empty(n.value, np.int64); axis = np.empty(n.value, np.int8); side = np.empty(n.value, np.int8)
    area = np.empty(n.value); kind = np.empty(n.value, np.int8); state = np.empty(n.value, np.int64)
    _check(h, lib().ufs_dvm_boundary_faces(h, C.byref(n), cell.ctypes.data, axis.ctypes.data, side.ctypes.data,
                                           area.ctypes.data, kind.ctypes.data, state.ctypes.data))
    return cell, axis, side, area, kind, state


def ufs_dvm_remesh(old_h, desc: ufs_dvm_desc, f_dev_ptrs, cuda_stream: int = 0):
    """(new handle, counts[4]: copied, refined, coarsened, from-fluid)."""
    h = C.c_void_p()
    arr = (C.c_void_p * 2)(f_dev_ptrs[0], f_dev_ptrs[1])
    counts = np.zeros(4, np.int64)
    rc = lib().ufs_dvm_remesh(old_h, C.byref(desc), arr, C.c_void_p(cuda_stream), C.byref(h), counts.ctypes.data)
    if rc != OK:
        msg = lib().ufs_dvm_last_error(h).decode() if h else ""
        lib().ufs_dvm_destroy(h)
        raise UfsDvmError(rc, msg)
    return h, counts


def ufs_dvm_remap_plan(old_h, new_h, n_new_kinetic: int):
    """(off, src, wgt, ghost_leaf) of the mesh-change map from old_h's mesh to new_h's (see include/ufs_dvm.h)."""
    n, ng = C.c_int64(), C.c_int64()
    _check(new_h, lib().ufs_dvm_remap_plan(old_h, new_h, C.byref(n), None, None, None, C.byref(ng), None))
    off = np.zeros(n_new_kinetic + 1, np.int64); src = np.zeros(n.value, np.int32); wgt = np.zeros(n.value)
    gl = np.zeros(ng.value, np.int64)
    _check(new_h, lib().ufs_dvm_remap_plan(old_h, new_h, C.byref(n), off.ctypes.data, src.ctypes.data, wgt.ctypes.data,
                                           C.byref(ng), gl.ctypes.data))
    return off, src, wgt, gl


def ufs_dvm_partition(desc: ufs_dvm_desc, n_ranks: int, w_kinetic: float = 1.0, w_fluid: float = 0.0) -> np.ndarray:
    """rank_of_leaf[n_leaves] int32."""
    out = np.empty(int(desc.n_leaves), np.int32)
    rc = lib().ufs_dvm_partition(C.byref(desc), int(n_ranks), float(w_kinetic), float(w_fluid), out.ctypes.data)
    if rc != OK:
        raise UfsDvmError(rc, "ufs_dvm_partition")
    return out


def _created(rc, h):
    if rc != OK:
        msg = lib().ufs_dvm_last_error(h).decode() if h else ""
        lib().ufs_dvm_destroy(h)
        raise UfsDvmError(rc, msg)
    return h


def ufs_dvm_create_part_host(desc: ufs_dvm_desc, rank_of_leaf: np.ndarray, my_rank: int, n_ranks: int) -> C.c_void_p:
    h = C.c_void_p()
    rol = np.ascontiguousarray(rank_of_leaf, np.int32)
    return _created(lib().ufs_dvm_create_part_host(C.byref(desc), rol.ctypes.data, int(my_rank), int(n_ranks), C.byref(h)), h)


def ufs_dvm_create_part(desc: ufs_dvm_desc, rank_of_leaf: np.ndarray, my_rank: int, n_ranks: int, f_dev_ptrs,
                        cuda_stream: int = 0) -> C.c_void_p:
    h = C.c_void_p()
    rol = np.ascontiguousarray(rank_of_leaf, np.int32)
    arr = (C.c_void_p * 2)(f_dev_ptrs[0], f_dev_ptrs[1])
    return _created(lib().ufs_dvm_create_part(C.byref(desc), rol.ctypes.data, int(my_rank), int(n_ranks), arr,
                                              C.c_void_p(cuda_stream), C.byref(h)), h)


def ufs_dvm_part_layout(h) -> dict:
    n_in, n_gh, g0 = C.c_int64(), C.c_int64(), C.c_int64()
    _check(h, lib().ufs_dvm_part_layout(h, C.byref(n_in), C.byref(n_gh), C.byref(g0), None, None))
    leaf = np.empty(n_in.value + n_gh.value, np.int64)
    owner = np.empty(n_gh.value, np.int32)
    _check(h, lib().ufs_dvm_part_layout(h, None, None, None, leaf.ctypes.data, owner.ctypes.data))
    return {"n_inner": n_in.value, "n_ghost": n_gh.value, "first_global_slab": g0.value, "leaf_of_slab": leaf,
            "owner_of_ghost": owner}


def ufs_dvm_halo(h, peer: int) -> dict:
    ns, nr = C.c_int64(), C.c_int64()
    _check(h, lib().ufs_dvm_halo(h, int(peer), C.byref(ns), None, None, C.byref(nr), None, None))
    ss, sm = np.empty(ns.value, np.int32), np.empty(ns.value, np.uint8)
    rs, rm = np.empty(nr.value, np.int32), np.empty(nr.value, np.uint8)
    _check(h, lib().ufs_dvm_halo(h, int(peer), None, ss.ctypes.data, sm.ctypes.data, None, rs.ctypes.data, rm.ctypes.data))
    return {"send_slab": ss, "send_mask": sm, "recv_slab": rs, "recv_mask": rm}


def ufs_dvm_halo_bytes(h, peer: int):
    sb, rb = C.c_int64(), C.c_int64()
    _check(h, lib().ufs_dvm_halo_bytes(h, int(peer), C.byref(sb), C.byref(rb)))
    return sb.value, rb.value


def ufs_dvm_halo_pack(h, peer: int, buf_dev_ptr: int):
    _check(h, lib().ufs_dvm_halo_pack(h, int(peer), C.c_void_p(buf_dev_ptr)))


def ufs_dvm_halo_unpack(h, peer: int, buf_dev_ptr: int):
    _check(h, lib().ufs_dvm_halo_unpack(h, int(peer), C.c_void_p(buf_dev_ptr)))


def ufs_dvm_halo_done(h):
    _check(h, lib().ufs_dvm_halo_done(h))


def ufs_dvm_halo_push_setup(h, peer_f0, peer_f1, dest_slab, peer_sums0=None, peer_sums1=None):
    """peer_f0 / peer_f1: per rank the device address of that rank's f buffers (None for ranks that need nothing from this
    one); dest_slab: per rank an int32 array (or None); peer_sums0 / peer_sums1: per rank the addresses ufs_dvm_sums_dev
    returns on that rank (both or neither)."""
    n = len(peer_f0)
    keep = [None if d is None else np.ascontiguousarray(d, np.int32) for d in dest_slab]
    arr = lambda xs: None if xs is None else (C.c_void_p * n)(*[C.c_void_p(x) for x in xs])
    ad = (C.c_void_p * n)(*[C.c_void_p(None if d is None else d.ctypes.data) for d in keep])
    _check(h, lib().ufs_dvm_halo_push_setup(h, arr(peer_f0), arr(peer_f1), ad, arr(peer_sums0), arr(peer_sums1)))


def ufs_dvm_sums_use(h, sums0_ptr: int, sums1_ptr: int):
    _check(h, lib().ufs_dvm_sums_use(h, C.c_void_p(sums0_ptr), C.c_void_p(sums1_ptr)))


def ufs_dvm_sums_dev(h):
    s0, s1 = C.c_void_p(), C.c_void_p()
    _check(h, lib().ufs_dvm_sums_dev(h, C.byref(s0), C.byref(s1)))
    return s0.value, s1.value


def ufs_dvm_push_entries(h) -> dict:
    n, nt = C.c_int64(), C.c_int64()
    _check(h, lib().ufs_dvm_push_entries(h, C.byref(n), C.byref(nt), None, None, None, None, None, None))
    slab, mask = np.empty(n.value, np.int32), np.empty(n.value, np.uint8)
    d0, d1, s0, s1 = (np.empty(n.value, np.uint64) for _ in range(4))
    _check(h, lib().ufs_dvm_push_entries(h, None, None, slab.ctypes.data, mask.ctypes.data, d0.ctypes.data, d1.ctypes.data,
                                         s0.ctypes.data, s1.ctypes.data))
    return {"n_push_tiles": int(nt.value), "slab": slab, "mask": mask, "dst0": d0, "dst1": d1, "sums0": s0, "sums1": s1}


def ufs_dvm_tiles(h) -> dict:
    """The flattener's tile records (see include/ufs_dvm.h); empty arrays if the handle uses another kernel."""
    n, pmax, ng = C.c_int64(), C.c_int32(), C.c_int64()
    _check(h, lib().ufs_dvm_tiles(h, C.byref(n), C.byref(pmax), None, None, None, C.byref(ng), None))
    nt, pm = int(n.value), int(pmax.value)
    hdr = np.zeros((nt, 8), np.int32); pieces = np.zeros((nt, 8, max(pm, 1)), np.uint32)
    cellidx = np.zeros((nt, 8, 8, 16), np.uint8)
    fluid_leaf = np.zeros(int(ng.value), np.int64)
    _check(h, lib().ufs_dvm_tiles(h, C.byref(n), C.byref(pmax), hdr.ctypes.data, pieces.ctypes.data if pm else None,
                                  cellidx.ctypes.data, C.byref(ng), fluid_leaf.ctypes.data))
    return {"n_tiles": nt, "pmax": pm, "s0": hdr[:, 0].copy(), "nc": hdr[:, 1].copy(),
            "np": hdr[:, 2:4].copy().view(np.uint8).reshape(nt, 8), "level": hdr[:, 4:6].copy().view(np.uint8).reshape(nt, 8),
            "pieces": pieces, "cellidx": cellidx, "fluid_leaf": fluid_leaf,
            "push_first": hdr[:, 6].copy(), "push_counts": hdr[:, 7].copy().view(np.uint32)}


def ufs_dvm_run_host(h, f_host_in_ptr: int, f_host_out_ptr: Optional[int], mom_dev_ptr: int, mom_host_ptr: int,
                     dt: float, nsteps: int):
    _check(h, lib().ufs_dvm_run_host(h, C.c_void_p(f_host_in_ptr), C.c_void_p(f_host_out_ptr or 0),
                                     C.c_void_p(mom_dev_ptr), C.c_void_p(mom_host_ptr), float(dt), int(nsteps)))


def ufs_dvm_launch_count(h) -> int:
    return int(lib().ufs_dvm_launch_count(h))


def ufs_dvm_kernel_info(h) -> dict:
    t, s, v, f = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
    _check(h, lib().ufs_dvm_kernel_info(h, C.byref(t), C.byref(s), C.byref(v), C.byref(f)))
    return {"threads": t.value, "smem_bytes": s.value, "vec": v.value, "fast": bool(f.value)}


def ufs_dvm_kernel_name(h) -> str:
    return lib().ufs_dvm_kernel_name(h).decode()


def ufs_dvm_last_error(h) -> str:
    return lib().ufs_dvm_last_error(h).decode()


# ---- a small holder: device tensors + handle (memory and streams only) ----------------------------
class DvmStepper:
    """Owns the two f tensors and the moments tensor (PyTorch, on `device`) and the library handle.

    f_rows given to / returned by load_canonical / read_canonical are [n_kinetic, Nv] with rows in
    kinetic-leaf order of the Case and velocities in canonical order; the permutation to and from the
    library's slab / slot order (ufs_dvm_layout) is applied here, on the host, with numpy."""

    def __init__(self, case: Case, device="cuda:0", kn: Optional[float] = None, storage: Optional[int] = None,
                 stream=None, remesh_from: Optional["DvmStepper"] = None):
        """With `remesh_from`, the handle is made by ufs_dvm_remesh: f starts as the old stepper's current f carried
        over to this case's mesh on the device (self.remesh_counts: copied, refined, coarsened, from-fluid)."""
        import torch
        self.torch = torch
        self.case = case
        self.storage = case.storage if storage is None else storage
        self.dtype = torch.float32 if self.storage == STORE_F32 else torch.float64
        self.device = torch.device(device)
        desc, self._keep = make_desc(case, kn=kn, storage=self.storage)
        n_kin = int((case.kind == 0).sum())
        self.Nv = case.Nv
        with torch.cuda.device(self.device):
            self.f = [torch.empty((n_kin, self.Nv), dtype=self.dtype, device=self.device) for _ in range(2)]
            self.mom = torch.empty((5, n_kin), dtype=torch.float64, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            if remesh_from is None:
                self.h = ufs_dvm_create(desc, [t.data_ptr() for t in self.f], self.stream.cuda_stream)
            else:
                self.h, self.remesh_counts = ufs_dvm_remesh(remesh_from.h, desc, [t.data_ptr() for t in self.f],
                                                            self.stream.cuda_stream)
        self.n_kinetic, self.cell_of_slab, self.vel_of_slot = ufs_dvm_layout(self.h, self.Nv)
        assert self.n_kinetic == n_kin
        kin = case.kinetic_leaves()
        row_of_leaf = np.full(case.n_leaves, -1, np.int64)
        row_of_leaf[kin] = np.arange(kin.size)
        self.row_of_slab = row_of_leaf[self.cell_of_slab]          # slab -> kinetic row of the Case

    # -- marshalling between canonical host arrays and the device layout
    def load_canonical(self, f_rows: np.ndarray):
        torch = self.torch
        f_rows = np.asarray(f_rows)
        assert f_rows.shape == (self.n_kinetic, self.Nv)
        cur = ufs_dvm_current(self.h)
        chunk = max(1, (1 << 28) // (self.Nv * 8))
        slot_t = torch.as_tensor(self.vel_of_slot.astype(np.int64), device=self.device)
        with torch.cuda.stream(self.stream):     # the copies must be ordered with the handle's stream
            for s0 in range(0, self.n_kinetic, chunk):
                s1 = min(s0 + chunk, self.n_kinetic)       # (a partitioned handle's tensors hold ghost slabs after these)
                rows = self.row_of_slab[s0:s1]
                part = torch.from_numpy(np.ascontiguousarray(f_rows[rows])).to(self.device)
                self.f[cur][s0:s1].copy_(part.index_select(1, slot_t).to(self.dtype))
        ufs_dvm_f_changed(self.h)

    def read_canonical(self, slabs: Optional[np.ndarray] = None) -> np.ndarray:
        """Current f as float64 [rows, Nv] in canonical velocity order.  With `slabs`, only those slabs, in the
        order given (rows are then slabs, not Case rows).  The slot permutation is applied on the device."""
        torch = self.torch
        cur = ufs_dvm_current(self.h)
        inv = np.empty(self.Nv, np.int64); inv[self.vel_of_slot] = np.arange(self.Nv)
        inv_t = torch.as_tensor(inv, device=self.device)
        chunk = max(1, (1 << 28) // (self.Nv * 8))
        with torch.cuda.stream(self.stream):
            if slabs is not None:
                slabs = np.asarray(slabs, np.int64)
                out = np.empty((slabs.size, self.Nv))
                for s0 in range(0, slabs.size, chunk):
                    idx = torch.as_tensor(slabs[s0:s0 + chunk], device=self.device)
                    out[s0:s0 + chunk] = self.f[cur].index_select(0, idx).index_select(1, inv_t).double().cpu().numpy()
                return out
            out = np.empty((self.n_kinetic, self.Nv))
            for s0 in range(0, self.n_kinetic, chunk):
                s1 = min(s0 + chunk, self.n_kinetic)
                part = self.f[cur][s0:s1].index_select(1, inv_t).double().cpu().numpy()
                out[self.row_of_slab[s0:s1]] = part
        return out

    def step(self, dt: float, nsteps: int = 1):
        ufs_dvm_step(self.h, dt, nsteps)

    def moments(self) -> np.ndarray:
        """[5, n_kinetic] in Case row order: n, n ux, n uy, n uz, E."""
        ufs_dvm_moments(self.h, self.mom.data_ptr())
        ufs_dvm_sync(self.h)
        m = self.mom.cpu().numpy()
        out = np.empty_like(m)
        out[:, self.row_of_slab] = m
        return out

    def moments_static(self, f=None) -> np.ndarray:
        """The same moments through ufs_dvm_moments_static (no allocation in the library: its sums go through the fixed
        array of STATIC_MAX_CELLS cells); `f`: a device tensor in the handle's layout, default the current f."""
        ufs_dvm_moments_static(self.h, None if f is None else f.data_ptr(), self.mom.data_ptr())
        ufs_dvm_sync(self.h)
        m = self.mom.cpu().numpy()
        out = np.empty_like(m)
        out[:, self.row_of_slab] = m
        return out

    def sync(self):
        ufs_dvm_sync(self.h)

    def close(self):
        if getattr(self, "h", None) is not None:
            ufs_dvm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
