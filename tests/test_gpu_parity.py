"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star, reading G17 = max|a-b| / max|b| per array):
1e-12 for fp64 storage, 2e-5 for fp32 storage with fp64 moment accumulation."""
import math

import numpy as np
import pytest

from oracle.dvm_oracle import Oracle
from paper_1503_00707_b200 import binding as B
from paper_1503_00707_b200 import inputs
from tests.helpers import assert_moments_close, periodic_case, random_tree, rel_linf

pytestmark = pytest.mark.gpu
TOL = {inputs.STORE_F64: 1e-12, inputs.STORE_F32: 2e-5}
P = (True, True, True)


def run_both(case, nsteps, kn=None, storage=None, f0=None):
    st = B.DvmStepper(case, kn=kn, storage=storage)
    if f0 is None:
        f0 = inputs.initial_f(case)
    if st.storage == inputs.STORE_F32:
        f0 = f0.astype(np.float32).astype(np.float64)
    st.load_canonical(f0)
    st.step(case.dt, nsteps)
    st.sync()
    f_gpu = st.read_canonical()
    m_gpu = st.moments()
    launches = B.ufs_dvm_launch_count(st.h)
    info = B.ufs_dvm_kernel_info(st.h)
    st.close()
    o = Oracle(case, kn=kn)
    f_ref = o.step(f0, case.dt, nsteps)
    m_ref = o.moments(f_ref)
    return f_gpu, m_gpu, f_ref, m_ref, launches, info


def check(case, nsteps, tol, **kw):
    f_gpu, m_gpu, f_ref, m_ref, launches, info = run_both(case, nsteps, **kw)
    assert launches >= nsteps + 1          # at least one kernel per step plus the moments kernel
    assert np.all(np.isfinite(f_gpu))
    err_f = rel_linf(f_gpu, f_ref)
    assert err_f <= tol, f"f: {err_f:.3e}"
    storage = kw.get("storage")
    storage = case.storage if storage is None else storage
    # moments: never tighter than the stated tolerance of the storage type (a tiny momentum field, e.g. noise only,
    # carries the summation round-off of n * sqrt(R T0) on a scale of its own norm)
    assert_moments_close(m_gpu, m_ref, max(tol, TOL[storage]), eps_storage=6e-8 if storage == inputs.STORE_F32 else 2.3e-16)
    return info


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_small_configs_match_oracle(cfg):
    case = inputs.small(cfg)
    info = check(case, case.nsteps, TOL[case.storage])
    assert info["fast"]


def test_config1_full_run_10_steps():
    case = inputs.config1()
    check(case, 10, 1e-12)


def test_config1_fp32_storage():
    case = inputs.config1()
    check(case, 10, 2e-5, storage=inputs.STORE_F32)


@pytest.mark.parametrize("cfg", [1, 3])
def test_transport_only_kn_inf(cfg):
    case = inputs.small(cfg)
    check(case, 3, 1e-13, kn=math.inf)


def test_small_config3_fp32():
    case = inputs.small(3)
    check(case, 3, 2e-5, storage=inputs.STORE_F32)


def test_small_config5_fp32():
    case = inputs.small(5)
    check(case, 3, 2e-5, storage=inputs.STORE_F32)


@pytest.mark.parametrize("nv,vmin,vmax", [((5, 4, 3), (-4.0, -3.0, -2.5), (4.0, 5.0, 2.5)),
                                          ((7, 7, 7), (-4.0,) * 3, (4.0,) * 3),
                                          ((6, 10, 2), (-4.0, -5.0, -2.0), (4.0, 5.0, 2.0))])
def test_generic_and_odd_velocity_grids(nv, vmin, vmax):
    """Odd nv (a zero node carries no flux on its axis), asymmetric limits, non-cubic grids."""
    lv, ijk = random_tree(np.random.default_rng(4), 1, 3, P, 0.3)
    case = periodic_case(lv, ijk, nv=nv, kn=0.2)
    case.vmin, case.vmax = vmin, vmax
    rng = np.random.default_rng(1)
    f0 = inputs.maxwellian_canonical(case, case.prim0) * (1 + 0.2 * rng.uniform(-1, 1, (case.n_leaves, case.Nv)))
    info = check(case, 3, 1e-12, f0=f0)
    sym_even = all(n % 2 == 0 and abs(a + b) < 1e-12 for n, a, b in zip(nv, vmin, vmax))
    assert info["fast"] == sym_even


@pytest.mark.parametrize("nv,storage,kernel", [((16, 16, 16), inputs.STORE_F64, "k_stream"),
                                               ((16, 8, 8), inputs.STORE_F32, "k_stream"),
                                               ((12, 12, 12), inputs.STORE_F64, "k_rows"),
                                               ((24, 12, 8), inputs.STORE_F32, "k_rows"),
                                               ((12, 12, 12), inputs.STORE_F32, "k_step_fast")])
def test_kernel_selection_and_parity_on_other_even_grids(nv, storage, kernel):
    """Every streaming kernel and its fallbacks: k_rows needs nh_x in {6, 12} (fp32: 12), k_stream a whole number of
    16-byte vectors per x run, the one-CTA-per-cell kernel takes the rest.  2:1 faces and specular walls included."""
    lv, ijk = random_tree(np.random.default_rng(11), 1, 3, (True, False, True), 0.3)
    bc = (inputs.BC_PERIODIC, inputs.BC_PERIODIC, inputs.BC_SPECULAR, inputs.BC_SPECULAR, inputs.BC_PERIODIC, inputs.BC_PERIODIC)
    case = periodic_case(lv, ijk, nv=nv, kn=0.2, bc=bc)
    rng = np.random.default_rng(3)
    f0 = inputs.maxwellian_canonical(case, case.prim0) * (1 + 0.2 * rng.uniform(-1, 1, (case.n_leaves, case.Nv)))
    st = B.DvmStepper(case, storage=storage)
    assert B.ufs_dvm_kernel_name(st.h) == kernel
    st.close()
    check(case, 3, TOL[storage], storage=storage, f0=f0)


@pytest.mark.parametrize("cfg,kernel", [(3, "rows"), (4, "rows"), (5, "rows"), (4, "stream"), (3, "cell")])
def test_fallback_kernels_on_the_24_cubed_grid(cfg, kernel, monkeypatch):
    """24^3 grids get k_tiles; UFS_DVM_KERNEL forces the kernels that serve the other grids: they must stay right."""
    monkeypatch.setenv("UFS_DVM_KERNEL", kernel)
    case = inputs.small(cfg)
    st = B.DvmStepper(case)
    assert B.ufs_dvm_kernel_name(st.h) == {"rows": "k_rows", "stream": "k_stream", "cell": "k_step_fast"}[kernel]
    st.close()
    check(case, case.nsteps, TOL[case.storage])


def test_small_configs_use_the_tile_kernel():
    for cfg in (2, 3, 4, 5):
        st = B.DvmStepper(inputs.small(cfg))
        assert B.ufs_dvm_kernel_name(st.h) == "k_tiles"
        st.close()


def test_specular_box_with_odd_grid_generic_path():
    lv, ijk = inputs.build_tree(2, 2, {}, P)
    case = periodic_case(lv, ijk, nv=(5, 5, 5), bc=(inputs.BC_SPECULAR,) * 6, kn=0.3)
    rng = np.random.default_rng(2)
    f0 = inputs.maxwellian_canonical(case, case.prim0) * (1 + 0.2 * rng.uniform(-1, 1, (case.n_leaves, case.Nv)))
    check(case, 3, 1e-12, f0=f0)


def test_newton_failure_is_reported():
    case = inputs.config1()
    st = B.DvmStepper(case)
    f0 = -inputs.initial_f(case)                     # negative density
    st.load_canonical(f0)
    st.step(case.dt, 1)
    with pytest.raises(B.UfsDvmError) as e:
        st.sync()
    assert e.value.code == B.ENEWTON
    with pytest.raises(B.UfsDvmError):               # sticky
        st.step(case.dt, 1)
    st.close()


def test_run_host_entry_point():
    import ctypes as C
    import torch
    case = inputs.small(2)
    st = B.DvmStepper(case)
    f0 = inputs.initial_f(case)
    host_in = np.ascontiguousarray(f0[st.row_of_slab][:, st.vel_of_slot])
    host_out = np.empty_like(host_in)
    mom_host = np.empty((5, st.n_kinetic))
    B.ufs_dvm_run_host(st.h, host_in.ctypes.data, host_out.ctypes.data, st.mom.data_ptr(), mom_host.ctypes.data,
                       case.dt, 2)
    o = Oracle(case)
    f_ref = o.step(f0, case.dt, 2)
    inv = np.empty(case.Nv, np.int64); inv[st.vel_of_slot] = np.arange(case.Nv)
    got = np.empty_like(f_ref); got[st.row_of_slab] = host_out[:, inv]
    assert rel_linf(got, f_ref) <= 1e-12
    m = np.empty_like(mom_host); m[:, st.row_of_slab] = mom_host
    assert rel_linf(m[0], o.moments(f_ref)[0]) <= 1e-12
    st.close()


def test_uniform_maxwellian_steady_on_gpu():
    """P1 on the device: adaptive periodic tree, same Maxwellian everywhere, collisions on."""
    case = inputs.config1(nv=24)
    case.vmin, case.vmax = (-5.0,) * 3, (5.0,) * 3
    prim = np.tile(np.array([[1.3, 0.4, -0.2, 0.1, 0.9]]), (case.n_leaves, 1))
    f0 = inputs.maxwellian_canonical(case, prim)
    st = B.DvmStepper(case)
    st.load_canonical(f0)
    st.step(case.dt, 3)
    st.sync()
    assert rel_linf(st.read_canonical(), f0) < 5e-14
    st.close()


def test_stalled_pipeline_traps_and_is_reported_not_hung():
    """Every wait of the persistent kernel has a wall-clock watchdog (device_util.cuh: smbar_wait): with the test hook
    UFS_DVM_TEST_STALL one producer warp withholds a barrier arrival, the consumers' wait times out, the kernel traps and
    ufs_dvm_sync returns UFS_DVM_ECUDA.  Run in a child process: a device trap takes the CUDA context with it."""
    import os
    import subprocess
    import sys
    import time
    code = (
        "import sys, time\n"
        "from paper_1503_00707_b200 import binding as B, inputs\n"
        "case = inputs.small(3)\n"
        "st = B.DvmStepper(case)\n"
        "assert B.ufs_dvm_kernel_name(st.h) == 'k_tiles'\n"
        "st.load_canonical(inputs.initial_f(case))\n"
        "t0 = time.time()\n"
        "try:\n"
        "    st.step(case.dt, 1)\n"
        "    st.sync()\n"
        "    print('NO ERROR')\n"
        "except B.UfsDvmError as e:\n"
        "    print('CODE', e.code, 'SECONDS %.1f' % (time.time() - t0))\n"
        "sys.stdout.flush()\n"
        "import os; os._exit(0)\n")
    env = dict(os.environ, UFS_DVM_TEST_STALL="1")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    t0 = time.time()
    res = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True, timeout=120)
    assert f"CODE {B.ECUDA}" in res.stdout, res.stdout + res.stderr
    assert time.time() - t0 < 60            # seconds, not a hang
    # and the same process without the hook is fine
    res = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ), capture_output=True, text=True, timeout=120)
    assert "NO ERROR" in res.stdout, res.stdout + res.stderr


def test_check_mode_catches_a_forgotten_f_changed(monkeypatch):
    """UFS_DVM_CHECK (include/ufs_dvm.h): rewriting f on the device without ufs_dvm_f_changed is reported as EINVAL at the
    next sync; with the call, or without a rewrite, nothing is reported."""
    monkeypatch.setenv("UFS_DVM_CHECK", "1")
    case = inputs.small(3)
    f0 = inputs.initial_f(case)
    st = B.DvmStepper(case)
    st.load_canonical(f0)
    st.step(case.dt, 2)
    st.step(case.dt, 1)
    st.sync()                                              # clean run: no report
    cur = B.ufs_dvm_current(st.h)
    st.f[cur].mul_(1.5)                                    # the caller rewrites f ...
    B.ufs_dvm_f_changed(st.h)                              # ... and says so
    st.step(case.dt, 1)
    st.sync()
    st.f[B.ufs_dvm_current(st.h)].mul_(1.5)                # ... and forgets to say so
    st.step(case.dt, 1)
    with pytest.raises(B.UfsDvmError) as e:
        st.sync()
    assert e.value.code == B.EINVAL and "ufs_dvm_f_changed" in str(e.value)
    st.close()


@pytest.mark.parametrize("storage", [inputs.STORE_F64, inputs.STORE_F32])
@pytest.mark.parametrize("nv", [(24, 16, 12), (24, 8, 24)])
def test_tile_kernel_on_non_cubic_velocity_grids(nv, storage):
    """k_tiles takes any even symmetric grid with 12 positive x nodes and whole row blocks (48 rows for fp32, 24 for fp64
    storage); the row-block / half-row arithmetic must not depend on nh_y = nh_z = 12."""
    lv, ijk = random_tree(np.random.default_rng(21), 1, 3, P, 0.3)
    case = periodic_case(lv, ijk, nv=nv, vlim=5.0, kn=0.1)
    case.storage = storage
    rng = np.random.default_rng(3)
    f0 = inputs.initial_f(case) * (1 + 0.2 * rng.uniform(-1, 1, (case.n_leaves, case.Nv)))
    st = B.DvmStepper(case)
    name = B.ufs_dvm_kernel_name(st.h)
    st.close()
    assert name == "k_tiles"
    check(case, 3, TOL[storage], f0=f0)
