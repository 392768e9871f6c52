"""Harness-side plumbing around the C-ABI library: device-resident initial states for cases whose f
does not fit a host array, clock sampling for the bench, and the windowed sub-problems used to
check full-size runs against the oracle.  None of the method's arithmetic lives here."""
from __future__ import annotations

import threading
import time
from typing import Optional

import numpy as np

from . import binding as B
from . import inputs as _inputs
from .inputs import STORE_F32, Case


def fill_initial_f_device(st: "B.DvmStepper", case: Case, chunk_slabs: int = 2048) -> None:
    """Write f(t=0) = pointwise Maxwellian of case.prim0 straight into the library's current device
    buffer, slab by slab, in slab/slot order, with plain PyTorch ops on the device (an INPUT recipe,
    the same formula as inputs.maxwellian_canonical; rounded to the storage type).  Noise-free cases only."""
    torch = st.torch
    assert case.noise_rel == 0.0, "seeded per-cell noise is generated on the host (inputs.initial_f)"
    dev = st.device
    cur = B.ufs_dvm_current(st.h)
    nvx, nvy, nvz = case.nv
    vel = torch.as_tensor(st.vel_of_slot.astype(np.int64), device=dev)
    kx, ky, kz = vel % nvx, (vel // nvx) % nvy, vel // (nvx * nvy)
    xs, ys, zs = (torch.as_tensor(case.xi_nodes(a), device=dev) for a in range(3))
    prim = torch.as_tensor(case.prim0[st.cell_of_slab], device=dev)            # [n_kin, 5] in slab order
    with torch.cuda.stream(st.stream):           # ordered with the handle's stream
        for s0 in range(0, st.n_kinetic, chunk_slabs):
            s1 = min(s0 + chunk_slabs, st.n_kinetic)     # (a partitioned handle's tensors hold ghost slabs after these)
            p = prim[s0:s1]
            n, ux, uy, uz, T = (p[:, c:c + 1] for c in range(5))
            ex = torch.exp(-(xs[None, :] - ux) ** 2 / (2 * T))
            ey = torch.exp(-(ys[None, :] - uy) ** 2 / (2 * T))
            ez = torch.exp(-(zs[None, :] - uz) ** 2 / (2 * T))
            a = n / (2 * np.pi * T) ** 1.5
            f = a * ez[:, kz] * ey[:, ky] * ex[:, kx]
            st.f[cur][s0:s1].copy_(f.to(st.dtype))
    B.ufs_dvm_f_changed(st.h)


# mesh slicing lives with the problem descriptions (no arithmetic of the method): re-exported for the tests
window_leaves, sub_case = _inputs.window_leaves, _inputs.sub_case


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while a timed region runs."""

    def __init__(self, index: int = 0, period_s: float = 0.1):
        self.index, self.period = index, period_s
        self.samples, self.reasons = [], set()
        self._stop = threading.Event()
        self._thr = None
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.handle, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self) -> dict:
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}
