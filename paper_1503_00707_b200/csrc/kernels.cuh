// kernels.cuh -- device-side parameter block and launchers of the DVM step kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "flatten.hpp"

namespace ufs {

// Velocity-grid tables in device memory (one per handle).
struct VelDev {
    double xi[3][NV_MAX];  // node values, canonical index
    int32_t nv[3];
    int32_t nh[3];
};

// Everything a step launch needs.  Passed by value (kernel parameter space).
struct StepParams {
    const void* f_in;           // [n_kin][Nv] storage type, current f
    void* f_out;                // [n_kin][Nv] next f
    const CellRec* cells;       // [n_kin]
    const void* tables;         // [n_tables][Nv] storage type, slot order (inflow ghosts)
    const FluidGhost* fluid;    // [n_fluid_ghosts]
    const VelDev* vel;
    const uchar4* slot_k;       // [Nv] (kx,ky,kz,0) of each slot          (generic path, moments)
    const int32_t* mirror_slot; // [3][Nv]                                  (generic path)
    int32_t* flags;             // bit 0: a Newton solve failed
    int64_t Nv;
    int32_t n_kin;
    int32_t nv[3], nh[3];
    int32_t collide;            // 0: Kn = inf, pure transport
    double dt, w, inv_len, inv_kn, visc_exp, nu_pref;
};

struct StepLaunch {
    int32_t threads, smem_bytes, vec, fast;
};

// Chooses the kernel variant for this storage type / grid and returns its launch geometry, or an
// error (negative) if the slab does not fit on chip.
int step_plan(int storage, const VelLayout& v, StepLaunch* plan, const char** why);

// Enqueue one fused step (transport + moments + discrete Maxwellian + relaxation) on `stream`.
cudaError_t launch_step(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t stream);

// Enqueue the moments kernel: mom[5][n_kin] = (n, n u, E) of f.
cudaError_t launch_moments(int storage, const StepParams& p, const void* f, double* mom, cudaStream_t stream);

}  // namespace ufs
