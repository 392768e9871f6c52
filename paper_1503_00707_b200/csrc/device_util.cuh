// device_util.cuh -- small device helpers shared by the DVM step kernels (sm_100a): 128-bit global /
// shared accessors with explicit cache policy, warp reductions, named barriers.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace ufs {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- four consecutive elements of the storage type (16 B for fp32, 32 B for fp64) ------------------
// Global reads of f go through the read-only path without allocating in L1: every value is used once by
// this CTA; the reuse (a slab is also the upwind source of its three downwind neighbours) is L2's job.
__device__ __forceinline__ void ldg4(const float* p, float (&r)[4]) {
    asm("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
        : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "l"(p));
}
__device__ __forceinline__ void ldg4(const double* p, double (&r)[4]) {
    asm("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r[0]), "=d"(r[1]) : "l"(p));
    asm("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r[2]), "=d"(r[3]) : "l"(p + 2));
}
// streaming store (evict-first in L2): the new f is not read again during this step
__device__ __forceinline__ void stg4_cs(float* p, const float (&r)[4]) {
    __stcs(reinterpret_cast<float4*>(p), make_float4(r[0], r[1], r[2], r[3]));
}
__device__ __forceinline__ void stg4_cs(double* p, const double (&r)[4]) {
    __stcs(reinterpret_cast<double2*>(p), make_double2(r[0], r[1]));
    __stcs(reinterpret_cast<double2*>(p) + 1, make_double2(r[2], r[3]));
}
__device__ __forceinline__ void lds4(const float* p, float (&r)[4]) {
    const float4 v = *reinterpret_cast<const float4*>(p);
    r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w;
}
__device__ __forceinline__ void lds4(const double* p, double (&r)[4]) {
    const double2 a = *reinterpret_cast<const double2*>(p), b = *(reinterpret_cast<const double2*>(p) + 1);
    r[0] = a.x; r[1] = a.y; r[2] = b.x; r[3] = b.y;
}
__device__ __forceinline__ void sts4(float* p, const float (&r)[4]) {
    *reinterpret_cast<float4*>(p) = make_float4(r[0], r[1], r[2], r[3]);
}
__device__ __forceinline__ void sts4(double* p, const double (&r)[4]) {
    *reinterpret_cast<double2*>(p) = make_double2(r[0], r[1]);
    *(reinterpret_cast<double2*>(p) + 1) = make_double2(r[2], r[3]);
}

// ---- named barriers (bar.sync / bar.arrive): producer / consumer hand-over between warp roles ------
__device__ __forceinline__ void bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int nthreads) {
    __threadfence_block();  // publish this thread's shared-memory writes before announcing them
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

}  // namespace ufs
