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


// ---- one 16-byte vector of the storage type (4 floats / 2 doubles) ----------------------------------
template <typename T> struct V16;
template <> struct V16<float> { static constexpr int N = 4; using type = float4; };
template <> struct V16<double> { static constexpr int N = 2; using type = double2; };
template <typename T>
__device__ __forceinline__ void lds16(const T* p, T (&r)[V16<T>::N]) {
    *reinterpret_cast<typename V16<T>::type*>(r) = *reinterpret_cast<const typename V16<T>::type*>(p);
}
template <typename T>
__device__ __forceinline__ void sts16(T* p, const T (&r)[V16<T>::N]) {
    *reinterpret_cast<typename V16<T>::type*>(p) = *reinterpret_cast<const typename V16<T>::type*>(r);
}
__device__ __forceinline__ void ldg16(const float* p, float (&r)[4]) {
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "l"(p));
}
__device__ __forceinline__ void ldg16(const double* p, double (&r)[2]) {
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r[0]), "=d"(r[1]) : "l"(p));
}
__device__ __forceinline__ void stg16_cs(float* p, const float (&r)[4]) {
    __stcs(reinterpret_cast<float4*>(p), make_float4(r[0], r[1], r[2], r[3]));
}
__device__ __forceinline__ void stg16_cs(double* p, const double (&r)[2]) {
    __stcs(reinterpret_cast<double2*>(p), make_double2(r[0], r[1]));
}

// ---- mbarrier + bulk async copy (TMA engine, SASS UBLKCP): producer / consumer ring -----------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("{ .reg .b64 t; mbarrier.arrive.shared::cta.b64 t, [%0]; }" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("{ .reg .b64 t; mbarrier.arrive.expect_tx.shared::cta.b64 t, [%0], %1; }"
                 ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// Blocks until the phase with the given parity has completed (try_wait suspends the thread for a
// hardware-defined time slice, so the loop is not a busy spin).  A watchdog turns a protocol bug into a trap
// (reported as a CUDA error at the next sync) instead of a hung GPU.
#ifdef UFS_DEBUG_WAIT
static __device__ int g_dbg[8];
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, int code = 0) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        ++spins;
        if ((spins & 1023u) == 0 && *((volatile int*)&g_dbg[0]) != 0) return;
        if (spins > (1u << 20)) {
            if (atomicCAS(&g_dbg[0], 0, code + 1000) == 0) {
                g_dbg[1] = blockIdx.x; g_dbg[2] = threadIdx.x >> 5; g_dbg[3] = (int)parity;
                g_dbg[4] = (int)(smem_u32(bar));
            }
            return;
        }
    }
}
#else
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity, int = 0) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 26)) __trap();
    }
}
#endif
// global -> shared bulk copy of `bytes` (multiple of 16, both addresses 16-byte aligned); completion is
// signalled on `bar` as a transaction count
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy) : "memory");
}

// ---- the same primitives on 32-bit shared-space addresses (no generic-pointer conversion, one register) ----
__device__ __forceinline__ void smbar_arrive(uint32_t bar) {
    asm volatile("{ .reg .b64 t; mbarrier.arrive.shared::cta.b64 t, [%0]; }" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void smbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("{ .reg .b64 t; mbarrier.arrive.expect_tx.shared::cta.b64 t, [%0], %1; }" ::"r"(bar), "r"(bytes) : "memory");
}
// try_wait with a suspend-time hint: the thread sleeps in hardware until the phase completes or the hint elapses
__device__ __forceinline__ bool smbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(bar), "r"(parity), "r"(0x989680u) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void smbar_wait(uint32_t bar, uint32_t parity) {
#ifdef UFS_DEBUG_WAIT
    uint32_t spins = 0;
    while (!smbar_try_wait(bar, parity)) {
        if (++spins > (1u << 9)) __trap();
    }
#else
    while (!smbar_try_wait(bar, parity)) {}
#endif
}
__device__ __forceinline__ void sbulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void slds16(uint32_t a, float (&r)[4]) {
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "r"(a));
}
__device__ __forceinline__ void slds16(uint32_t a, double (&r)[2]) {
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(r[0]), "=d"(r[1]) : "r"(a));
}
__device__ __forceinline__ void ssts16(uint32_t a, const float (&r)[4]) {
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]) : "memory");
}
__device__ __forceinline__ void ssts16(uint32_t a, const double (&r)[2]) {
    asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(a), "d"(r[0]), "d"(r[1]) : "memory");
}
__device__ __forceinline__ float slds(uint32_t a, float) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ double slds(uint32_t a, double) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ int slds_i32(uint32_t a) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ int slds_i32_volatile(uint32_t a) { int v; asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ void ssts_i32_volatile(uint32_t a, int v) { asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

// pull `bytes` (multiple of 16) at a global address into L2 without a destination (TMA prefetch)
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

}  // namespace ufs
