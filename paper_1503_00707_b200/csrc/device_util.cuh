// device_util.cuh -- small device helpers shared by the DVM step kernels (sm_100a): 128-bit global /
// shared accessors with explicit cache policy, warp reductions, mbarrier + bulk-copy (TMA) primitives.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace ufs {

// Watchdog of the persistent kernels' waits: a wait that lasts this long (wall clock, %globaltimer) can only be a
// protocol bug or a faulted copy.
#ifndef UFS_WAIT_TIMEOUT_NS
#define UFS_WAIT_TIMEOUT_NS 2000000000ull
#endif

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
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
// plain 16-byte store (peer memory: the ghost slabs of another rank)
__device__ __forceinline__ void stg16(float* p, const float (&r)[4]) { *reinterpret_cast<float4*>(p) = make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ void stg16(double* p, const double (&r)[2]) { *reinterpret_cast<double2*>(p) = make_double2(r[0], r[1]); }

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
// (reported as UFS_DVM_ECUDA at the next ufs_dvm_sync) instead of a hung GPU.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 26)) __trap();
    }
}
// global -> shared bulk copy of `bytes` (multiple of 16, both addresses 16-byte aligned); completion is
// signalled on `bar` as a transaction count
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
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
__device__ __forceinline__ unsigned long long globaltimer_ns() {
    unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t;
}
// Waits of the persistent kernels.  try_wait suspends the thread in hardware until the phase completes or a short,
// hardware-defined time has passed (the hint above is an upper bound, in practice a fraction of a microsecond), so the
// loop is not a busy spin.  The watchdog is a wall-clock one: UFS_WAIT_TIMEOUT_NS without the phase completing traps, so
// that the failure surfaces as UFS_DVM_ECUDA at ufs_dvm_sync instead of hanging the GPU; a kernel slowed down many times
// over (a profiler's replay pass, a debugger) does not trip it.  The timer is read in the slow path only.
__device__ __forceinline__ void smbar_wait(uint32_t bar, uint32_t parity) {
    if (smbar_try_wait(bar, parity)) return;
    const unsigned long long t0 = globaltimer_ns();
    while (!smbar_try_wait(bar, parity)) {
        if (globaltimer_ns() - t0 > UFS_WAIT_TIMEOUT_NS) __trap();
    }
}
// The same wait for a warp that is in no hurry (a producer waiting for a ring slot, several stages ahead of the
// consumers): sleeps between polls so that it does not take issue slots and power from the warps that do the work.
__device__ __forceinline__ void smbar_wait_relaxed(uint32_t bar, uint32_t parity) {
    if (smbar_try_wait(bar, parity)) return;
    const unsigned long long t0 = globaltimer_ns();
    while (!smbar_try_wait(bar, parity)) {
        __nanosleep(256);
        if (globaltimer_ns() - t0 > UFS_WAIT_TIMEOUT_NS) __trap();
    }
}
__device__ __forceinline__ void sbulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ int slds_i32(uint32_t a) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ int slds_i32_volatile(uint32_t a) { int v; asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ void ssts_i32_volatile(uint32_t a, int v) { asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void ssts_i32(uint32_t a, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

}  // namespace ufs
