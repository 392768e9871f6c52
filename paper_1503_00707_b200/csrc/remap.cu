// remap.cu -- k_remap: f of a new mesh from f of the old one, on the device.
//
// The paper redoes its steps 2 and 4 (array of f, stencil records) "each time the spatial mesh is changed"
// and names host preparation + transfer as the bottleneck; here the new records are
// flattened on the host (flatten.cpp) while f itself never leaves HBM: every new slab is a weighted sum of old slabs
// (reading G20: the volume average of the old piecewise-constant field -- copy, injection, or restriction over the old
// leaves inside the new one) or the frozen Maxwellian of an old FLUID leaf.  Pure streaming: one
// coalesced 16-byte vector per thread and source, fp64 accumulation, one store.
#include "device_util.cuh"
#include "kernels.cuh"

namespace ufs {
namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_remap(const T* __restrict__ f_old, T* __restrict__ f_new, const int64_t* __restrict__ off,
                                               const int32_t* __restrict__ src, const double* __restrict__ wgt,
                                               const FluidGhost* __restrict__ ghosts, const uchar4* __restrict__ slot_k,
                                               int64_t n_new, int64_t Nv) {
    constexpr int VEC = V16<T>::N;
    const int64_t nvec = Nv / VEC;
    for (int64_t s = blockIdx.x; s < n_new; s += gridDim.x) {
        const int64_t b = off[s], e = off[s + 1];
        T* dst = f_new + s * Nv;
        if (e - b == 1 && src[b] >= 0) {
            // unchanged leaf or injection: a plain copy of the covering slab
            const T* sp = f_old + (int64_t)src[b] * Nv;
            for (int64_t v = threadIdx.x; v < nvec; v += blockDim.x) {
                T x[VEC];
                ldg16(sp + v * VEC, x);
                stg16_cs(dst + v * VEC, x);
            }
            continue;
        }
        for (int64_t v = threadIdx.x; v < nvec; v += blockDim.x) {
            double acc[VEC];
#pragma unroll
            for (int i = 0; i < VEC; i++) acc[i] = 0.0;
            for (int64_t k = b; k < e; k++) {
                const int32_t c = src[k];
                const double w = wgt[k];
                if (c >= 0) {
                    T x[VEC];
                    ldg16(f_old + (int64_t)c * Nv + v * VEC, x);
#pragma unroll
                    for (int i = 0; i < VEC; i++) acc[i] = fma(w, (double)x[i], acc[i]);
                } else {
                    const FluidGhost* g = ghosts + (-1 - c);
#pragma unroll
                    for (int i = 0; i < VEC; i++) {
                        const uchar4 kk = slot_k[v * VEC + i];
                        acc[i] = fma(w, g->amp * g->g[2][kk.z] * g->g[1][kk.y] * g->g[0][kk.x], acc[i]);
                    }
                }
            }
            T out[VEC];
#pragma unroll
            for (int i = 0; i < VEC; i++) out[i] = (T)acc[i];
            stg16_cs(dst + v * VEC, out);
        }
    }
}

}  // namespace

cudaError_t launch_remap(int storage, const void* f_old, void* f_new, const int64_t* off, const int32_t* src, const double* wgt,
                         const FluidGhost* ghosts, const uchar4* slot_k, int64_t n_new, int64_t Nv, int sm_count, cudaStream_t st) {
    if (n_new == 0) return cudaSuccess;
    const int64_t want = (int64_t)sm_count * 8;
    const int grid = (int)(n_new < want ? n_new : want);
    if (storage == UFS_STORE_F32)
        k_remap<float><<<grid, 256, 0, st>>>(reinterpret_cast<const float*>(f_old), reinterpret_cast<float*>(f_new), off, src, wgt, ghosts, slot_k, n_new, Nv);
    else
        k_remap<double><<<grid, 256, 0, st>>>(reinterpret_cast<const double*>(f_old), reinterpret_cast<double*>(f_new), off, src, wgt, ghosts, slot_k, n_new, Nv);
    return cudaGetLastError();
}

}  // namespace ufs
