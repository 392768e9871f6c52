// stream_common.cuh -- device helpers shared by the streaming step kernels (step_stream.cu, step_rows.cu).
#pragma once
#include "device_util.cuh"
#include "kernels.cuh"

namespace ufs {

// ---------------------------------------------------------------- the cell sums (SUMS_STRIDE doubles per cell)
// [0..4] H,  [5 + (2a+s)*5 + k] G[a][s][k];  s = 1: xi_a > 0.
__device__ __forceinline__ constexpr int g_index(int a, int s, int k) { return 5 + (2 * a + s) * 5 + k; }

// Warp-level sum of the 35 partials, stored to dst[0..35].  Butterfly with halving: at each of the five exchange
// steps a lane keeps one half of its values and hands the other half to its partner, so 36 -> 18 -> 9 -> 5 -> 3 -> 2
// values per lane and 37 exchanges in all (a plain shuffle reduction of 35 values takes 175).
template <int N, int OFF>
__device__ __forceinline__ void halve(double (&v)[36], int lane) {
    constexpr int H = (N + 1) / 2;
    const bool up = (lane & OFF) != 0;
#pragma unroll
    for (int i = 0; i < H; i++) {
        const double a = v[i], b = (i + H < N) ? v[i + H] : 0.0;
        const double recv = __shfl_xor_sync(0xffffffffu, up ? a : b, OFF);
        v[i] = (up ? b : a) + recv;
    }
}
__device__ __forceinline__ void warp_store_sums(const double (&acc)[35], double* dst, int lane) {
    double v[36];
#pragma unroll
    for (int i = 0; i < 35; i++) v[i] = acc[i];
    v[35] = 0.0;
    halve<36, 16>(v, lane);
    halve<18, 8>(v, lane);
    halve<9, 4>(v, lane);
    halve<5, 2>(v, lane);
    halve<3, 1>(v, lane);
    // lane holds v[t], t = 0, 1: entry t + 2 b0 + 3 b1 + 5 b2 + 9 b3 + 18 b4 of the sums (if every partial index is real)
    const int b0 = lane & 1, b1 = (lane >> 1) & 1, b2 = (lane >> 2) & 1, b3 = (lane >> 3) & 1, b4 = (lane >> 4) & 1;
#pragma unroll
    for (int t = 0; t < 2; t++) {
        const int j4 = t + 2 * b0, j3 = j4 + 3 * b1, j2 = j3 + 5 * b2, j1 = j2 + 9 * b3, j0 = j1 + 18 * b4;
        if (j4 < 3 && j3 < 5 && j2 < 9 && j1 < 18 && j0 < 36) dst[j0] = v[t];
    }
}

// ---------------------------------------------------------------- gather path (cells that are not "simple")
// value of the upwind source on axis a for octant o: one chunk, or 4 finer neighbours each weighted 1/4
// (reading G3), or the pointwise Maxwellian of a fluid leaf's frozen moments
template <typename T>
__device__ __forceinline__ void gather_axis(const StepParams& p, const int* __restrict__ rec, const T* fin, int a, int o,
                                            int CH, int e, int rx, int ry, int rz, T (&out)[V16<T>::N]) {
    constexpr int VEC = V16<T>::N;
    const int s = (o >> a) & 1;
    const int dir = 2 * a + (1 - s);  // xi_a > 0: data comes from the low side
    const int n = __ldg(rec + dir * 4 + 1) >= 0 ? 4 : 1;
    T acc[VEC];
#pragma unroll
    for (int i = 0; i < VEC; i++) acc[i] = T(0);
    for (int k = 0; k < n; k++) {
        const int code = __ldg(rec + dir * 4 + k);
        const int kind = code >> SRC_SHIFT;
        const int64_t idx = code & SRC_INDEX_MASK;
        if (kind == SRC_FLUID) {
            const FluidGhost* g = p.fluid + idx;
            const int kz = ((o >> 2) & 1) ? p.nh[2] + rz : p.nh[2] - 1 - rz;
            const int ky = ((o >> 1) & 1) ? p.nh[1] + ry : p.nh[1] - 1 - ry;
            const double b = g->amp * g->g[2][kz] * g->g[1][ky];
#pragma unroll
            for (int i = 0; i < VEC; i++) {
                const int kx = (o & 1) ? p.nh[0] + rx + i : p.nh[0] - 1 - rx - i;
                acc[i] += (T)(b * g->g[0][kx]);
            }
        } else {
            const T* base = (kind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + idx * p.Nv
                            + (int64_t)(kind == SRC_MIRROR ? (o ^ (1 << a)) : o) * CH;
            T v[VEC];
            ldg16(base + e, v);
#pragma unroll
            for (int i = 0; i < VEC; i++) acc[i] += v[i];
        }
    }
    const T wgt = (n == 4) ? T(0.25) : T(1);
#pragma unroll
    for (int i = 0; i < VEC; i++) out[i] = acc[i] * wgt;
}

// Table layout of one cell (TABN elements of T): [axis][sign][nhp] factors by rank of |xi|
// (axis 2 carries the amplitude), then dt*nu.
__host__ __device__ inline int nhp_of(const int32_t nh[3]) {
    int m = nh[0] > nh[1] ? nh[0] : nh[1];
    m = m > nh[2] ? m : nh[2];
    return (m + 3) & ~3;
}
__host__ __device__ inline int tabn_of(const int32_t nh[3]) { return 6 * nhp_of(nh) + 4; }

}  // namespace ufs
