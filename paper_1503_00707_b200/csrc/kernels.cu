// kernels.cu -- sm_100a kernels of the fused DVM step.
//
// One CTA per kinetic cell.  f is stored velocity-fastest, the 8 velocity octants (sign groups,
// PAPER.md:106-112) contiguous inside a cell's slab, and inside an octant the nodes are ordered by
// increasing |xi| on every axis.  Consequences used below:
//   * for one octant the upwind neighbour is the same for every velocity, so the
//     transport update of a whole octant chunk is  f* = c0*f_own + cx*f_X + cy*f_Y + cz*f_Z  with
//     four contiguous, fully coalesced 128-bit streams (own cell + one upwind source per axis);
//   * a thread keeps the same |xi| (hence the same c's) for all 8 octants: only signs change;
//   * specular reflection maps an octant chunk onto the mirrored octant chunk at the same offset.
// f* of the cell is staged in shared memory (the slab buffer), the 5 moments are reduced with warp
// shuffles + one shared-memory pass, warp 0 runs the Newton iteration for the discrete Maxwellian
// on the separable 1-D sums, and the relaxation epilogue streams the slab buffer out once.
// HBM traffic per phase-space cell update: 1 read + 1 write of f; the 3 upwind re-reads are L2 hits
// when the slabs are visited in Morton order.
#include "kernels.cuh"

namespace ufs {
namespace {

// ---------------------------------------------------------------- vector load / store helpers
template <typename T, int VEC> struct VecOf;
template <> struct VecOf<float, 4> { using type = float4; };
template <> struct VecOf<float, 2> { using type = float2; };
template <> struct VecOf<float, 1> { using type = float; };
template <> struct VecOf<double, 2> { using type = double2; };
template <> struct VecOf<double, 1> { using type = double; };

template <typename T, int VEC>
__device__ __forceinline__ void ld_global_nc(const T* p, T (&r)[VEC]) {
    using V = typename VecOf<T, VEC>::type;
    const V v = __ldg(reinterpret_cast<const V*>(p));
    *reinterpret_cast<V*>(r) = v;
}
template <typename T, int VEC>
__device__ __forceinline__ void st_global_cs(T* p, const T (&r)[VEC]) {
    using V = typename VecOf<T, VEC>::type;
    __stcs(reinterpret_cast<V*>(p), *reinterpret_cast<const V*>(r));
}
template <typename T, int VEC>
__device__ __forceinline__ void ld_shared(const T* p, T (&r)[VEC]) {
    using V = typename VecOf<T, VEC>::type;
    *reinterpret_cast<V*>(r) = *reinterpret_cast<const V*>(p);
}
template <typename T, int VEC>
__device__ __forceinline__ void st_shared(T* p, const T (&r)[VEC]) {
    using V = typename VecOf<T, VEC>::type;
    *reinterpret_cast<V*>(p) = *reinterpret_cast<const V*>(r);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---------------------------------------------------------------- shared-memory carve-up
struct Smem {
    unsigned char* slab;  // [Nv] T : f* of the cell
    double* red;          // [32][5] per-warp partial moments, then rho in red[0..4]
    double* res;          // [4] amp, omega
    double* g;            // [3][NVP] Maxwellian factors exp(alpha_a xi + alpha_4 xi^2), canonical node index
    float* gf;            // [3][NVP] float copy (fp32 storage)
    const void** ptr;     // [8][4] per octant: own chunk, x/y/z upwind chunk (simple cells)
    int* rec;             // [32] the cell record
};
__host__ __device__ inline size_t smem_bytes_for(int64_t Nv, size_t elem, int nvp, int nwarps) {
    size_t b = ((size_t)Nv * elem + 15) & ~(size_t)15;
    b += (size_t)nwarps * 5 * 8 + 4 * 8 + (size_t)3 * nvp * 8 + (size_t)3 * nvp * 4 + 32 * 8 + 32 * 4;
    return (b + 15) & ~(size_t)15;
}
__device__ __forceinline__ Smem carve(unsigned char* base, int64_t Nv, size_t elem, int nvp, int nwarps) {
    Smem s;
    s.slab = base;
    size_t off = ((size_t)Nv * elem + 15) & ~(size_t)15;
    s.red = reinterpret_cast<double*>(base + off); off += (size_t)nwarps * 5 * 8;
    s.res = reinterpret_cast<double*>(base + off); off += 4 * 8;
    s.g = reinterpret_cast<double*>(base + off); off += (size_t)3 * nvp * 8;
    s.ptr = reinterpret_cast<const void**>(base + off); off += 32 * 8;
    s.gf = reinterpret_cast<float*>(base + off); off += (size_t)3 * nvp * 4;
    s.rec = reinterpret_cast<int*>(base + off);
    return s;
}

// ---------------------------------------------------------------- discrete Maxwellian (a3)
// Newton iteration for alpha with  w sum_i m(xi_i) exp(alpha . m(xi_i)) = rho.
// exp(alpha.m) = e^{alpha_0} gx[kx] gy[ky] gz[kz] with g_a[k] = exp(alpha_a xi_k + alpha_4 xi_k^2), so the
// residual and the 5x5 Jacobian follow from the 1-D sums P_a^r = sum_k xi_k^r g_a[k], r = 0..4.
// Run by warp 0 (all 32 lanes; every lane ends with the same alpha).  Same start and stop rule as
// the oracle; the per-cell 5x5 solve is the analogue of PAPER.md:179 ("Gauss method").
__device__ __noinline__ void newton_warp(const VelDev* __restrict__ vel, int nvx, int nvy, int nvz, int nvp,
                                         double w, double dt, double inv_kn, double visc_exp, double nu_pref,
                                         int32_t* flags, const double* rho_s, double* sg, float* sgf, double* sres) {
    const int lane = threadIdx.x & 31;
    double rho[5];
#pragma unroll
    for (int a = 0; a < 5; a++) rho[a] = rho_s[a];
    const double n = rho[0];
    const double ux = rho[1] / n, uy = rho[2] / n, uz = rho[3] / n;
    const double uu = ux * ux + uy * uy + uz * uz;
    const double T = (rho[4] - n * uu) / (3.0 * n);
    bool ok = (n > 0.0) && (T > 0.0);
    double al[5];
    al[0] = log(n / (2.0 * 3.14159265358979323846 * T * sqrt(2.0 * 3.14159265358979323846 * T))) - uu / (2.0 * T);
    al[1] = ux / T; al[2] = uy / T; al[3] = uz / T; al[4] = -1.0 / (2.0 * T);
    const double sT = n * sqrt(T);
    const double scale[5] = {n, sT + fabs(rho[1]), sT + fabs(rho[2]), sT + fabs(rho[3]), rho[4]};
    const int nvs[3] = {nvx, nvy, nvz};
    bool converged = false;
    if (ok) {
        for (int it = 0; it <= 50; it++) {
            double P[3][5];
#pragma unroll
            for (int a = 0; a < 3; a++) {
                double p0 = 0, p1 = 0, p2 = 0, p3 = 0, p4 = 0;
                for (int k = lane; k < nvs[a]; k += 32) {
                    const double x = vel->xi[a][k];
                    const double g = exp(al[1 + a] * x + al[4] * x * x);
                    sg[a * nvp + k] = g;
                    double t = g;
                    p0 += t; t *= x; p1 += t; t *= x; p2 += t; t *= x; p3 += t; t *= x; p4 += t;
                }
                P[a][0] = warp_sum(p0); P[a][1] = warp_sum(p1); P[a][2] = warp_sum(p2);
                P[a][3] = warp_sum(p3); P[a][4] = warp_sum(p4);
            }
            const double A = exp(al[0]) * w;
            const double* X = P[0]; const double* Y = P[1]; const double* Z = P[2];
            double J[5][5], F[5];
            J[0][0] = A * X[0] * Y[0] * Z[0];
            J[0][1] = A * X[1] * Y[0] * Z[0];
            J[0][2] = A * X[0] * Y[1] * Z[0];
            J[0][3] = A * X[0] * Y[0] * Z[1];
            J[0][4] = A * (X[2] * Y[0] * Z[0] + X[0] * Y[2] * Z[0] + X[0] * Y[0] * Z[2]);
            J[1][1] = A * X[2] * Y[0] * Z[0];
            J[1][2] = A * X[1] * Y[1] * Z[0];
            J[1][3] = A * X[1] * Y[0] * Z[1];
            J[1][4] = A * (X[3] * Y[0] * Z[0] + X[1] * Y[2] * Z[0] + X[1] * Y[0] * Z[2]);
            J[2][2] = A * X[0] * Y[2] * Z[0];
            J[2][3] = A * X[0] * Y[1] * Z[1];
            J[2][4] = A * (X[2] * Y[1] * Z[0] + X[0] * Y[3] * Z[0] + X[0] * Y[1] * Z[2]);
            J[3][3] = A * X[0] * Y[0] * Z[2];
            J[3][4] = A * (X[2] * Y[0] * Z[1] + X[0] * Y[2] * Z[1] + X[0] * Y[0] * Z[3]);
            J[4][4] = A * (X[4] * Y[0] * Z[0] + X[0] * Y[4] * Z[0] + X[0] * Y[0] * Z[4]
                           + 2.0 * (X[2] * Y[2] * Z[0] + X[2] * Y[0] * Z[2] + X[0] * Y[2] * Z[2]));
            double res = 0.0;
#pragma unroll
            for (int a = 0; a < 5; a++) {
                F[a] = J[0][a] - rho[a];
                const double r = fabs(F[a]) / scale[a];
                if (!(r <= res)) res = r;  // NaN propagates
            }
            if (res <= 1e-13) { converged = true; break; }
            if (it == 50 || !(res == res)) break;
            // symmetric positive definite 5x5: Gauss elimination, no pivoting needed
#pragma unroll
            for (int a = 0; a < 5; a++)
#pragma unroll
                for (int b = 0; b < a; b++) J[a][b] = J[b][a];
#pragma unroll
            for (int c = 0; c < 5; c++) {
                const double inv = 1.0 / J[c][c];
#pragma unroll
                for (int r = c + 1; r < 5; r++) {
                    const double m = J[r][c] * inv;
#pragma unroll
                    for (int k = c + 1; k < 5; k++) J[r][k] -= m * J[c][k];
                    F[r] -= m * F[c];
                }
            }
            double dx[5];
#pragma unroll
            for (int r = 4; r >= 0; r--) {
                double s = F[r];
#pragma unroll
                for (int k = r + 1; k < 5; k++) s -= J[r][k] * dx[k];
                dx[r] = s / J[r][r];
            }
#pragma unroll
            for (int a = 0; a < 5; a++) al[a] -= dx[a];
        }
    }
    if (converged) {
        // G9: nu = c_nu n T^(1-omega) / Kn (omega = 1/2: sqrt)
        const double Tp = (visc_exp == 0.5) ? sqrt(T) : pow(T, 1.0 - visc_exp);
        const double amp = exp(al[0]);
#pragma unroll
        for (int a = 0; a < 3; a++)
            for (int k = lane; k < nvs[a]; k += 32) sgf[a * nvp + k] = (float)sg[a * nvp + k];
        if (lane == 0) { sres[0] = amp; sres[1] = dt * nu_pref * n * Tp * inv_kn; }
    } else {
        // no Maxwellian: pass f* through unchanged and raise the sticky flag (UFS_DVM_ENEWTON)
#pragma unroll
        for (int a = 0; a < 3; a++)
            for (int k = lane; k < nvs[a]; k += 32) { sg[a * nvp + k] = 0.0; sgf[a * nvp + k] = 0.f; }
        if (lane == 0) { sres[0] = 0.0; sres[1] = 0.0; atomicOr(flags, 1); }
    }
}

// block-wide sum of the 5 partial moments; result (times w) in s.red[0..4], visible after the barrier
__device__ __forceinline__ void block_reduce_moments(double (&mom)[5], const Smem& s, double w) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int a = 0; a < 5; a++) mom[a] = warp_sum(mom[a]);
    __syncthreads();  // everybody is done with s.red / s.ptr users of the previous phase
    if (lane == 0) {
#pragma unroll
        for (int a = 0; a < 5; a++) s.red[warp * 5 + a] = mom[a];
    }
    __syncthreads();
    if (warp == 0) {
        double r[5];
#pragma unroll
        for (int a = 0; a < 5; a++) r[a] = warp_sum(lane < nwarp ? s.red[lane * 5 + a] : 0.0);
        __syncwarp();
        if (lane == 0) {
#pragma unroll
            for (int a = 0; a < 5; a++) s.red[a] = r[a] * w;
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------- octant fast path
// value of an upwind source that is not a plain chunk pointer: 4 finer neighbours and / or fluid ghosts
template <typename T, int VEC>
__device__ __forceinline__ void gather_axis(const StepParams& p, const int* rec, const T* fin, int a, int o, int e,
                                            int CH, int rx, int ry, int rz, T (&out)[VEC]) {
    const int s = (o >> a) & 1;
    const int dir = 2 * a + (1 - s);  // xi_a > 0: data comes from the low side
    const int n = rec[dir * 4 + 1] >= 0 ? 4 : 1;
    T acc[VEC];
#pragma unroll
    for (int i = 0; i < VEC; i++) acc[i] = T(0);
    for (int k = 0; k < n; k++) {
        const int code = rec[dir * 4 + k];
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
            alignas(16) T v[VEC];
            ld_global_nc<T, VEC>(base + e, v);
#pragma unroll
            for (int i = 0; i < VEC; i++) acc[i] += v[i];
        }
    }
    const T wgt = (n == 4) ? T(0.25) : T(1);
#pragma unroll
    for (int i = 0; i < VEC; i++) out[i] = acc[i] * wgt;
}

template <typename T, int VEC, bool SIMPLE>
__device__ __forceinline__ void transport_pass(const StepParams& p, const Smem& s, int slab, int CH, int CV,
                                               double dth, double (&mom)[5]) {
    const T* __restrict__ fin = reinterpret_cast<const T*>(p.f_in);
    T* sf = reinterpret_cast<T*>(s.slab);
    const int nhx = p.nh[0], nhy = p.nh[1];
    const T* const* sp = reinterpret_cast<const T* const*>(s.ptr);
    for (int v = threadIdx.x; v < CV; v += blockDim.x) {
        const int e = v * VEC;
        const int rx = e % nhx, t2 = e / nhx, ry = t2 % nhy, rz = t2 / nhy;
        // |xi| of this thread's nodes: the same for all 8 octants (symmetric grid, rank order)
        const double ay = __ldg(&p.vel->xi[1][nhy + ry]), az = __ldg(&p.vel->xi[2][p.nh[2] + rz]);
        double ax[VEC];
        T cx[VEC], c0[VEC];
        const T cy = (T)(dth * ay), cz = (T)(dth * az);
#pragma unroll
        for (int i = 0; i < VEC; i++) {
            ax[i] = __ldg(&p.vel->xi[0][nhx + rx + i]);
            cx[i] = (T)(dth * ax[i]);
            c0[i] = (T)(1.0 - dth * (ax[i] + ay + az));
        }
        const double ayz2 = ay * ay + az * az;
#pragma unroll 2
        for (int o = 0; o < 8; o++) {
            alignas(16) T own[VEC], X[VEC], Y[VEC], Z[VEC], fs[VEC];
            if (SIMPLE) {
                ld_global_nc<T, VEC>(sp[o * 4 + 0] + e, own);
                ld_global_nc<T, VEC>(sp[o * 4 + 1] + e, X);
                ld_global_nc<T, VEC>(sp[o * 4 + 2] + e, Y);
                ld_global_nc<T, VEC>(sp[o * 4 + 3] + e, Z);
            } else {
                ld_global_nc<T, VEC>(fin + (int64_t)slab * p.Nv + (int64_t)o * CH + e, own);
                gather_axis<T, VEC>(p, s.rec, fin, 0, o, e, CH, rx, ry, rz, X);
                gather_axis<T, VEC>(p, s.rec, fin, 1, o, e, CH, rx, ry, rz, Y);
                gather_axis<T, VEC>(p, s.rec, fin, 2, o, e, CH, rx, ry, rz, Z);
            }
#pragma unroll
            for (int i = 0; i < VEC; i++) fs[i] = c0[i] * own[i] + cx[i] * X[i] + cy * Y[i] + cz * Z[i];
            st_shared<T, VEC>(sf + o * CH + e, fs);
            if (p.collide) {
                // a2: fp64 accumulation; sums over the vector first, signs and y/z weights once per vector
                double s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
                for (int i = 0; i < VEC; i++) {
                    const double d = (double)fs[i];
                    s0 += d;
                    s1 = fma(ax[i], d, s1);
                    s2 = fma(ax[i] * ax[i], d, s2);
                }
                mom[0] += s0;
                mom[1] += (o & 1) ? s1 : -s1;
                const double sy = ay * s0, sz = az * s0;
                mom[2] += (o & 2) ? sy : -sy;
                mom[3] += (o & 4) ? sz : -sz;
                mom[4] += fma(ayz2, s0, s2);
            }
        }
    }
}

template <typename T, int VEC, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_step_fast(const StepParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nvp = nvp_of(p.nv);
    const Smem s = carve(smem_raw, p.Nv, sizeof(T), nvp, (blockDim.x + 31) >> 5);
    const int slab = blockIdx.x;
    const int tid = threadIdx.x;
    const int CH = p.nh[0] * p.nh[1] * p.nh[2];
    const int CV = CH / VEC;
    if (tid < 32) s.rec[tid] = reinterpret_cast<const int*>(p.cells + slab)[tid];
    __syncthreads();
    const bool simple = (s.rec[25] & CELL_SIMPLE) != 0;
    const T* fin = reinterpret_cast<const T*>(p.f_in);
    if (simple && tid < 32) {
        // chunk pointers per octant: own, and the single upwind source on each axis
        const int o = tid >> 2, k = tid & 3;
        const T* ptr;
        if (k == 0) {
            ptr = fin + (int64_t)slab * p.Nv + (int64_t)o * CH;
        } else {
            const int a = k - 1;
            const int dir = 2 * a + (1 - ((o >> a) & 1));
            const int code = s.rec[dir * 4];
            const int kind = code >> SRC_SHIFT;
            const int64_t idx = code & SRC_INDEX_MASK;
            ptr = (kind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + idx * p.Nv
                  + (int64_t)(kind == SRC_MIRROR ? (o ^ (1 << a)) : o) * CH;
        }
        s.ptr[tid] = ptr;
    }
    __syncthreads();
    const double dth = p.dt * p.inv_len * (double)(1 << s.rec[24]);  // dt / h

    double mom[5] = {0, 0, 0, 0, 0};
    if (simple) transport_pass<T, VEC, true>(p, s, slab, CH, CV, dth, mom);
    else transport_pass<T, VEC, false>(p, s, slab, CH, CV, dth, mom);

    if (p.collide) {
        block_reduce_moments(mom, s, p.w);
        if (tid < 32)
            newton_warp(p.vel, p.nv[0], p.nv[1], p.nv[2], nvp, p.w, p.dt, p.inv_kn, p.visc_exp, p.nu_pref, p.flags,
                        s.red, s.g, s.gf, s.res);
    }
    __syncthreads();

    // a4: relaxation epilogue, one pass over the slab buffer, streaming stores
    const T* sf = reinterpret_cast<const T*>(s.slab);
    T* fout = reinterpret_cast<T*>(p.f_out) + (int64_t)slab * p.Nv;
    if (!p.collide) {
        for (int v = tid; v < CV * 8; v += blockDim.x) {
            alignas(16) T fs[VEC];
            ld_shared<T, VEC>(sf + v * VEC, fs);
            st_global_cs<T, VEC>(fout + v * VEC, fs);
        }
        return;
    }
    const double amp = s.res[0];
    const T omega = (T)s.res[1];
    const int nhx = p.nh[0], nhy = p.nh[1], nhz = p.nh[2];
    for (int v = tid; v < CV; v += blockDim.x) {
        const int e = v * VEC;
        const int rx = e % nhx, t2 = e / nhx, ry = t2 % nhy, rz = t2 / nhy;
#pragma unroll 2
        for (int o = 0; o < 8; o++) {
            alignas(16) T fs[VEC], out[VEC];
            ld_shared<T, VEC>(sf + o * CH + e, fs);
            const int kz = (o & 4) ? nhz + rz : nhz - 1 - rz;
            const int ky = (o & 2) ? nhy + ry : nhy - 1 - ry;
            const int kx0 = (o & 1) ? nhx + rx : nhx - 1 - rx;
            const int kxs = (o & 1) ? 1 : -1;
            const T b = (T)(amp * s.g[2 * nvp + kz] * s.g[nvp + ky]);
#pragma unroll
            for (int i = 0; i < VEC; i++) {
                T gx;
                if (sizeof(T) == 4) gx = (T)s.gf[kx0 + kxs * i];
                else gx = (T)s.g[kx0 + kxs * i];
                const T M = b * gx;
                out[i] = fs[i] + omega * (M - fs[i]);
            }
            st_global_cs<T, VEC>(fout + (int64_t)o * CH + e, out);
        }
    }
}

// ---------------------------------------------------------------- generic per-slot path
// Any velocity grid (odd nv, asymmetric limits): slot -> (kx,ky,kz) through a table, upwind side from
// the sign of xi, zero nodes carry no flux on that axis.
template <typename T, int MAXT>
__global__ void __launch_bounds__(MAXT) k_step_generic(const StepParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nvp = nvp_of(p.nv);
    const Smem s = carve(smem_raw, p.Nv, sizeof(T), nvp, (blockDim.x + 31) >> 5);
    const int slab = blockIdx.x, tid = threadIdx.x;
    if (tid < 32) s.rec[tid] = reinterpret_cast<const int*>(p.cells + slab)[tid];
    __syncthreads();
    const T* __restrict__ fin = reinterpret_cast<const T*>(p.f_in);
    const T* __restrict__ tab = reinterpret_cast<const T*>(p.tables);
    T* sf = reinterpret_cast<T*>(s.slab);
    const double dth = p.dt * p.inv_len * (double)(1 << s.rec[24]);
    const int64_t Nv = p.Nv;
    double mom[5] = {0, 0, 0, 0, 0};
    for (int sl = tid; sl < Nv; sl += blockDim.x) {
        const uchar4 k4 = p.slot_k[sl];
        const int kk[3] = {k4.x, k4.y, k4.z};
        const double own = (double)fin[(int64_t)slab * Nv + sl];
        double xi[3], fs = own;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            xi[a] = p.vel->xi[a][kk[a]];
            if (xi[a] == 0.0) continue;
            const int dir = 2 * a + (xi[a] > 0.0 ? 0 : 1);
            const int n = s.rec[dir * 4 + 1] >= 0 ? 4 : 1;
            double X = 0.0;
            for (int t = 0; t < n; t++) {
                const int code = s.rec[dir * 4 + t];
                const int kind = code >> SRC_SHIFT;
                const int64_t idx = code & SRC_INDEX_MASK;
                if (kind == SRC_SLAB) X += (double)fin[idx * Nv + sl];
                else if (kind == SRC_MIRROR) X += (double)fin[idx * Nv + p.mirror_slot[(int64_t)a * Nv + sl]];
                else if (kind == SRC_TABLE) X += (double)tab[idx * Nv + sl];
                else { const FluidGhost* g = p.fluid + idx; X += g->amp * g->g[2][kk[2]] * g->g[1][kk[1]] * g->g[0][kk[0]]; }
            }
            if (n == 4) X *= 0.25;
            fs += dth * fabs(xi[a]) * (X - own);
        }
        const T fst = (T)fs;
        sf[sl] = fst;
        const double d = (double)fst;
        mom[0] += d; mom[1] += xi[0] * d; mom[2] += xi[1] * d; mom[3] += xi[2] * d;
        mom[4] += (xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2]) * d;
    }
    if (p.collide) {
        block_reduce_moments(mom, s, p.w);
        if (tid < 32)
            newton_warp(p.vel, p.nv[0], p.nv[1], p.nv[2], nvp, p.w, p.dt, p.inv_kn, p.visc_exp, p.nu_pref, p.flags,
                        s.red, s.g, s.gf, s.res);
    }
    __syncthreads();
    T* fout = reinterpret_cast<T*>(p.f_out) + (int64_t)slab * Nv;
    const double amp = p.collide ? s.res[0] : 0.0, omega = p.collide ? s.res[1] : 0.0;
    for (int sl = tid; sl < Nv; sl += blockDim.x) {
        const double fs = (double)sf[sl];
        double out = fs;
        if (p.collide) {
            const uchar4 k4 = p.slot_k[sl];
            const double M = amp * s.g[2 * nvp + k4.z] * s.g[nvp + k4.y] * s.g[k4.x];
            out = fs + omega * (M - fs);
        }
        fout[sl] = (T)out;
    }
}

// ---------------------------------------------------------------- moments of f (S7)
template <typename T>
__global__ void __launch_bounds__(256) k_moments(const StepParams p, const T* __restrict__ f, double* __restrict__ mom) {
    __shared__ double red[8][5];
    const int slab = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const T* fc = f + (int64_t)slab * p.Nv;
    double m[5] = {0, 0, 0, 0, 0};
    for (int sl = tid; sl < p.Nv; sl += blockDim.x) {
        const uchar4 k4 = p.slot_k[sl];
        const double x = p.vel->xi[0][k4.x], y = p.vel->xi[1][k4.y], z = p.vel->xi[2][k4.z];
        const double d = (double)fc[sl];
        m[0] += d; m[1] += x * d; m[2] += y * d; m[3] += z * d; m[4] += (x * x + y * y + z * z) * d;
    }
#pragma unroll
    for (int a = 0; a < 5; a++) m[a] = warp_sum(m[a]);
    if (lane == 0)
        for (int a = 0; a < 5; a++) red[warp][a] = m[a];
    __syncthreads();
    if (tid < 5) {
        double t = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) t += red[w][tid];
        t *= p.w;
        mom[(int64_t)tid * p.n_kin + slab] = (tid == 4) ? 0.5 * t : t;
    }
}

// ---------------------------------------------------------------- launch plumbing
constexpr int FAST_MAXT = 256;
constexpr size_t SMEM_CAP = 227 * 1024;

template <typename K>
cudaError_t set_smem(K kernel, int bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

template <typename T, int VEC>
cudaError_t launch_fast(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    // register budget follows the occupancy the slab buffer allows: 2, 3 or 4 CTAs per SM
    const int per_sm = (int)((228 * 1024) / (plan.smem_bytes + 1024));
    cudaError_t e;
    if (per_sm >= 4) {
        auto k = k_step_fast<T, VEC, FAST_MAXT, 4>;
        if ((e = set_smem(k, plan.smem_bytes)) != cudaSuccess) return e;
        k<<<p.n_kin, plan.threads, plan.smem_bytes, st>>>(p);
    } else if (per_sm == 3) {
        auto k = k_step_fast<T, VEC, FAST_MAXT, 3>;
        if ((e = set_smem(k, plan.smem_bytes)) != cudaSuccess) return e;
        k<<<p.n_kin, plan.threads, plan.smem_bytes, st>>>(p);
    } else {
        auto k = k_step_fast<T, VEC, FAST_MAXT, 2>;
        if ((e = set_smem(k, plan.smem_bytes)) != cudaSuccess) return e;
        k<<<p.n_kin, plan.threads, plan.smem_bytes, st>>>(p);
    }
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_generic(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    auto k = k_step_generic<T, 256>;
    cudaError_t e = set_smem(k, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    k<<<p.n_kin, plan.threads, plan.smem_bytes, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

int step_plan(int storage, const VelLayout& v, StepLaunch* plan, const char** why) {
    const size_t elem = storage == UFS_STORE_F32 ? 4 : 8;
    const int nvp = nvp_of(v.nv);
    plan->ring = 0;
    plan->grid = plan->ncw = plan->pieces = plan->stages = 0;
    plan->fast = v.fast ? 1 : 0;
    plan->vec = 1;
    int threads = 256;
    if (v.fast) {
        const int nhx = v.nh[0];
        if (elem == 4) plan->vec = (nhx % 4 == 0) ? 4 : (nhx % 2 == 0) ? 2 : 1;
        else plan->vec = (nhx % 2 == 0) ? 2 : 1;
        // threads: cover the CV vectors of an octant chunk in 1..4 sweeps with the least idle lanes
        const int CV = v.nh[0] * v.nh[1] * v.nh[2] / plan->vec;
        int best_waste = 1 << 30;
        for (int sweeps = 1; sweeps <= 8; sweeps++) {
            int t = ((CV + sweeps - 1) / sweeps + 31) / 32 * 32;
            if (t > FAST_MAXT || t < 64) { if (t < 64 && sweeps > 1) break; if (t > FAST_MAXT) continue; }
            const int waste = t * sweeps - CV;
            if (waste < best_waste) { best_waste = waste; threads = t; }
        }
    }
    plan->threads = threads;
    const size_t sm = smem_bytes_for(v.Nv, elem, nvp, (threads + 31) / 32);
    if (sm > SMEM_CAP) { *why = "Nv * sizeof(element) does not fit the 227 KB on-chip slab buffer"; return UFS_DVM_EINVAL; }
    plan->smem_bytes = (int32_t)sm;
    return UFS_DVM_OK;
}

cudaError_t launch_step(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    if (plan.ring == 4) return launch_tiles(storage, plan, p, st);
    if (plan.ring == 3) return launch_rows(storage, plan, p, st);
    if (plan.ring == 2) return launch_stream(storage, plan, p, st);
    if (plan.ev0) cudaEventRecord(plan.ev0, st);
    cudaError_t e;
    if (plan.fast) {
        if (storage == UFS_STORE_F32) {
            if (plan.vec == 4) e = launch_fast<float, 4>(plan, p, st);
            else if (plan.vec == 2) e = launch_fast<float, 2>(plan, p, st);
            else e = launch_fast<float, 1>(plan, p, st);
        } else {
            e = plan.vec == 2 ? launch_fast<double, 2>(plan, p, st) : launch_fast<double, 1>(plan, p, st);
        }
    } else {
        e = storage == UFS_STORE_F32 ? launch_generic<float>(plan, p, st) : launch_generic<double>(plan, p, st);
    }
    if (plan.ev1) cudaEventRecord(plan.ev1, st);
    return e;
}

cudaError_t launch_moments(int storage, const StepParams& p, const void* f, double* mom, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    if (storage == UFS_STORE_F32) k_moments<float><<<p.n_kin, 256, 0, st>>>(p, reinterpret_cast<const float*>(f), mom);
    else k_moments<double><<<p.n_kin, 256, 0, st>>>(p, reinterpret_cast<const double*>(f), mom);
    return cudaGetLastError();
}

}  // namespace ufs
