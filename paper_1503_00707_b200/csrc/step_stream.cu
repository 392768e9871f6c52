// step_stream.cu -- the single-pass streaming DVM step, sm_100a.
//
// Idea.  Transport (Eq. 2) is linear in f, so the five moments of f* of a cell are a linear
// combination of velocity sums of the OLD f of the cell and of its upwind neighbours:
//     rho*_j = H_j - (dt/h_j) sum_{a,s} G_j[a][s] + (dt/h_j) sum_{a,s} wgt * G_src(j,a,s)[a][s]
// with, per cell,  H = sum_i m(xi_i) f_i  and  G[a][s] = sum_{i: sign(xi_a,i) = s} m(xi_i) |xi_a,i| f_i
// (m = 1, xi, |xi|^2; 35 fp64 numbers).  These sums are produced for f^{n+1} by the pass that writes
// f^{n+1}, so a step is
//   k_prep   : per cell (8 lanes each), rho* from the stored sums -> Newton for the discrete Maxwellian (the per-cell 5x5
//              problem of PAPER.md:145-163, 179, separable form) -> factor table + dt*nu;   (~1 KB per cell)
//   k_stream : per cell and velocity octant (sign group), four contiguous streams (own chunk
//              + one upwind chunk per axis) arrive through a TMA ring (cp.async.bulk + mbarrier), and each
//              value is finished in registers:  f* = c0 f + cx fX + cy fY + cz fZ,  f' = f* + dt nu (M - f*)
//              (BGK), stored once, and folded into the cell's sums for the next step (fp64).
// f crosses HBM once in and once out; nothing of a cell is parked on chip, no block-wide barrier sits between
// the load and the store, and the Newton solve is off the streaming path.
// Cells with a 2:1 face towards finer neighbours or a kinetic/fluid face gather their sources
// with plain vector loads instead of the ring.
#include <cmath>

#include "device_util.cuh"
#include "kernels.cuh"
#include "stream_common.cuh"

namespace ufs {
namespace {

enum { ST_RING = 0, ST_GATHER = 1, ST_STOP = 2 };
constexpr int RED_SLOTS = 2;   // per-warp partial sums of the last two cells

// ---------------------------------------------------------------- per-thread velocity constants
// A thread keeps the same |xi| on every axis for all 8 octants (symmetric grid, slots ordered by increasing
// |xi| inside an octant): only the signs change.
template <typename T>
struct Pos {
    static constexpr int VEC = V16<T>::N;
    double ax[VEC], ax2[VEC], ay, az, r2;  // |xi_x| of the VEC nodes, squares, |xi_y|, |xi_z|, ay^2 + az^2
    int rx, ry, rz;                        // rank of |xi| on each axis (rx: first of VEC)
};
template <typename T>
__device__ __forceinline__ Pos<T> pos_of(const StepParams& p, int v) {
    constexpr int VEC = V16<T>::N;
    Pos<T> c;
    const int e = v * VEC;
    c.rx = e % p.nh[0];
    const int row = e / p.nh[0];
    c.ry = row % p.nh[1];
    c.rz = row / p.nh[1];
#pragma unroll
    for (int i = 0; i < VEC; i++) {
        c.ax[i] = __ldg(&p.vel->xi[0][p.nh[0] + c.rx + i]);
        c.ax2[i] = c.ax[i] * c.ax[i];
    }
    c.ay = __ldg(&p.vel->xi[1][p.nh[1] + c.ry]);
    c.az = __ldg(&p.vel->xi[2][p.nh[2] + c.rz]);
    c.r2 = fma(c.ay, c.ay, c.az * c.az);
    return c;
}

// a2': fold one vector of the new f (octant O) into the thread's 35 partial sums.  Four sums along the x run
// (1, |xi_x|, xi_x^2, |xi_x|^3 weights), then the y/z weights and the signs once per vector.
template <typename T, int O>
__device__ __forceinline__ void add_sums(const T (&f)[V16<T>::N], const Pos<T>& c, double (&acc)[35]) {
    constexpr int SX = O & 1, SY = (O >> 1) & 1, SZ = (O >> 2) & 1;
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
#pragma unroll
    for (int i = 0; i < V16<T>::N; i++) {
        const double d = (double)f[i];
        const double t = c.ax[i] * d;
        s0 += d;
        s1 += t;
        s2 = fma(c.ax2[i], d, s2);
        s3 = fma(c.ax2[i], t, s3);
    }
    double h[5], g[5];
    h[0] = s0;
    h[1] = SX ? s1 : -s1;
    h[2] = (SY ? c.ay : -c.ay) * s0;
    h[3] = (SZ ? c.az : -c.az) * s0;
    h[4] = fma(c.r2, s0, s2);
    g[0] = s1;
    g[1] = SX ? s2 : -s2;
    g[2] = (SY ? c.ay : -c.ay) * s1;
    g[3] = (SZ ? c.az : -c.az) * s1;
    g[4] = fma(c.r2, s1, s3);
#pragma unroll
    for (int k = 0; k < 5; k++) {
        acc[k] += h[k];
        acc[g_index(0, SX, k)] += g[k];
        acc[g_index(1, SY, k)] = fma(c.ay, h[k], acc[g_index(1, SY, k)]);
        acc[g_index(2, SZ, k)] = fma(c.az, h[k], acc[g_index(2, SZ, k)]);
    }
}

// ---------------------------------------------------------------- k_prep: rho* and the discrete Maxwellian (a2, a3)
// 1/x to about one ulp: hardware seed (20 bits) + two Newton steps
__device__ __forceinline__ double frcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}
template <typename T> struct SeriesTol;   // residual below which one more (series) update ends the solve
template <> struct SeriesTol<double> { static constexpr double value = 1e-7; };   // error after it ~1e-14
template <> struct SeriesTol<float> { static constexpr double value = 1e-4; };    // ~1e-8 << fp32 storage rounding

// Solve  w sum_i m(xi_i) exp(alpha . m(xi_i)) = rho, eight lanes per cell (four cells per warp).
// exp(alpha.m) = A gx gy gz, g_b[k] = exp(alpha_b xi_k + alpha_4 xi_k^2).  With the 1-D power sums
// P_b^r = sum_k xi_k^r g_b[k] the five equations read  P_b^1/P_b^0 = u_b,  sum_b P_b^2/P_b^0 = rho_4/n,
// A w Px^0 Py^0 Pz^0 = n: an arrow-shaped 4x4 Newton system (closed-form Schur complement) plus the amplitude.  Same
// root as a 5x5 Newton on alpha (the solution is unique).  Stop: scaled residual <= 1e-13, or one more update after a
// residual <= SeriesTol (quadratic convergence), that update applied to g through its series.  Lane sl of a group holds
// nodes sl, sl + 8, sl + 16, sl + 24 of every axis (nv <= 32).
constexpr int PREP_NPL = 4;  // nodes per lane and axis
__device__ __forceinline__ double group_sum(double v) {  // over the 8 lanes of a cell
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// four kinetic cells per warp
template <typename T>
__global__ void __launch_bounds__(256, 3) k_prep(const StepParams p) {
    const int lane = threadIdx.x & 31, sl = lane & 7;
    const int cell_raw = (blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 4 + (lane >> 3);
    const bool valid = cell_raw < p.n_kin;
    const int cell = valid ? cell_raw : 0;
    const int* rec = reinterpret_cast<const int*>(p.cells + cell);
    const double* S = p.sums_in + (int64_t)cell * SUMS_STRIDE;
    const int level = __ldg(rec + 24);
    const double dth = p.dt * p.inv_len * (double)(1 << level);
    // pair (d, k): net gain of moment k through direction d = 2*axis + side, in units of dt/h; a lane takes pairs
    // sl, sl + 8, ... of the 30
    double part[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (int idx = sl; idx < 30; idx += 8) {
        const int d = idx / 5, k = idx % 5, a = d >> 1, side = d & 1, sin = 1 - side;
        const int nsrc = __ldg(rec + d * 4 + 1) >= 0 ? 4 : 1;
        double in = 0.0;
        for (int j = 0; j < nsrc; j++) {
            const int code = __ldg(rec + d * 4 + j);
            const int kind = code >> SRC_SHIFT;
            const int64_t idx2 = code & SRC_INDEX_MASK;
            double v;
            if (kind == SRC_SLAB) v = p.sums_in[idx2 * SUMS_STRIDE + g_index(a, sin, k)];
            else if (kind == SRC_MIRROR) v = (k == 1 + a ? -1.0 : 1.0) * S[g_index(a, 1 - sin, k)];
            else v = p.ghost_sums[(kind == SRC_TABLE ? idx2 : p.n_tables + idx2) * SUMS_STRIDE + g_index(a, sin, k)];
            in += v;
        }
        const double contrib = (nsrc == 4 ? 0.25 : 1.0) * in - S[g_index(a, side, k)];
#pragma unroll
        for (int kk = 0; kk < 5; kk++) part[kk] += kk == k ? contrib : 0.0;
    }
    double rho[5];
#pragma unroll
    for (int k = 0; k < 5; k++) rho[k] = p.w * fma(dth, group_sum(part[k]), S[k]);

    const int nhp = nhp_of(p.nh);
    const double n = rho[0];
    const double inv_n = frcp(n);
    const double u[3] = {rho[1] * inv_n, rho[2] * inv_n, rho[3] * inv_n};
    const double e2 = rho[4] * inv_n;
    const double T0 = (e2 - (u[0] * u[0] + u[1] * u[1] + u[2] * u[2])) * (1.0 / 3.0);
    bool ok = valid && (n > 0.0) && (T0 > 0.0);
    const double sqT = sqrt(ok ? T0 : 1.0);
    const double isc[4] = {frcp(sqT + fabs(u[0])), frcp(sqT + fabs(u[1])), frcp(sqT + fabs(u[2])), frcp(e2)};
    const double invT = frcp(T0);
    double al[4] = {u[0] * invT, u[1] * invT, u[2] * invT, -0.5 * invT};
    double g[3][PREP_NPL], P0f[3] = {1.0, 1.0, 1.0};
#pragma unroll
    for (int b = 0; b < 3; b++)
#pragma unroll
        for (int j = 0; j < PREP_NPL; j++) g[b][j] = 0.0;
    bool done = false;
    for (int it = 0; it <= 50; it++) {
        const bool act = ok && !done;
        if (!__any_sync(0xffffffffu, act)) break;
        double P[3][5];
#pragma unroll
        for (int b = 0; b < 3; b++) {
            double ps[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int j = 0; j < PREP_NPL; j++) {
                const int node = sl + 8 * j;
                if (act && node < p.nv[b]) {
                    const double x = p.vel->xi[b][node];
                    double t = exp((al[b] + al[3] * x) * x);
                    g[b][j] = t;
#pragma unroll
                    for (int r = 0; r < 5; r++) { ps[r] += t; t *= x; }
                }
            }
#pragma unroll
            for (int r = 0; r < 5; r++) P[b][r] = group_sum(ps[r]);
        }
        if (!act) continue;
        double m1[3], m2[3], i0[3], r[4];
        r[3] = -e2;
#pragma unroll
        for (int b = 0; b < 3; b++) {
            i0[b] = frcp(P[b][0]);
            m1[b] = P[b][1] * i0[b]; m2[b] = P[b][2] * i0[b];
            r[b] = m1[b] - u[b];
            r[3] += m2[b];
        }
        double res = 0.0;
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const double q = fabs(r[k]) * isc[k];
            if (!(q <= res)) res = q;  // NaN propagates
        }
        if (res <= 1e-13) {
#pragma unroll
            for (int b = 0; b < 3; b++) P0f[b] = P[b][0];
            done = true;
            continue;
        }
        if (!(res == res) || it == 50) { ok = false; continue; }
        // arrow system: var_b d_b + c_b d_4 = -r_b ;  sum_b c_b d_b + dd d_4 = -r_4
        double iv[3], cb[3], num = r[3], dd = 0.0, schur = 0.0;
#pragma unroll
        for (int b = 0; b < 3; b++) {
            const double m3 = P[b][3] * i0[b], m4 = P[b][4] * i0[b];
            iv[b] = frcp(m2[b] - m1[b] * m1[b]);
            cb[b] = m3 - m1[b] * m2[b];
            dd += m4 - m2[b] * m2[b];
            schur += cb[b] * cb[b] * iv[b];
            num -= cb[b] * r[b] * iv[b];
        }
        double dl[4];
        dl[3] = -num * frcp(dd - schur);
#pragma unroll
        for (int b = 0; b < 3; b++) dl[b] = -(r[b] + cb[b] * dl[3]) * iv[b];
#pragma unroll
        for (int k = 0; k < 4; k++) al[k] += dl[k];
        if (res <= SeriesTol<T>::value) {
            // the update is small: apply it to g and to the zeroth power sums by expansion
#pragma unroll
            for (int b = 0; b < 3; b++) {
#pragma unroll
                for (int j = 0; j < PREP_NPL; j++) {
                    const int node = sl + 8 * j;
                    if (node < p.nv[b]) {
                        const double x = p.vel->xi[b][node];
                        const double z = (dl[b] + dl[3] * x) * x;
                        g[b][j] *= 1.0 + z * (1.0 + z * (0.5 + z * (1.0 / 6.0)));
                    }
                }
                P0f[b] = P[b][0] + dl[b] * P[b][1] + dl[3] * P[b][2]
                         + 0.5 * (dl[b] * dl[b] * P[b][2] + 2.0 * dl[b] * dl[3] * P[b][3] + dl[3] * dl[3] * P[b][4]);
            }
            done = true;
        }
    }
    if (!valid) return;
    double amp = 0.0, omega = 0.0;
    if (done) {
        amp = n * frcp(p.w * P0f[0] * P0f[1] * P0f[2]);
        // G9: nu = c_nu n T^(1-omega) / Kn (omega = 1/2: sqrt)
        const double Tp = (p.visc_exp == 0.5) ? sqT : pow(T0, 1.0 - p.visc_exp);
        omega = p.dt * p.nu_pref * n * Tp * p.inv_kn;
    } else if (sl == 0) {
        atomicOr(p.flags, 1);  // no Maxwellian: f* passes through unchanged (UFS_DVM_ENEWTON)
    }
    // table layout: stream_common.cuh
    T* tab = reinterpret_cast<T*>(p.tabs) + (int64_t)cell * tabn_of(p.nh);
#pragma unroll
    for (int b = 0; b < 3; b++) {
#pragma unroll
        for (int j = 0; j < PREP_NPL; j++) {
            const int node = sl + 8 * j;
            if (node < p.nv[b]) {
                const int s = node >= p.nh[b] ? 1 : 0;
                const int rk = s ? node - p.nh[b] : p.nh[b] - 1 - node;
                tab[(2 * b + s) * nhp + rk] = done ? (T)(b == 2 ? g[b][j] * amp : g[b][j]) : T(0);
            }
        }
    }
    if (sl == 0) tab[6 * nhp] = (T)omega;
}

// moments of the current f from its stored sums: mom[5][n_kin] = (n, n u, E = rho_4 / 2)
__global__ void k_moments_from_sums(const StepParams p, const double* __restrict__ sums, double* __restrict__ mom) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)p.n_kin * 5) return;
    const int64_t cell = i / 5;
    const int k = (int)(i % 5);
    mom[(int64_t)k * p.n_kin + cell] = (k == 4 ? 0.5 : 1.0) * p.w * sums[cell * SUMS_STRIDE + k];
}

// ---------------------------------------------------------------- k_stream
// Shared memory of a CTA: the ring (NS slots of 4 pieces + room for the factor table that travels with the first
// stage of a cell), mbarriers, stage headers, RED_SLOTS x NCW x SUMS_STRIDE partial sums.
template <typename T>
struct StreamSmem {
    unsigned char* ring;  // [NS][slot_bytes]: 4 pieces, then the table
    double* red;          // [RED_SLOTS][NCW][SUMS_STRIDE]
    uint64_t* full;       // [NS]
    uint64_t* empty;      // [NS]
    uint64_t* rfull;      // [RED_SLOTS]
    uint64_t* rempty;     // [RED_SLOTS]
    int4* info;           // [NS] cell, level, kind, -
    int* rcell;           // [RED_SLOTS]
};
__host__ __device__ inline size_t stream_slot_bytes(size_t elem, size_t stage_bytes, int tabn) {
    return (stage_bytes + (size_t)tabn * elem + 127) & ~(size_t)127;
}
__host__ __device__ inline size_t stream_smem_bytes(size_t elem, int ns, size_t stage_bytes, int ncw, int tabn) {
    size_t b = (size_t)ns * stream_slot_bytes(elem, stage_bytes, tabn);
    b += (size_t)RED_SLOTS * ncw * SUMS_STRIDE * 8;
    b += (size_t)ns * (8 + 8 + 16) + RED_SLOTS * (8 + 8 + 4) + 16;
    return (b + 127) & ~(size_t)127;
}
template <typename T>
__device__ __forceinline__ StreamSmem<T> stream_carve(unsigned char* base, int ns, size_t stage_bytes, int ncw, int tabn) {
    StreamSmem<T> s;
    size_t off = 0;
    s.ring = base; off += (size_t)ns * stream_slot_bytes(sizeof(T), stage_bytes, tabn);
    s.red = reinterpret_cast<double*>(base + off); off += (size_t)RED_SLOTS * ncw * SUMS_STRIDE * 8;
    s.full = reinterpret_cast<uint64_t*>(base + off); off += (size_t)ns * 8;
    s.empty = reinterpret_cast<uint64_t*>(base + off); off += (size_t)ns * 8;
    s.rfull = reinterpret_cast<uint64_t*>(base + off); off += RED_SLOTS * 8;
    s.rempty = reinterpret_cast<uint64_t*>(base + off); off += RED_SLOTS * 8;
    s.info = reinterpret_cast<int4*>(base + off); off += (size_t)ns * 16;
    s.rcell = reinterpret_cast<int*>(base + off);
    return s;
}

// everything a consumer thread needs to finish the vectors of one cell
template <typename T, int PIECES>
struct CellCtx {
    T cx[PIECES][V16<T>::N], cy[PIECES], cz[PIECES], c0[PIECES][V16<T>::N];  // update coefficients (level of the cell)
    T gx[PIECES][2][V16<T>::N];       // Maxwellian factors of the thread's |xi_x| ranks for either sign
    T gy[PIECES][2], gz[PIECES][2];   // ... of its |xi_y|, |xi_z| (gz carries the amplitude)
    T omega;                          // dt * nu
};

// a1 + a4 + a2' for one vector: transport, relaxation, store, fold into the sums
template <typename T, int O, int PIECES>
__device__ __forceinline__ void finish_vec(const StepParams& p, const CellCtx<T, PIECES>& cc, int q, const Pos<T>& c, int nhp,
                                           const T (&own)[V16<T>::N], const T (&X)[V16<T>::N], const T (&Y)[V16<T>::N],
                                           const T (&Z)[V16<T>::N], T* gdst, double (&acc)[35]) {
    constexpr int VEC = V16<T>::N;
    T out[VEC];
#pragma unroll
    for (int i = 0; i < VEC; i++)
        out[i] = cc.c0[q][i] * own[i] + cc.cx[q][i] * X[i] + cc.cy[q] * Y[i] + cc.cz[q] * Z[i];
    if (p.collide) {
        const T b = cc.gz[q][(O >> 2) & 1] * cc.gy[q][(O >> 1) & 1];
#pragma unroll
        for (int i = 0; i < VEC; i++) {
            const T M = b * cc.gx[q][O & 1][i];
            out[i] = out[i] + cc.omega * (M - out[i]);
        }
    }
    stg16_cs(gdst, out);
    add_sums<T, O>(out, c, acc);
}

template <typename T, int O, int PIECES>
__device__ __forceinline__ void octant_from_ring(const StepParams& p, const StreamSmem<T>& s, const CellCtx<T, PIECES>& cc,
                                                 const Pos<T> (&pos)[PIECES], int nhp, int PV, int CH, bool active, int tid,
                                                 int lane, T* gout, double (&acc)[35], int& slot, uint32_t& ph, int NS,
                                                 uint32_t slot_bytes) {
    constexpr int VEC = V16<T>::N;
#pragma unroll
    for (int q = 0; q < PIECES; q++) {
        if (O + q > 0) mbar_wait(&s.full[slot], ph);
        const int pe = PV * VEC;  // elements per piece
        const int mask = s.info[slot].w;  // axes whose upwind face has four finer sources (reading G3); warp-uniform
        T* const st = reinterpret_cast<T*>(s.ring + (size_t)slot * slot_bytes + (size_t)tid * 16);
        if (mask) {
            // The next three slots bring sources 1..3 of those axes (piece t = axis t).  They are added, in order,
            // onto source 0 where it lies in this slot (each thread touches only its own 16 bytes), so the common
            // path below needs no extra registers.
            int sl = slot;
            uint32_t sp = ph;
#pragma unroll 1
            for (int j = 1; j < 4; j++) {
                if (++sl == NS) { sl = 0; sp ^= 1u; }
                mbar_wait(&s.full[sl], sp);
                if (active) {
                    const T* se = reinterpret_cast<const T*>(s.ring + (size_t)sl * slot_bytes + (size_t)tid * 16);
#pragma unroll 1
                    for (int t = 0; t < 3; t++) {
                        if ((mask >> t) & 1) {
                            T v[VEC], x[VEC];
                            lds16(se + t * pe, v);
                            lds16(st + (t + 1) * pe, x);
#pragma unroll
                            for (int i = 0; i < VEC; i++) x[i] += v[i];
                            sts16(st + (t + 1) * pe, x);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&s.empty[sl]);
            }
        }
        T own[VEC], X[VEC], Y[VEC], Z[VEC];
        if (active) {
            lds16(st, own);
            lds16(st + pe, X);
            lds16(st + 2 * pe, Y);
            lds16(st + 3 * pe, Z);
            if (mask) {  // each of the four sources weighs 1/4
#pragma unroll
                for (int i = 0; i < VEC; i++) {
                    if (mask & 1) X[i] *= T(0.25);
                    if (mask & 2) Y[i] *= T(0.25);
                    if (mask & 4) Z[i] *= T(0.25);
                }
            }
            finish_vec<T, O, PIECES>(p, cc, q, pos[q], nhp, own, X, Y, Z, gout + O * CH + q * pe, acc);
        }
        // this slot was written with ordinary stores: order them before the bulk copy that refills it
        if (mask) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&s.empty[slot]);
        if (++slot == NS) { slot = 0; ph ^= 1u; }
        if (mask) {  // step over the three slots consumed above
#pragma unroll 1
            for (int j = 1; j < 4; j++) if (++slot == NS) { slot = 0; ph ^= 1u; }
        }
    }
}

template <typename T, int O, int PIECES>
__device__ __forceinline__ void octant_from_gather(const StepParams& p, const CellCtx<T, PIECES>& cc, const Pos<T> (&pos)[PIECES],
                                                   int nhp, int PV, int CH, int tid, const int* rec, const T* fin,
                                                   const T* own_base, T* gout, double (&acc)[35]) {
    constexpr int VEC = V16<T>::N;
#pragma unroll
    for (int q = 0; q < PIECES; q++) {
        const int pe = PV * VEC;
        const int e = q * pe + tid * VEC;
        T own[VEC], X[VEC], Y[VEC], Z[VEC];
        ldg16(own_base + O * CH + q * pe, own);
        gather_axis<T>(p, rec, fin, 0, O, CH, e, pos[q].rx, pos[q].ry, pos[q].rz, X);
        gather_axis<T>(p, rec, fin, 1, O, CH, e, pos[q].rx, pos[q].ry, pos[q].rz, Y);
        gather_axis<T>(p, rec, fin, 2, O, CH, e, pos[q].rx, pos[q].ry, pos[q].rz, Z);
        finish_vec<T, O, PIECES>(p, cc, q, pos[q], nhp, own, X, Y, Z, gout + O * CH + q * pe, acc);
    }
}

// Warp roles: NCW consumer warps, one producer warp (index NCW), one finisher warp (index NCW + 1).
template <typename T, int NCW, int PIECES>
__global__ void __launch_bounds__((NCW + 2) * 32, 1) k_stream(const StepParams p) {
    constexpr int VEC = V16<T>::N;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nhp = nhp_of(p.nh), tabn = tabn_of(p.nh);
    const int CH = p.nh[0] * p.nh[1] * p.nh[2];
    const int PV = CH / VEC / PIECES;  // 16-byte vectors per piece and stream
    const uint32_t piece_bytes = (uint32_t)PV * 16u;
    const uint32_t stage_bytes = 4u * piece_bytes;
    const uint32_t tab_bytes = (uint32_t)tabn * (uint32_t)sizeof(T);
    const uint32_t slot_bytes = (uint32_t)stream_slot_bytes(sizeof(T), stage_bytes, tabn);
    const int NS = p.ring_stages;
    const StreamSmem<T> s = stream_carve<T>(smem_raw, NS, stage_bytes, NCW, tabn);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int i = 0; i < NS; i++) { mbar_init(&s.full[i], 1); mbar_init(&s.empty[i], NCW); }
        for (int i = 0; i < RED_SLOTS; i++) { mbar_init(&s.rfull[i], NCW); mbar_init(&s.rempty[i], 1); }
        mbar_init_fence();
        if (blockIdx.x == 0) *p.counter_reset = 0;  // the other launch parity's cell counter
    }
    __syncthreads();
    const T* fin = reinterpret_cast<const T*>(p.f_in);
    int slot = 0;
    uint32_t ph = 0;
    auto advance = [&]() { if (++slot == NS) { slot = 0; ph ^= 1u; } };

    if (warp == NCW) {
        // ------------------------------------------------ producer warp: cell tickets, TMA copies
        auto fetch_async = [&]() -> int { return lane == 0 ? atomicAdd(p.counter, 1) : 0; };
        auto load_rec = [&](int cell) -> int {
            return cell < p.n_kin ? __ldg(reinterpret_cast<const int*>(p.cells + cell) + lane) : 0;
        };
        int cur = __shfl_sync(0xffffffffu, fetch_async(), 0);
        int rec = load_rec(cur);
        int nxt_raw = 0;
        const int o_l = lane >> 2, t_l = lane & 3;
        while (true) {
            if (cur >= p.n_kin) {
                mbar_wait(&s.empty[slot], ph ^ 1u);
                if (lane == 0) { s.info[slot] = make_int4(0, 0, ST_STOP, 0); mbar_arrive(&s.full[slot]); }
                break;
            }
            const int level = __shfl_sync(0xffffffffu, rec, 24), flags = __shfl_sync(0xffffffffu, rec, 25);
            const bool ringable = (flags & CELL_NOFLUID) != 0;
            // bit d: direction d has four (finer) sources instead of one
            int four = 0;
#pragma unroll
            for (int d = 0; d < 6; d++) four |= (__shfl_sync(0xffffffffu, rec, d * 4 + 1) >= 0 ? 1 : 0) << d;
            // the first stage of a cell also carries its factor table (behind the four pieces of the slot)
            void* tab_dst = s.ring + (size_t)slot * slot_bytes + stage_bytes;
            const T* tab_src = reinterpret_cast<const T*>(p.tabs) + (int64_t)cur * tabn;
            const uint32_t extra = p.collide ? tab_bytes : 0u;
            if (ringable) {
                // lane (o,t): stream t of octant o -- t = 0 own chunk, t = 1..3 the upwind chunk on axis t-1
                const int a = t_l > 0 ? t_l - 1 : 0;
                const int dir = 2 * a + (1 - ((o_l >> a) & 1));
                const int code = __shfl_sync(0xffffffffu, rec, dir * 4);
                const int kind = code >> SRC_SHIFT;
                const int64_t idx = code & SRC_INDEX_MASK;
                const T* ptr = (t_l == 0) ? fin + (int64_t)cur * p.Nv + (int64_t)o_l * CH
                                          : (kind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + idx * p.Nv
                                                + (int64_t)(kind == SRC_MIRROR ? (o_l ^ (1 << a)) : o_l) * CH;
                for (int o = 0; o < 8; o++) {
                    // the next ticket is drawn late, so that the cells in flight stay consecutive in slab order
                    if (o == 7) nxt_raw = fetch_async();
                    // axes whose upwind face of this octant has four finer sources: sources 1..3 follow in three
                    // more slots (piece t = axis t)
                    int mask = 0;
#pragma unroll
                    for (int b = 0; b < 3; b++) mask |= ((four >> (2 * b + (1 - ((o >> b) & 1)))) & 1) << b;
                    const int xdir = lane < 3 ? 2 * lane + (1 - ((o >> lane) & 1)) : 0;
#pragma unroll
                    for (int q = 0; q < PIECES; q++) {
                        const bool first = (o + q) == 0;
                        mbar_wait(&s.empty[slot], ph ^ 1u);
                        if (lane == 0) {
                            s.info[slot] = make_int4(cur, level, ST_RING, mask);
                            mbar_arrive_expect_tx(&s.full[slot], stage_bytes + (first ? extra : 0u));
                            if (first && extra) bulk_g2s(tab_dst, tab_src, tab_bytes, &s.full[slot]);
                        }
                        __syncwarp();
                        if (o_l == o) {
                            void* dst = s.ring + (size_t)slot * slot_bytes + (size_t)t_l * piece_bytes;
                            bulk_g2s(dst, ptr + (size_t)q * PV * VEC, piece_bytes, &s.full[slot]);
                        }
                        advance();
                        if (mask) {
#pragma unroll 1
                            for (int j = 1; j < 4; j++) {
                                const int xcode = __shfl_sync(0xffffffffu, rec, xdir * 4 + j);
                                mbar_wait(&s.empty[slot], ph ^ 1u);
                                if (lane == 0) {
                                    s.info[slot] = make_int4(cur, level, ST_RING, mask);
                                    mbar_arrive_expect_tx(&s.full[slot], (uint32_t)__popc(mask) * piece_bytes);
                                }
                                __syncwarp();
                                if (lane < 3 && ((mask >> lane) & 1)) {
                                    const int xkind = xcode >> SRC_SHIFT;
                                    const int64_t xidx = xcode & SRC_INDEX_MASK;
                                    const T* xptr = (xkind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + xidx * p.Nv
                                                    + (int64_t)(xkind == SRC_MIRROR ? (o ^ (1 << lane)) : o) * CH;
                                    void* dst = s.ring + (size_t)slot * slot_bytes + (size_t)lane * piece_bytes;
                                    bulk_g2s(dst, xptr + (size_t)q * PV * VEC, piece_bytes, &s.full[slot]);
                                }
                                advance();
                            }
                        }
                    }
                }
            } else {
                nxt_raw = fetch_async();
                mbar_wait(&s.empty[slot], ph ^ 1u);
                if (lane == 0) {
                    s.info[slot] = make_int4(cur, level, ST_GATHER, 0);
                    if (extra) {
                        mbar_arrive_expect_tx(&s.full[slot], extra);
                        bulk_g2s(tab_dst, tab_src, tab_bytes, &s.full[slot]);
                    } else {
                        mbar_arrive(&s.full[slot]);
                    }
                }
                advance();
            }
            cur = __shfl_sync(0xffffffffu, nxt_raw, 0);
            rec = load_rec(cur);
        }
        return;
    }

    if (warp == NCW + 1) {
        // ------------------------------------------------ finisher warp: per-cell sums of the new f
        for (int k = 0;; k++) {
            const int rs = k % RED_SLOTS;
            mbar_wait(&s.rfull[rs], (uint32_t)((k / RED_SLOTS) & 1));
            const int cell = s.rcell[rs];
            if (cell < 0) break;
            if (lane < SUMS_STRIDE / 2) {
                // lane handles two adjacent entries (16-byte accesses)
                double2 t = make_double2(0.0, 0.0);
                const double2* src = reinterpret_cast<const double2*>(s.red + (size_t)rs * NCW * SUMS_STRIDE) + lane;
#pragma unroll
                for (int w = 0; w < NCW; w++) {
                    const double2 v = src[w * (SUMS_STRIDE / 2)];
                    t.x += v.x; t.y += v.y;
                }
                reinterpret_cast<double2*>(p.sums_out + (int64_t)cell * SUMS_STRIDE)[lane] = t;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&s.rempty[rs]);
        }
        return;
    }

    // ---------------------------------------------------- consumer warps
    const bool active = tid < PV;
    Pos<T> pos[PIECES];
#pragma unroll
    for (int q = 0; q < PIECES; q++) pos[q] = pos_of<T>(p, active ? q * PV + tid : 0);
    for (int k = 0;; k++) {
        mbar_wait(&s.full[slot], ph);
        const int4 inf = s.info[slot];
        const int rs = k % RED_SLOTS;
        double* red = s.red + ((size_t)rs * NCW + warp) * SUMS_STRIDE;
        if (inf.z == ST_STOP) {
            if (k >= RED_SLOTS) mbar_wait(&s.rempty[rs], (uint32_t)(((k / RED_SLOTS) - 1) & 1));
            if (warp == 0 && lane == 0) s.rcell[rs] = -1;
            __syncwarp();
            if (lane == 0) mbar_arrive(&s.rfull[rs]);
            break;
        }
        const int cell = inf.x;
        const double dth = p.dt * p.inv_len * (double)(1 << inf.y);  // dt / h
        CellCtx<T, PIECES> cc;
        // the table sits in the slot of the cell's first stage: copy what this thread needs before releasing it
        const T* tab = reinterpret_cast<const T*>(s.ring + (size_t)slot * slot_bytes + stage_bytes);
        cc.omega = p.collide ? tab[6 * nhp] : T(0);
#pragma unroll
        for (int q = 0; q < PIECES; q++) {
            cc.cy[q] = (T)(dth * pos[q].ay);
            cc.cz[q] = (T)(dth * pos[q].az);
#pragma unroll
            for (int i = 0; i < VEC; i++) {
                cc.cx[q][i] = (T)(dth * pos[q].ax[i]);
                cc.c0[q][i] = (T)(1.0 - dth * (pos[q].ax[i] + pos[q].ay + pos[q].az));
            }
#pragma unroll
            for (int sg = 0; sg < 2; sg++) {
                cc.gy[q][sg] = p.collide ? tab[(2 + sg) * nhp + pos[q].ry] : T(0);
                cc.gz[q][sg] = p.collide ? tab[(4 + sg) * nhp + pos[q].rz] : T(0);
                if (p.collide) lds16(tab + sg * nhp + pos[q].rx, cc.gx[q][sg]);
            }
        }
        T* const gout = reinterpret_cast<T*>(p.f_out) + (int64_t)cell * p.Nv + (size_t)tid * VEC;
        double acc[35];
#pragma unroll
        for (int i = 0; i < 35; i++) acc[i] = 0.0;
        if (inf.z == ST_RING) {
#define UFS_OCT(O) octant_from_ring<T, O, PIECES>(p, s, cc, pos, nhp, PV, CH, active, tid, lane, gout, acc, slot, ph, NS, slot_bytes);
            UFS_OCT(0) UFS_OCT(1) UFS_OCT(2) UFS_OCT(3) UFS_OCT(4) UFS_OCT(5) UFS_OCT(6) UFS_OCT(7)
#undef UFS_OCT
        } else {
            // the ring carries only the cell header (and the table): gather with plain loads
            __syncwarp();
            if (lane == 0) mbar_arrive(&s.empty[slot]);
            advance();
            if (active) {
                const int* rec = reinterpret_cast<const int*>(p.cells + cell);
                const T* own_base = fin + (int64_t)cell * p.Nv + (size_t)tid * VEC;
#define UFS_OCT(O) octant_from_gather<T, O, PIECES>(p, cc, pos, nhp, PV, CH, tid, rec, fin, own_base, gout, acc);
                UFS_OCT(0) UFS_OCT(1) UFS_OCT(2) UFS_OCT(3) UFS_OCT(4) UFS_OCT(5) UFS_OCT(6) UFS_OCT(7)
#undef UFS_OCT
            }
        }
        // the warp's partial sums of f' go to the finisher warp
        if (k >= RED_SLOTS) mbar_wait(&s.rempty[rs], (uint32_t)(((k / RED_SLOTS) - 1) & 1));
        warp_store_sums(acc, red, lane);
        if (warp == 0 && lane == 0) s.rcell[rs] = cell;
        __syncwarp();
        if (lane == 0) mbar_arrive(&s.rfull[rs]);
    }
}

// ---------------------------------------------------------------- k_sums: the sums of an f nobody summed yet
// One CTA per cell, same thread <-> velocity mapping as the consumers of k_stream.  Runs once after the caller
// has written f (first step, ufs_dvm_f_changed).
template <typename T, int O, int PIECES>
__device__ __forceinline__ void octant_sums(const Pos<T> (&pos)[PIECES], int PV, int CH, const T* base, double (&acc)[35]) {
    constexpr int VEC = V16<T>::N;
#pragma unroll
    for (int q = 0; q < PIECES; q++) {
        T v[VEC];
        ldg16(base + O * CH + q * PV * VEC, v);
        add_sums<T, O>(v, pos[q], acc);
    }
}
template <typename T, int NCW, int PIECES>
__global__ void __launch_bounds__(NCW * 32) k_sums(const StepParams p, const T* __restrict__ f, double* __restrict__ sums) {
    constexpr int VEC = V16<T>::N;
    __shared__ double red[NCW][SUMS_STRIDE];
    const int CH = p.nh[0] * p.nh[1] * p.nh[2];
    const int PV = CH / VEC / PIECES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cell = blockIdx.x;
    const bool active = tid < PV;
    Pos<T> pos[PIECES];
#pragma unroll
    for (int q = 0; q < PIECES; q++) pos[q] = pos_of<T>(p, active ? q * PV + tid : 0);
    double acc[35];
#pragma unroll
    for (int i = 0; i < 35; i++) acc[i] = 0.0;
    if (active) {
        const T* base = f + (int64_t)cell * p.Nv + (size_t)tid * VEC;
#define UFS_OCT(O) octant_sums<T, O, PIECES>(pos, PV, CH, base, acc);
        UFS_OCT(0) UFS_OCT(1) UFS_OCT(2) UFS_OCT(3) UFS_OCT(4) UFS_OCT(5) UFS_OCT(6) UFS_OCT(7)
#undef UFS_OCT
    }
    warp_store_sums(acc, red[warp], lane);
    __syncthreads();
    if (tid < SUMS_STRIDE) {
        double t = 0.0;
        if (tid < 35) {
#pragma unroll
            for (int w = 0; w < NCW; w++) t += red[w][tid];
        }
        sums[(int64_t)cell * SUMS_STRIDE + tid] = t;
    }
}

constexpr int STREAM_NCW = 14;
constexpr size_t SMEM_PER_CTA_MAX = 227 * 1024;

template <typename T, int PIECES>
cudaError_t launch_stream_t(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    if (p.collide) {
        const int wpb = 8;
        k_prep<T><<<(p.n_kin + 4 * wpb - 1) / (4 * wpb), wpb * 32, 0, st>>>(p);
    }
    auto k = k_stream<T, STREAM_NCW, PIECES>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    const int grid = p.n_kin < plan.grid ? p.n_kin : plan.grid;
    if (plan.ev0) cudaEventRecord(plan.ev0, st);
    k<<<grid, (STREAM_NCW + 2) * 32, plan.smem_bytes, st>>>(p);
    if (plan.ev1) cudaEventRecord(plan.ev1, st);
    return cudaGetLastError();
}

}  // namespace

int stream_tabn(const VelLayout& v) { return tabn_of(v.nh); }

// Launch geometry of the streaming step for this storage type / velocity grid, or false if the grid does not fit
// its assumptions (the one-CTA-per-cell kernels of kernels.cu then take over).
bool stream_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan) {
    if (!v.fast) return false;
    const size_t elem = storage == UFS_STORE_F32 ? 4 : 8;
    const int vec = (int)(16 / elem);
    const int ncw = STREAM_NCW;
    for (int a = 0; a < 3; a++)
        if (v.nv[a] > 32) return false;
    const int CH = v.nh[0] * v.nh[1] * v.nh[2];
    if (v.nh[0] % vec != 0 || CH % vec != 0) return false;
    const int chv = CH / vec;
    const int pieces = (chv + ncw * 32 - 1) / (ncw * 32);
    if (pieces > 2 || chv % pieces != 0) return false;
    const size_t stage = (size_t)4 * (chv / pieces) * 16;
    const int tabn = tabn_of(v.nh);
    int ns = 16 * pieces;  // at most two cells deep
    while (ns >= 4 && stream_smem_bytes(elem, ns, stage, ncw, tabn) > SMEM_PER_CTA_MAX) ns--;
    if (ns < 4) return false;  // a 2:1 face needs four slots in flight at once
    plan->ring = 2;
    plan->ncw = ncw;
    plan->pieces = pieces;
    plan->stages = ns;
    plan->threads = (ncw + 2) * 32;
    plan->smem_bytes = (int32_t)stream_smem_bytes(elem, ns, stage, ncw, tabn);
    plan->vec = vec;
    plan->fast = 1;
    plan->grid = sm_count;
    return true;
}

cudaError_t launch_prep(int storage, const StepParams& p, cudaStream_t st) {
    if (p.n_kin == 0 || !p.collide) return cudaSuccess;
    const int wpb = 8;
    const int blocks = (p.n_kin + 4 * wpb - 1) / (4 * wpb);  // four cells per warp
    if (storage == UFS_STORE_F32) k_prep<float><<<blocks, wpb * 32, 0, st>>>(p);
    else k_prep<double><<<blocks, wpb * 32, 0, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_stream(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    if (storage == UFS_STORE_F32)
        return plan.pieces == 2 ? launch_stream_t<float, 2>(plan, p, st) : launch_stream_t<float, 1>(plan, p, st);
    return plan.pieces == 2 ? launch_stream_t<double, 2>(plan, p, st) : launch_stream_t<double, 1>(plan, p, st);
}

// sums[n_kin][SUMS_STRIDE] of f (same layout and thread mapping as the streaming step)
cudaError_t launch_sums(int storage, const StepLaunch& plan, const StepParams& p, const void* f, double* sums, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    if (storage == UFS_STORE_F32) {
        const float* ff = reinterpret_cast<const float*>(f);
        if (plan.pieces == 2) k_sums<float, STREAM_NCW, 2><<<p.n_kin, STREAM_NCW * 32, 0, st>>>(p, ff, sums);
        else k_sums<float, STREAM_NCW, 1><<<p.n_kin, STREAM_NCW * 32, 0, st>>>(p, ff, sums);
    } else {
        const double* ff = reinterpret_cast<const double*>(f);
        if (plan.pieces == 2) k_sums<double, STREAM_NCW, 2><<<p.n_kin, STREAM_NCW * 32, 0, st>>>(p, ff, sums);
        else k_sums<double, STREAM_NCW, 1><<<p.n_kin, STREAM_NCW * 32, 0, st>>>(p, ff, sums);
    }
    return cudaGetLastError();
}

// UFS_DVM_CHECK: flags bit 1 if the freshly formed sums of cell `cell` (in `fresh`) differ from the carried ones
__global__ void k_check_sums(const double* __restrict__ carried, const double* __restrict__ fresh, int64_t cell, int32_t* flags) {
    const int j = threadIdx.x;
    if (j >= 35) return;
    const double a = carried[cell * SUMS_STRIDE + j], b = fresh[j];
    const double scale = fabs(carried[cell * SUMS_STRIDE]) + fabs(fresh[0]);   // the cell's density sum
    if (!(fabs(a - b) <= 1e-6 * scale)) atomicOr(flags, 2);
}
cudaError_t launch_check_sums(int storage, const StepLaunch& plan, const StepParams& p, const void* f, const double* carried, int64_t cell,
                              double* scratch, int32_t* flags, cudaStream_t st) {
    StepParams q = p;
    q.n_kin = 1;
    const size_t elem = storage == UFS_STORE_F32 ? 4 : 8;
    cudaError_t e = launch_sums(storage, plan, q, static_cast<const char*>(f) + (size_t)cell * p.Nv * elem, scratch, st);
    if (e != cudaSuccess) return e;
    k_check_sums<<<1, 64, 0, st>>>(carried, scratch, cell, flags);
    return cudaGetLastError();
}

cudaError_t launch_moments_from_sums(const StepParams& p, const double* sums, double* mom, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    const int64_t n = (int64_t)p.n_kin * 5;
    k_moments_from_sums<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, sums, mom);
    return cudaGetLastError();
}

}  // namespace ufs
