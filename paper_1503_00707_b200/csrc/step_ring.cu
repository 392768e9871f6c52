// step_ring.cu -- the TMA-fed, warp-specialised, persistent fused DVM step.
//
// A few persistent CTAs per SM pull kinetic cells from a global counter in Morton order.
// Warp roles inside a CTA:
//   * one PRODUCER warp.  For the cell in flight it turns the gather record (the first-order form of the
//     paper's per-cell, per-sign-group stencil records) into bulk asynchronous copies
//     (cp.async.bulk, the TMA engine): per velocity octant (sign group) the own chunk and
//     the single upwind chunk on each axis, cut into pieces, land in a ring of shared-memory stages; an
//     mbarrier per stage counts the bytes.  The producer runs ahead of the consumers by the depth of the
//     ring, across cell boundaries, so HBM/L2 requests stay in flight while a cell is being solved.
//   * NCW CONSUMER warps.  Thread t owns the same 16-byte vector of every piece: it forms
//     f* = c0 f_own + cx f_X + cy f_Y + cz f_Z (Eq. 2, first-order upwind), parks f* in the
//     cell's shared-memory slab (slots private to the thread), accumulates the five moments in fp64,
//     and after the block reduction three of the consumer warps (one per velocity axis) solve for the
//     discrete Maxwellian (the per-cell 5x5 problem of PAPER.md:145-163, 179 in its separable form); then
//     every consumer applies the BGK relaxation to its slots and streams f' out.
// Cells with a 2:1 face towards finer neighbours or a kinetic/fluid face are not fed through
// the ring: their consumers gather the sources with plain vector loads.
// HBM sees one read and one write of f per phase-space cell; the three upwind re-reads are L2 hits.
#include <cmath>

#include "device_util.cuh"
#include "kernels.cuh"

namespace ufs {
namespace {

enum { RING_SIMPLE = 0, RING_GATHER = 1, RING_STOP = 2 };
enum { BAR_CONS = 1, BAR_NEWTON = 2 };  // named barriers (0 is __syncthreads)

// ---------------------------------------------------------------- shared-memory carve-up
template <typename T>
struct RingSmem {
    T* slab;              // [Nv] f* of the cell in flight (thread-private slots)
    unsigned char* ring;  // [NS][4][piece_bytes]
    uint64_t* full;       // [NS]
    uint64_t* empty;      // [NS]
    int4* info;           // [NS] slab, level, kind, -
    double* red;          // [NCW][5] per-warp partial moments
    double* P;            // [2][3][5] power sums exchanged between the Newton warps
    T* tab;               // [3][nvp] Maxwellian factors gx, gy, amp*gz (canonical node index)
    T* omg;               // [4] dt * nu
};
__host__ __device__ inline size_t ring_aux_bytes(int ns, int ncw, int nvp, size_t elem) {
    size_t b = (size_t)ns * (8 + 8 + 16);
    b += (size_t)ncw * 5 * 8 + 2 * 3 * 5 * 8;
    b += (((size_t)3 * nvp * elem + 15) & ~(size_t)15) + 16;
    return (b + 127) & ~(size_t)127;
}
__host__ __device__ inline size_t ring_smem_bytes(int64_t Nv, size_t elem, int ns, size_t stage_bytes, int ncw, int nvp) {
    return (((size_t)Nv * elem + 127) & ~(size_t)127) + (size_t)ns * stage_bytes + ring_aux_bytes(ns, ncw, nvp, elem);
}
template <typename T>
__device__ __forceinline__ RingSmem<T> ring_carve(unsigned char* base, int64_t Nv, int ns, size_t stage_bytes, int ncw, int nvp) {
    RingSmem<T> s;
    size_t off = 0;
    s.slab = reinterpret_cast<T*>(base); off += ((size_t)Nv * sizeof(T) + 127) & ~(size_t)127;
    s.ring = base + off; off += (size_t)ns * stage_bytes;
    s.full = reinterpret_cast<uint64_t*>(base + off); off += (size_t)ns * 8;
    s.empty = reinterpret_cast<uint64_t*>(base + off); off += (size_t)ns * 8;
    s.info = reinterpret_cast<int4*>(base + off); off += (size_t)ns * 16;
    s.red = reinterpret_cast<double*>(base + off); off += (size_t)ncw * 5 * 8;
    s.P = reinterpret_cast<double*>(base + off); off += 2 * 3 * 5 * 8;
    s.tab = reinterpret_cast<T*>(base + off); off += ((size_t)3 * nvp * sizeof(T) + 15) & ~(size_t)15;
    s.omg = reinterpret_cast<T*>(base + off);
    return s;
}

// ---------------------------------------------------------------- per-thread velocity constants
// A consumer thread keeps the same |xi| on every axis for all 8 octants (symmetric grid, slots ordered by
// increasing |xi| inside an octant); one set per piece.
template <typename T>
struct PosConst {
    static constexpr int VEC = V16<T>::N;
    double ax[VEC], ay, az;
    int rx, ry, rz;  // rank of |xi| on each axis (rx: first of VEC)
};
template <typename T>
__device__ __forceinline__ PosConst<T> pos_const(const StepParams& p, int v) {
    constexpr int VEC = V16<T>::N;
    PosConst<T> c;
    const int e = v * VEC;
    c.rx = e % p.nh[0];
    const int row = e / p.nh[0];
    c.ry = row % p.nh[1];
    c.rz = row / p.nh[1];
#pragma unroll
    for (int i = 0; i < VEC; i++) c.ax[i] = __ldg(&p.vel->xi[0][p.nh[0] + c.rx + i]);
    c.ay = __ldg(&p.vel->xi[1][p.nh[1] + c.ry]);
    c.az = __ldg(&p.vel->xi[2][p.nh[2] + c.rz]);
    return c;
}
template <typename T>
struct Coef {  // update coefficients of one position for the level of the cell in flight
    static constexpr int VEC = V16<T>::N;
    T c0[VEC], cx[VEC], cy, cz;
};
template <typename T>
__device__ __forceinline__ Coef<T> coef_of(const PosConst<T>& c, double dth) {
    Coef<T> k;
    k.cy = (T)(dth * c.ay);
    k.cz = (T)(dth * c.az);
#pragma unroll
    for (int i = 0; i < Coef<T>::VEC; i++) {
        k.cx[i] = (T)(dth * c.ax[i]);
        k.c0[i] = (T)(1.0 - dth * (c.ax[i] + c.ay + c.az));
    }
    return k;
}

// a2: fp64 accumulation of the five moments of one vector of f* (octant o): three sums along the x run
// (3 fp64 operations per value), signs and the y/z weights folded once per vector
template <typename T>
__device__ __forceinline__ void add_moments(const T (&fs)[V16<T>::N], const PosConst<T>& c, int o, double (&mom)[5]) {
    double s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
    for (int i = 0; i < V16<T>::N; i++) {
        const double d = (double)fs[i];
        s0 += d;
        s1 = fma(c.ax[i], d, s1);
        s2 = fma(c.ax[i] * c.ax[i], d, s2);
    }
    mom[0] += s0;
    mom[1] += (o & 1) ? s1 : -s1;
    mom[2] = fma((o & 2) ? c.ay : -c.ay, s0, mom[2]);
    mom[3] = fma((o & 4) ? c.az : -c.az, s0, mom[3]);
    mom[4] += fma(fma(c.ay, c.ay, c.az * c.az), s0, s2);
}

// ---------------------------------------------------------------- gather path (cells that are not "simple")
// value of the upwind source on axis a for octant o: one chunk, or 4 finer neighbours each weighted 1/4
// (reading G3), or the pointwise Maxwellian of a fluid leaf's frozen moments
template <typename T>
__device__ __forceinline__ void gather_axis16(const StepParams& p, const int* __restrict__ rec, const T* fin, int a, int o,
                                              int CH, int e, const PosConst<T>& c, T (&out)[V16<T>::N]) {
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
            const int kz = ((o >> 2) & 1) ? p.nh[2] + c.rz : p.nh[2] - 1 - c.rz;
            const int ky = ((o >> 1) & 1) ? p.nh[1] + c.ry : p.nh[1] - 1 - c.ry;
            const double b = g->amp * g->g[2][kz] * g->g[1][ky];
#pragma unroll
            for (int i = 0; i < VEC; i++) {
                const int kx = (o & 1) ? p.nh[0] + c.rx + i : p.nh[0] - 1 - c.rx - i;
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

// ---------------------------------------------------------------- discrete Maxwellian (a3), three warps
// Solve  w sum_i m(xi_i) exp(alpha . m(xi_i)) = rho.  exp(alpha.m) = A gx gy gz with
// g_b[k] = exp(alpha_b xi_k + alpha_4 xi_k^2).  With the 1-D power sums P_b^r = sum_k xi_k^r g_b[k] the five
// equations read  P_b^1/P_b^0 = u_b (b = x,y,z),  sum_b P_b^2/P_b^0 = rho_4/n,  A w Px^0 Py^0 Pz^0 = n: an
// arrow-shaped 4x4 Newton system (closed-form Schur complement) plus the amplitude.  Same root as the
// oracle's 5x5 Newton (the solution is unique); stop rule: scaled residual <= 1e-13, or one more update
// after a residual <= 1e-7 (quadratic convergence), that last update applied to g through its series.
// Warp `axis` holds node k of its axis in lane k (nv <= 32).
// 1/x to about one ulp: hardware seed (20 bits) + two Newton steps; a full IEEE division costs three
// times as many dependent fp64 operations and the solve below is latency-bound
__device__ __forceinline__ double frcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}
template <typename T> struct NewtonTol;   // residual below which one more (series) update ends the solve
template <> struct NewtonTol<double> { static constexpr double series = 1e-7; };   // error after it ~1e-14
template <> struct NewtonTol<float> { static constexpr double series = 1e-4; };    // ~1e-8 << fp32 storage rounding

template <typename T>
__device__ __forceinline__ void newton_arrow(const StepParams& p, int axis, int lane, int ncw, const double* red,
                                             double* Pbuf, T* tab, T* omg, int nvp) {
    double rho[5];
#pragma unroll
    for (int a = 0; a < 5; a++) rho[a] = p.w * warp_sum(lane < ncw ? red[lane * 5 + a] : 0.0);
    const double n = rho[0];
    const double inv_n = frcp(n);
    const double u[3] = {rho[1] * inv_n, rho[2] * inv_n, rho[3] * inv_n};
    const double e2 = rho[4] * inv_n;
    const double T0 = (e2 - (u[0] * u[0] + u[1] * u[1] + u[2] * u[2])) * (1.0 / 3.0);
    const bool ok = (n > 0.0) && (T0 > 0.0);
    const double sqT = sqrt(ok ? T0 : 1.0);
    const double isc[4] = {frcp(sqT + fabs(u[0])), frcp(sqT + fabs(u[1])), frcp(sqT + fabs(u[2])), frcp(e2)};
    const double invT = frcp(T0);
    double al[4] = {u[0] * invT, u[1] * invT, u[2] * invT, -0.5 * invT};
    const int nv = p.nv[axis];
    const double x = lane < nv ? p.vel->xi[axis][lane] : 0.0;
    double g = 0.0, P0f[3] = {1.0, 1.0, 1.0};
    bool done = false;
    if (ok) {
        for (int it = 0; it <= 50 && !done; it++) {
            g = lane < nv ? exp((al[axis] + al[3] * x) * x) : 0.0;
            double t = g, ps[5];
#pragma unroll
            for (int r = 0; r < 5; r++) { ps[r] = t; t *= x; }
#pragma unroll
            for (int r = 0; r < 5; r++) ps[r] = warp_sum(ps[r]);
            double* Pw = Pbuf + (it & 1) * 15;
            if (lane == 0) {
#pragma unroll
                for (int r = 0; r < 5; r++) Pw[axis * 5 + r] = ps[r];
            }
            bar_sync(BAR_NEWTON, 96);
            double P[3][5], m1[3], m2[3], i0[3], r[4];
            r[3] = -e2;
#pragma unroll
            for (int b = 0; b < 3; b++) {
#pragma unroll
                for (int k = 0; k < 5; k++) P[b][k] = Pw[b * 5 + k];
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
                break;
            }
            if (!(res == res) || it == 50) break;
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
            if (res <= NewtonTol<T>::series) {
                // the update is small: apply it to g and to the zeroth power sums by expansion
                const double z = (dl[axis] + dl[3] * x) * x;
                g *= 1.0 + z * (1.0 + z * (0.5 + z * (1.0 / 6.0)));
#pragma unroll
                for (int b = 0; b < 3; b++)
                    P0f[b] = P[b][0] + dl[b] * P[b][1] + dl[3] * P[b][2]
                             + 0.5 * (dl[b] * dl[b] * P[b][2] + 2.0 * dl[b] * dl[3] * P[b][3] + dl[3] * dl[3] * P[b][4]);
                done = true;
            }
        }
    }
    if (done) {
        const double amp = n * frcp(p.w * P0f[0] * P0f[1] * P0f[2]);
        if (lane < nv) tab[axis * nvp + lane] = (T)(axis == 2 ? g * amp : g);
        if (axis == 0 && lane == 0) {
            // G9: nu = c_nu n T^(1-omega) / Kn (omega = 1/2: sqrt)
            const double Tp = (p.visc_exp == 0.5) ? sqT : pow(T0, 1.0 - p.visc_exp);
            omg[0] = (T)(p.dt * p.nu_pref * n * Tp * p.inv_kn);
        }
    } else {
        // no Maxwellian: pass f* through unchanged and raise the sticky flag (UFS_DVM_ENEWTON)
        if (lane < nv) tab[axis * nvp + lane] = T(0);
        if (axis == 0 && lane == 0) { omg[0] = T(0); atomicOr(p.flags, 1); }
    }
}

// ---------------------------------------------------------------- the kernel
template <typename T, int NCW, int PIECES, int MINB>
__global__ void __launch_bounds__((NCW + 1) * 32, MINB) k_step_ring(const StepParams p) {
    constexpr int VEC = V16<T>::N;
    constexpr int NCT = NCW * 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nvp = nvp_of(p.nv);
    const int CH = p.nh[0] * p.nh[1] * p.nh[2];
    const int PV = CH / VEC / PIECES;  // 16-byte vectors per piece and stream
    const uint32_t piece_bytes = (uint32_t)PV * 16u;
    const uint32_t stage_bytes = 4u * piece_bytes;
    const int NS = p.ring_stages;
    const RingSmem<T> s = ring_carve<T>(smem_raw, p.Nv, NS, stage_bytes, NCW, nvp);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int i = 0; i < NS; i++) { mbar_init(&s.full[i], 1); mbar_init(&s.empty[i], NCW); }
        mbar_init_fence();
        if (blockIdx.x == 0) *p.counter_reset = 0;  // the other launch parity's cell counter
    }
    __syncthreads();
    const T* fin = reinterpret_cast<const T*>(p.f_in);
    int slot = 0;
    uint32_t ph = 0;
    auto advance = [&]() { if (++slot == NS) { slot = 0; ph ^= 1u; } };

    if (warp == NCW) {
        // ------------------------------------------------ producer warp
        auto fetch_async = [&]() -> int { return lane == 0 ? atomicAdd(p.counter, 1) : 0; };
        auto load_rec = [&](int cell) -> int {
            return cell < p.n_kin ? __ldg(reinterpret_cast<const int*>(p.cells + cell) + lane) : 0;
        };
        // ticket_mode 0: the next cell's ticket is drawn while the current cell starts (its record is in
        // flight during the copies); 1: drawn when the current cell's last octant is issued, so that the
        // cells in flight stay consecutive in slab order; 2: static round-robin over the grid
        const int tm = p.ticket_mode;
        auto next_ticket = [&](int c) -> int { return tm == 2 ? c + (int)gridDim.x : fetch_async(); };
        int cur = tm == 2 ? (int)blockIdx.x : __shfl_sync(0xffffffffu, fetch_async(), 0);
        int nxt_raw = tm == 1 ? 0 : next_ticket(cur);
        int rec = load_rec(cur);
        const int o_l = lane >> 2, t_l = lane & 3;
        // L2 policy of this lane's stream.  Every chunk is read four times per step (by its own cell and by
        // one neighbour per axis); the reader that comes last in Morton order is the own cell for the
        // all-negative octant, else the high-side neighbour on the highest axis with positive velocity.
        uint64_t pol = 0;
        if (p.l2_mode > 0) {
            const int a_l = t_l - 1;
            const bool last = (t_l == 0) ? (o_l == 0) : (((o_l >> a_l) & 1) && (o_l >> (a_l + 1)) == 0);
            uint64_t keep, drop;
            asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(keep));
            asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(drop));
            if (p.l2_mode == 1) pol = keep;
            else if (p.l2_mode == 2) pol = last ? drop : keep;
            else pol = last ? drop : 0;
        }
        while (true) {
            if (cur >= p.n_kin) {
                mbar_wait(&s.empty[slot], ph ^ 1u);
                if (lane == 0) { s.info[slot] = make_int4(0, 0, RING_STOP, 0); mbar_arrive(&s.full[slot]); }
                break;
            }
            int nxt = 0, nrec = 0;
            if (tm != 1) {
                nxt = __shfl_sync(0xffffffffu, nxt_raw, 0);
                nxt_raw = next_ticket(nxt);
                nrec = load_rec(nxt);  // in flight while this cell's copies are issued
            }
            const int level = __shfl_sync(0xffffffffu, rec, 24), flags = __shfl_sync(0xffffffffu, rec, 25);
            if (flags & CELL_SIMPLE) {
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
                    if (tm == 1 && o == 7) nxt_raw = fetch_async();
#pragma unroll
                    for (int q = 0; q < PIECES; q++) {
                        mbar_wait(&s.empty[slot], ph ^ 1u);
                        if (lane == 0) {
                            s.info[slot] = make_int4(cur, level, RING_SIMPLE, o * PIECES + q);
                            mbar_arrive_expect_tx(&s.full[slot], stage_bytes);
                        }
                        __syncwarp();
                        if (o_l == o) {
                            void* dst = s.ring + (size_t)slot * stage_bytes + (size_t)t_l * piece_bytes;
                            if (pol) bulk_g2s_hint(dst, ptr + (size_t)q * PV * VEC, piece_bytes, &s.full[slot], pol);
                            else bulk_g2s(dst, ptr + (size_t)q * PV * VEC, piece_bytes, &s.full[slot]);
                        }
                        advance();
                    }
                }
            } else {
                if (tm == 1) nxt_raw = fetch_async();
                mbar_wait(&s.empty[slot], ph ^ 1u);
                if (lane == 0) { s.info[slot] = make_int4(cur, level, RING_GATHER, 0); mbar_arrive(&s.full[slot]); }
                advance();
            }
            if (tm == 1) {
                nxt = __shfl_sync(0xffffffffu, nxt_raw, 0);
                nrec = load_rec(nxt);
            }
            cur = nxt;
            rec = nrec;
        }
        return;
    }

    // ---------------------------------------------------- consumer warps
    const bool active = tid < PV;
    PosConst<T> pos[PIECES];
#pragma unroll
    for (int q = 0; q < PIECES; q++) pos[q] = pos_const<T>(p, active ? q * PV + tid : 0);
    T* const myslab = s.slab + (size_t)tid * VEC;
    while (true) {
        mbar_wait(&s.full[slot], ph);
        const int4 inf = s.info[slot];
        if (inf.z == RING_STOP) break;
        const int cell = inf.x;
        const double dth = p.dt * p.inv_len * (double)(1 << inf.y);  // dt / h
        Coef<T> kf[PIECES];
#pragma unroll
        for (int q = 0; q < PIECES; q++) kf[q] = coef_of<T>(pos[q], dth);
        T* const gout = reinterpret_cast<T*>(p.f_out) + (int64_t)cell * p.Nv + (size_t)tid * VEC;
        double mom[5] = {0, 0, 0, 0, 0};
        if (inf.z == RING_SIMPLE) {
            // a1 + a2 from the ring: one stage per (octant, piece)
#pragma unroll 1
            for (int o = 0; o < 8; o++) {
#pragma unroll
                for (int q = 0; q < PIECES; q++) {
                    if (o + q > 0) mbar_wait(&s.full[slot], ph);
                    if (active) {
                        const T* st = reinterpret_cast<const T*>(s.ring + (size_t)slot * stage_bytes + (size_t)tid * 16);
                        const int pe = PV * VEC;  // elements per piece
                        T own[VEC], X[VEC], Y[VEC], Z[VEC], fs[VEC];
                        lds16(st, own);
                        lds16(st + pe, X);
                        lds16(st + 2 * pe, Y);
                        lds16(st + 3 * pe, Z);
#pragma unroll
                        for (int i = 0; i < VEC; i++)
                            fs[i] = kf[q].c0[i] * own[i] + kf[q].cx[i] * X[i] + kf[q].cy * Y[i] + kf[q].cz * Z[i];
                        if (p.collide) {
                            sts16(myslab + o * CH + q * pe, fs);
                            add_moments<T>(fs, pos[q], o, mom);
                        } else {
                            stg16_cs(gout + o * CH + q * pe, fs);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&s.empty[slot]);
                    advance();
                }
            }
        } else {
            // the ring carries only the cell header: gather with plain loads
            __syncwarp();
            if (lane == 0) mbar_arrive(&s.empty[slot]);
            advance();
            if (active) {
                const int* rec = reinterpret_cast<const int*>(p.cells + cell);
                const T* own_base = fin + (int64_t)cell * p.Nv + (size_t)tid * VEC;
#pragma unroll 1
                for (int o = 0; o < 8; o++) {
#pragma unroll
                    for (int q = 0; q < PIECES; q++) {
                        const int pe = PV * VEC;
                        const int e = q * pe + tid * VEC;
                        T own[VEC], X[VEC], Y[VEC], Z[VEC], fs[VEC];
                        ldg16(own_base + o * CH + q * pe, own);
                        gather_axis16<T>(p, rec, fin, 0, o, CH, e, pos[q], X);
                        gather_axis16<T>(p, rec, fin, 1, o, CH, e, pos[q], Y);
                        gather_axis16<T>(p, rec, fin, 2, o, CH, e, pos[q], Z);
#pragma unroll
                        for (int i = 0; i < VEC; i++)
                            fs[i] = kf[q].c0[i] * own[i] + kf[q].cx[i] * X[i] + kf[q].cy * Y[i] + kf[q].cz * Z[i];
                        if (p.collide) {
                            sts16(myslab + o * CH + q * pe, fs);
                            add_moments<T>(fs, pos[q], o, mom);
                        } else {
                            stg16_cs(gout + o * CH + q * pe, fs);
                        }
                    }
                }
            }
        }
        if (!p.collide) continue;

        // a2 (block reduction) + a3 (three warps, one per axis)
#pragma unroll
        for (int a = 0; a < 5; a++) mom[a] = warp_sum(mom[a]);
        if (lane == 0) {
#pragma unroll
            for (int a = 0; a < 5; a++) s.red[warp * 5 + a] = mom[a];
        }
        bar_sync(BAR_CONS, NCT);
        if (warp < 3) newton_arrow<T>(p, warp, lane, NCW, s.red, s.P, s.tab, s.omg, nvp);
        bar_sync(BAR_CONS, NCT);

        // a4: f' = f* + dt nu (M - f*), M = amp gz gy gx from the factor tables; streaming stores
        if (active) {
            const T omega = s.omg[0];
#pragma unroll
            for (int q = 0; q < PIECES; q++) {
                const PosConst<T>& c = pos[q];
                const int pe = PV * VEC;
                T gxp[VEC], gxm[VEC];
#pragma unroll
                for (int i = 0; i < VEC; i++) {
                    gxp[i] = s.tab[p.nh[0] + c.rx + i];
                    gxm[i] = s.tab[p.nh[0] - 1 - c.rx - i];
                }
                const T gy[2] = {s.tab[nvp + p.nh[1] - 1 - c.ry], s.tab[nvp + p.nh[1] + c.ry]};
                const T gz[2] = {s.tab[2 * nvp + p.nh[2] - 1 - c.rz], s.tab[2 * nvp + p.nh[2] + c.rz]};
#pragma unroll
                for (int o = 0; o < 8; o++) {
                    T fs[VEC], out[VEC];
                    lds16(myslab + o * CH + q * pe, fs);
                    const T b = gz[(o >> 2) & 1] * gy[(o >> 1) & 1];
#pragma unroll
                    for (int i = 0; i < VEC; i++) {
                        const T M = b * ((o & 1) ? gxp[i] : gxm[i]);
                        out[i] = fs[i] + omega * (M - fs[i]);
                    }
                    stg16_cs(gout + o * CH + q * pe, out);
                }
            }
        }
    }
}

template <typename T, int NCW, int PIECES, int MINB>
cudaError_t launch_ring_t(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    auto k = k_step_ring<T, NCW, PIECES, MINB>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    const int grid = p.n_kin < plan.grid ? p.n_kin : plan.grid;
    k<<<grid, (NCW + 1) * 32, plan.smem_bytes, st>>>(p);
    return cudaGetLastError();
}

template <typename T, int NCW, int PIECES, int MINB>
int ring_occupancy_t(const StepLaunch& plan) {
    auto k = k_step_ring<T, NCW, PIECES, MINB>;
    if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes) != cudaSuccess) return 0;
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k, (NCW + 1) * 32, plan.smem_bytes) != cudaSuccess) return 0;
    return n;
}

constexpr int RING_NCW_F32 = 7, RING_NCW_F64 = 14;
constexpr size_t SMEM_PER_SM = 228 * 1024, SMEM_PER_CTA_MAX = 227 * 1024, SMEM_CTA_RESERVED = 1024;

}  // namespace

// Launch geometry of the ring kernel for this storage type / velocity grid, or false if the grid does not
// fit its assumptions (the one-CTA-per-cell kernels of kernels.cu then take over).
bool ring_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan) {
    if (!v.fast) return false;
    const size_t elem = storage == UFS_STORE_F32 ? 4 : 8;
    const int vec = (int)(16 / elem);
    const int ncw = storage == UFS_STORE_F32 ? RING_NCW_F32 : RING_NCW_F64;
    for (int a = 0; a < 3; a++)
        if (v.nv[a] > 32) return false;
    const int CH = v.nh[0] * v.nh[1] * v.nh[2];
    if (v.nh[0] % vec != 0 || CH % vec != 0) return false;
    const int chv = CH / vec;
    const int pieces = (chv + ncw * 32 - 1) / (ncw * 32);
    if (pieces > 2 || chv % pieces != 0) return false;
    const size_t stage = (size_t)4 * (chv / pieces) * 16;
    const int nvp = nvp_of(v.nv);
    const int per_cell = 8 * pieces;
    // as many CTAs per SM as keep a ring of at least 4 stages (at most two cells deep)
    for (int ctas = 4; ctas >= 1; ctas--) {
        size_t budget = SMEM_PER_SM / ctas - SMEM_CTA_RESERVED;
        if (budget > SMEM_PER_CTA_MAX) budget = SMEM_PER_CTA_MAX;
        int ns = 2 * per_cell;
        while (ns >= 4 && ring_smem_bytes(v.Nv, elem, ns, stage, ncw, nvp) > budget) ns--;
        if (ns < 4) continue;
        if ((ncw + 1) * 32 * ctas > 2048) continue;
        plan->ring = 1;
        plan->ncw = ncw;
        plan->pieces = pieces;
        plan->stages = ns;
        plan->threads = (ncw + 1) * 32;
        plan->smem_bytes = (int32_t)ring_smem_bytes(v.Nv, elem, ns, stage, ncw, nvp);
        plan->vec = vec;
        plan->fast = 1;
        plan->grid = sm_count * ctas;
        return true;
    }
    return false;
}

// resident CTAs per SM of the planned kernel on the current device (0: it cannot be launched)
int ring_occupancy(int storage, const StepLaunch& plan) {
    if (storage == UFS_STORE_F32)
        return plan.pieces == 2 ? ring_occupancy_t<float, RING_NCW_F32, 2, 2>(plan) : ring_occupancy_t<float, RING_NCW_F32, 1, 2>(plan);
    return plan.pieces == 2 ? ring_occupancy_t<double, RING_NCW_F64, 2, 1>(plan) : ring_occupancy_t<double, RING_NCW_F64, 1, 1>(plan);
}

cudaError_t launch_ring(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    if (storage == UFS_STORE_F32)
        return plan.pieces == 2 ? launch_ring_t<float, RING_NCW_F32, 2, 2>(plan, p, st)
                                : launch_ring_t<float, RING_NCW_F32, 1, 2>(plan, p, st);
    return plan.pieces == 2 ? launch_ring_t<double, RING_NCW_F64, 2, 1>(plan, p, st)
                            : launch_ring_t<double, RING_NCW_F64, 1, 1>(plan, p, st);
}

}  // namespace ufs
