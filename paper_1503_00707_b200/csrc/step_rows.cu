// step_rows.cu -- k_rows: the streaming pass of the DVM step (see step_stream.cu for the scheme) with one velocity
// ROW per thread.
//
// An octant chunk (sign group) of a slab is nh_y*nh_z rows of nh_x values (x fastest).  A thread
// takes a whole row of a stage, so
//   * |xi_x| and its powers are the same for every thread: they are kernel parameters (constant bank operands of
//     the fp64 FMAs, no registers),
//   * the four x sums of the row (weights 1, |xi_x|, xi_x^2, |xi_x|^3) stay in the thread and the y/z weights and
//     signs are folded in once per row ("fold xi_y, xi_z once per run"),
//   * the update is  f' = B f + Cx_k (fX - f) + Cy fY + Cz fZ + W gx_k  with the BGK factor (1 - dt nu) already
//     inside B, C (Eq. 2, PAPER.md:103, and PAPER.md:231 in one expression).
// Warp roles: NG groups of GW consumer warps and one producer warp.  Stage n of the CTA (an octant chunk, or one of
// NQ row blocks of it) belongs to group n mod NG; its four streams (own chunk + the upwind chunk on each axis, the
// first-order stencil records of PAPER.md:113-115) arrive by cp.async.bulk in a ring slot, a 2:1 face brings three
// more slots.  What is constant for a cell (level, kind, the 2:1 masks of its octants, the Maxwellian factor table
// of k_prep) travels in a small ring of cell headers.  The warp that finishes a cell last adds up the per-warp
// partial sums and writes the cell's 35 velocity sums for the next step.
#include <cmath>

#include "device_util.cuh"
#include "kernels.cuh"
#include "stream_common.cuh"

namespace ufs {
namespace {

enum { CK_RING = 0, CK_GATHER = 1, CK_STOP = 2 };
constexpr int CELL_SLOTS = 3;
constexpr int HDR_INTS = 16;  // cell, level, kind, -, masks[8], -

struct RowsSmem {
    unsigned char* ring;   // [NS][slot_bytes]: 4 pieces
    unsigned char* cells;  // [CELL_SLOTS][cell_bytes]: HDR_INTS ints, then the factor table
    double* red;           // [CELL_SLOTS][NW][SUMS_STRIDE]
    double2* ayz;          // [NR] |xi_y|, |xi_z| of each row
    uint64_t* full;        // [NS]
    uint64_t* empty;       // [NS]
    uint64_t* cfull;       // [CELL_SLOTS]
    uint64_t* cempty;      // [CELL_SLOTS]
    int* cnt;              // [CELL_SLOTS] warps that have delivered their partial sums
};
__host__ __device__ inline size_t rows_cell_bytes(size_t elem, int tabn) {
    return ((size_t)HDR_INTS * 4 + (size_t)tabn * elem + 127) & ~(size_t)127;
}
__host__ __device__ inline size_t rows_smem_bytes(size_t elem, int ns, size_t slot_bytes, int nw, int tabn, int nr) {
    size_t b = (size_t)ns * slot_bytes + CELL_SLOTS * rows_cell_bytes(elem, tabn);
    b += (size_t)CELL_SLOTS * nw * SUMS_STRIDE * 8 + (size_t)nr * 16;
    b += (size_t)ns * 16 + CELL_SLOTS * 16 + CELL_SLOTS * 4 + 16;
    return (b + 127) & ~(size_t)127;
}
__device__ __forceinline__ RowsSmem rows_carve(unsigned char* base, size_t elem, int ns, size_t slot_bytes, int nw, int tabn, int nr) {
    RowsSmem s;
    size_t off = 0;
    s.ring = base; off += (size_t)ns * slot_bytes;
    s.cells = base + off; off += CELL_SLOTS * rows_cell_bytes(elem, tabn);
    s.red = reinterpret_cast<double*>(base + off); off += (size_t)CELL_SLOTS * nw * SUMS_STRIDE * 8;
    s.ayz = reinterpret_cast<double2*>(base + off); off += (size_t)nr * 16;
    s.full = reinterpret_cast<uint64_t*>(base + off); off += (size_t)ns * 8;
    s.empty = reinterpret_cast<uint64_t*>(base + off); off += (size_t)ns * 8;
    s.cfull = reinterpret_cast<uint64_t*>(base + off); off += CELL_SLOTS * 8;
    s.cempty = reinterpret_cast<uint64_t*>(base + off); off += CELL_SLOTS * 8;
    s.cnt = reinterpret_cast<int*>(base + off);
    return s;
}

// fold the four x sums of one row of octant O into the thread's 35 partial sums (layout: stream_common.cuh)
template <int O>
__device__ __forceinline__ void fold_row(double s0, double s1, double s2, double s3, double ay, double az, double (&acc)[35]) {
    constexpr int SX = O & 1, SY = (O >> 1) & 1, SZ = (O >> 2) & 1;
    const double r2 = fma(ay, ay, az * az);
    double h[5], g[5];
    h[0] = s0;
    h[1] = SX ? s1 : -s1;
    h[2] = (SY ? ay : -ay) * s0;
    h[3] = (SZ ? az : -az) * s0;
    h[4] = fma(r2, s0, s2);
    g[0] = s1;
    g[1] = SX ? s2 : -s2;
    g[2] = (SY ? ay : -ay) * s1;
    g[3] = (SZ ? az : -az) * s1;
    g[4] = fma(r2, s1, s3);
#pragma unroll
    for (int k = 0; k < 5; k++) {
        acc[k] += h[k];
        acc[g_index(0, SX, k)] += g[k];
        acc[g_index(1, SY, k)] = fma(ay, h[k], acc[g_index(1, SY, k)]);
        acc[g_index(2, SZ, k)] = fma(az, h[k], acc[g_index(2, SZ, k)]);
    }
}
__device__ __forceinline__ void fold_row_rt(int o, double s0, double s1, double s2, double s3, double ay, double az, double (&acc)[35]) {
    switch (o) {
        case 0: fold_row<0>(s0, s1, s2, s3, ay, az, acc); break;
        case 1: fold_row<1>(s0, s1, s2, s3, ay, az, acc); break;
        case 2: fold_row<2>(s0, s1, s2, s3, ay, az, acc); break;
        case 3: fold_row<3>(s0, s1, s2, s3, ay, az, acc); break;
        case 4: fold_row<4>(s0, s1, s2, s3, ay, az, acc); break;
        case 5: fold_row<5>(s0, s1, s2, s3, ay, az, acc); break;
        case 6: fold_row<6>(s0, s1, s2, s3, ay, az, acc); break;
        default: fold_row<7>(s0, s1, s2, s3, ay, az, acc); break;
    }
}

// |xi_x| in the storage type, from the kernel parameters
template <typename T> __device__ __forceinline__ T x_of(const StepParams& p, int k);
template <> __device__ __forceinline__ float x_of<float>(const StepParams& p, int k) { return p.xf[k]; }
template <> __device__ __forceinline__ double x_of<double>(const StepParams& p, int k) { return p.xpow[0][k]; }

// per-cell, per-thread coefficients of the row(s) this thread owns
template <typename T, int NQ>
struct RowCtx {
    T base[NQ], cy[NQ], cz[NQ];  // (1 - dt nu) (1 - dt/h (|xi_y| + |xi_z|)), (1 - dt nu) dt/h |xi_y|, ... |xi_z|
    T sx;                        // (1 - dt nu) dt/h: times |xi_x,k| it is the x coefficient
    T omega;                     // dt nu
    double ay[NQ], az[NQ];
    int ry[NQ], rz[NQ];
};

// One row from four shared-memory streams: transport + relaxation + store + the four x sums (a1, a4, a2').
template <typename T, int NHX, int NQ>
__device__ __forceinline__ void row_from_ring(const StepParams& p, const RowCtx<T, NQ>& rc, int q, T wb, const T* st, int pe,
                                              const T* gxrow, T* gdst, double& s0, double& s1, double& s2, double& s3) {
    constexpr int VEC = V16<T>::N, RV = NHX / VEC;
#pragma unroll
    for (int j = 0; j < RV; j++) {
        T own[VEC], X[VEC], Y[VEC], Z[VEC], out[VEC];
        lds16(st + j * VEC, own);
        lds16(st + pe + j * VEC, X);
        lds16(st + 2 * pe + j * VEC, Y);
        lds16(st + 3 * pe + j * VEC, Z);
#pragma unroll
        for (int i = 0; i < VEC; i++) {
            const int k = j * VEC + i;
            const T cx = rc.sx * x_of<T>(p, k);
            out[i] = rc.base[q] * own[i] + cx * (X[i] - own[i]) + rc.cy[q] * Y[i] + rc.cz[q] * Z[i];
        }
        if (p.collide) {
            T gx[VEC];
            lds16(gxrow + j * VEC, gx);
#pragma unroll
            for (int i = 0; i < VEC; i++) out[i] += wb * gx[i];
        }
        stg16_cs(gdst + j * VEC, out);
#pragma unroll
        for (int i = 0; i < VEC; i++) {
            const int k = j * VEC + i;
            const double d = (double)out[i];
            s0 += d;
            s1 = fma(p.xpow[0][k], d, s1);
            s2 = fma(p.xpow[1][k], d, s2);
            s3 = fma(p.xpow[2][k], d, s3);
        }
    }
}

// The same row for a cell with a kinetic/fluid face: sources gathered with plain loads.
template <typename T, int NHX, int NQ>
__device__ __forceinline__ void row_from_gather(const StepParams& p, const RowCtx<T, NQ>& rc, int q, T wb, int o, int CH, int row,
                                                const int* rec, const T* fin, int cell, const T* gxrow, T* gdst,
                                                double& s0, double& s1, double& s2, double& s3) {
    constexpr int VEC = V16<T>::N, RV = NHX / VEC;
    const T* own_base = fin + (int64_t)cell * p.Nv + (int64_t)o * CH + (int64_t)row * NHX;
#pragma unroll 1
    for (int j = 0; j < RV; j++) {
        T own[VEC], X[VEC], Y[VEC], Z[VEC], out[VEC];
        const int e = row * NHX + j * VEC;
        ldg16(own_base + j * VEC, own);
        gather_axis<T>(p, rec, fin, 0, o, CH, e, j * VEC, rc.ry[q], rc.rz[q], X);
        gather_axis<T>(p, rec, fin, 1, o, CH, e, j * VEC, rc.ry[q], rc.rz[q], Y);
        gather_axis<T>(p, rec, fin, 2, o, CH, e, j * VEC, rc.ry[q], rc.rz[q], Z);
#pragma unroll
        for (int i = 0; i < VEC; i++) {
            const T cx = rc.sx * x_of<T>(p, j * VEC + i);
            out[i] = rc.base[q] * own[i] + cx * (X[i] - own[i]) + rc.cy[q] * Y[i] + rc.cz[q] * Z[i];
        }
        if (p.collide) {
            T gx[VEC];
            lds16(gxrow + j * VEC, gx);
#pragma unroll
            for (int i = 0; i < VEC; i++) out[i] += wb * gx[i];
        }
        stg16_cs(gdst + j * VEC, out);
#pragma unroll
        for (int i = 0; i < VEC; i++) {
            const double d = (double)out[i];
            s0 += d;
            s1 = fma(p.xpow[0][j * VEC + i], d, s1);
            s2 = fma(p.xpow[1][j * VEC + i], d, s2);
            s3 = fma(p.xpow[2][j * VEC + i], d, s3);
        }
    }
}

template <typename T, int NHX, int GW, int NG, int NQ>
__global__ void __launch_bounds__((NG * GW + 1) * 32, 1) k_rows(const StepParams p) {
    constexpr int VEC = V16<T>::N, RV = NHX / VEC, NW = NG * GW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nhp = nhp_of(p.nh), tabn = tabn_of(p.nh);
    const int NR = p.nh[1] * p.nh[2];       // rows of an octant chunk
    const int NRQ = NR / NQ;                // rows of a stage
    const int CH = NR * NHX;
    const int pe = NRQ * NHX;               // elements per piece
    const uint32_t piece_bytes = (uint32_t)pe * (uint32_t)sizeof(T);
    const uint32_t slot_bytes = 4u * piece_bytes;
    const uint32_t tab_bytes = (uint32_t)tabn * (uint32_t)sizeof(T);
    const uint32_t cell_bytes = (uint32_t)rows_cell_bytes(sizeof(T), tabn);
    const int NS = p.ring_stages;
    const RowsSmem s = rows_carve(smem_raw, sizeof(T), NS, slot_bytes, NW, tabn, NR);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int i = 0; i < NS; i++) { mbar_init(&s.full[i], 1); mbar_init(&s.empty[i], NW); }
        for (int i = 0; i < CELL_SLOTS; i++) { mbar_init(&s.cfull[i], 1); mbar_init(&s.cempty[i], NW); s.cnt[i] = 0; }
        mbar_init_fence();
        if (blockIdx.x == 0) *p.counter_reset = 0;  // the other launch parity's cell counter
    }
    for (int r = tid; r < NR; r += blockDim.x)
        s.ayz[r] = make_double2(p.vel->xi[1][p.nh[1] + r % p.nh[1]], p.vel->xi[2][p.nh[2] + r / p.nh[1]]);
    __syncthreads();
    const T* fin = reinterpret_cast<const T*>(p.f_in);

    if (warp == NW) {
        // ------------------------------------------------ producer warp: cell tickets, headers, TMA copies
        auto fetch_async = [&]() -> int { return lane == 0 ? atomicAdd(p.counter, 1) : 0; };
        auto load_rec = [&](int cell) -> int {
            return cell < p.n_kin ? __ldg(reinterpret_cast<const int*>(p.cells + cell) + lane) : 0;
        };
        int slot = 0;
        uint32_t ph = 0;
        auto advance = [&]() { if (++slot == NS) { slot = 0; ph ^= 1u; } };
        int cur = __shfl_sync(0xffffffffu, fetch_async(), 0);
        int rec = load_rec(cur);
        int nxt_raw = 0;
        const int o_l = lane >> 2, t_l = lane & 3;
        for (int ncell = 0;; ncell++) {
            const int cs = ncell % CELL_SLOTS;
            int* hdr = reinterpret_cast<int*>(s.cells + (size_t)cs * cell_bytes);
            mbar_wait(&s.cempty[cs], (uint32_t)(((ncell / CELL_SLOTS) & 1) ^ 1), 1);
            if (cur >= p.n_kin) {
                if (lane == 0) { hdr[2] = CK_STOP; mbar_arrive(&s.cfull[cs]); }
                break;
            }
            const int level = __shfl_sync(0xffffffffu, rec, 24), flags = __shfl_sync(0xffffffffu, rec, 25);
            const bool ringable = (flags & CELL_NOFLUID) != 0;
            // bit d: direction d has four (finer) sources instead of one
            int four = 0;
#pragma unroll
            for (int d = 0; d < 6; d++) four |= (__shfl_sync(0xffffffffu, rec, d * 4 + 1) >= 0 ? 1 : 0) << d;
            // axes whose upwind face has four finer sources, for the octant of this lane (lanes 0..7)
            int mymask = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) mymask |= ((four >> (2 * b + (1 - ((lane >> b) & 1)))) & 1) << b;
            if (lane < 8) hdr[4 + lane] = ringable ? mymask : 0;
            if (lane == 0) { hdr[0] = cur; hdr[1] = level; hdr[2] = ringable ? CK_RING : CK_GATHER; }
            __syncwarp();
            if (lane == 0) {
                if (p.collide) {
                    mbar_arrive_expect_tx(&s.cfull[cs], tab_bytes);
                    bulk_g2s(hdr + HDR_INTS, reinterpret_cast<const T*>(p.tabs) + (int64_t)cur * tabn, tab_bytes, &s.cfull[cs]);
                } else {
                    mbar_arrive(&s.cfull[cs]);
                }
            }
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
                    const int mask = __shfl_sync(0xffffffffu, mymask, o);
                    const int xdir = lane < 3 ? 2 * lane + (1 - ((o >> lane) & 1)) : 0;
#pragma unroll
                    for (int q = 0; q < NQ; q++) {
                        mbar_wait(&s.empty[slot], ph ^ 1u, 2);
                        if (lane == 0) mbar_arrive_expect_tx(&s.full[slot], slot_bytes);
                        __syncwarp();
                        if (o_l == o) {
                            void* dst = s.ring + (size_t)slot * slot_bytes + (size_t)t_l * piece_bytes;
                            bulk_g2s(dst, ptr + (size_t)q * pe, piece_bytes, &s.full[slot]);
                        }
                        advance();
                        if (mask) {
                            // sources 1..3 of the axes in `mask` follow in three more slots (piece t = axis t)
#pragma unroll 1
                            for (int j = 1; j < 4; j++) {
                                const int xcode = __shfl_sync(0xffffffffu, rec, xdir * 4 + j);
                                mbar_wait(&s.empty[slot], ph ^ 1u, 3);
                                if (lane == 0) mbar_arrive_expect_tx(&s.full[slot], (uint32_t)__popc(mask) * piece_bytes);
                                __syncwarp();
                                if (lane < 3 && ((mask >> lane) & 1)) {
                                    const int xkind = xcode >> SRC_SHIFT;
                                    const int64_t xidx = xcode & SRC_INDEX_MASK;
                                    const T* xptr = (xkind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + xidx * p.Nv
                                                    + (int64_t)(xkind == SRC_MIRROR ? (o ^ (1 << lane)) : o) * CH;
                                    void* dst = s.ring + (size_t)slot * slot_bytes + (size_t)lane * piece_bytes;
                                    bulk_g2s(dst, xptr + (size_t)q * pe, piece_bytes, &s.full[slot]);
                                }
                                advance();
                            }
                        }
                    }
                }
            } else {
                nxt_raw = fetch_async();
            }
            cur = __shfl_sync(0xffffffffu, nxt_raw, 0);
            rec = load_rec(cur);
        }
        return;
    }

    // ---------------------------------------------------- consumer warps: group g takes stages n = g (mod NG)
    const int g = warp / GW;
    const int r = (warp % GW) * 32 + lane;  // row inside a stage
    const bool active = r < NRQ;
    int slot = 0, turn = 0;                 // turn = n mod NG
    uint32_t ph = 0;
    for (int ncell = 0;; ncell++) {
        const int cs = ncell % CELL_SLOTS;
        const int* hdr = reinterpret_cast<const int*>(s.cells + (size_t)cs * cell_bytes);
        mbar_wait(&s.cfull[cs], (uint32_t)((ncell / CELL_SLOTS) & 1), 4);
        const int kind = hdr[2];
        if (kind == CK_STOP) break;
        const int cell = hdr[0];
        const T* tab = reinterpret_cast<const T*>(hdr + HDR_INTS);
        const double dth = p.dt * p.inv_len * (double)(1 << hdr[1]);  // dt / h
        int masks = 0;
#pragma unroll
        for (int o = 0; o < 8; o++) masks |= hdr[4 + o] << (3 * o);
        RowCtx<T, NQ> rc;
        rc.omega = p.collide ? tab[6 * nhp] : T(0);
        const double om1 = 1.0 - (double)rc.omega;
        rc.sx = (T)(om1 * dth);
#pragma unroll
        for (int q = 0; q < NQ; q++) {
            const int row = active ? q * NRQ + r : 0;
            const double2 yz = s.ayz[row];
            rc.ay[q] = yz.x; rc.az[q] = yz.y;
            rc.ry[q] = row % p.nh[1]; rc.rz[q] = row / p.nh[1];
            rc.base[q] = (T)(om1 * (1.0 - dth * (yz.x + yz.y)));
            rc.cy[q] = (T)(om1 * dth * yz.x);
            rc.cz[q] = (T)(om1 * dth * yz.y);
        }
        T* const gcell = reinterpret_cast<T*>(p.f_out) + (int64_t)cell * p.Nv;
        const int* rec = reinterpret_cast<const int*>(p.cells + cell);
        double acc[35];
#pragma unroll
        for (int i = 0; i < 35; i++) acc[i] = 0.0;
#pragma unroll 1
        for (int o = 0; o < 8; o++) {
            const int mask = (masks >> (3 * o)) & 7;
#pragma unroll
            for (int q = 0; q < NQ; q++) {
                const bool mine = turn == g;
                if (++turn == NG) turn = 0;
                if (kind == CK_RING) {
                    if (mine) {
                        mbar_wait(&s.full[slot], ph, 5);
                        T* const st = reinterpret_cast<T*>(s.ring + (size_t)slot * slot_bytes) + (size_t)r * NHX;
                        if (mask) {
                            // 2:1 face (reading G3): the next three slots bring sources 1..3 of the axes in `mask`; they
                            // are added, in order, onto source 0 where it lies in this slot (a thread touches its own
                            // row only)
                            int sl = slot;
                            uint32_t sp = ph;
#pragma unroll 1
                            for (int j = 1; j < 4; j++) {
                                if (++sl == NS) { sl = 0; sp ^= 1u; }
                                mbar_wait(&s.full[sl], sp, 6);
                                if (active) {
                                    const T* se = reinterpret_cast<const T*>(s.ring + (size_t)sl * slot_bytes) + (size_t)r * NHX;
#pragma unroll 1
                                    for (int t = 0; t < 3; t++) {
                                        if ((mask >> t) & 1) {
#pragma unroll
                                            for (int jj = 0; jj < RV; jj++) {
                                                T v[VEC], x[VEC];
                                                lds16(se + t * pe + jj * VEC, v);
                                                lds16(st + (t + 1) * pe + jj * VEC, x);
#pragma unroll
                                                for (int i = 0; i < VEC; i++) x[i] += v[i];
                                                sts16(st + (t + 1) * pe + jj * VEC, x);
                                            }
                                        }
                                    }
                                }
                                __syncwarp();
                                if (lane == 0) mbar_arrive(&s.empty[sl]);
                            }
                            if (active) {  // each of the four sources weighs 1/4
#pragma unroll 1
                                for (int t = 0; t < 3; t++) {
                                    if ((mask >> t) & 1) {
#pragma unroll
                                        for (int jj = 0; jj < RV; jj++) {
                                            T x[VEC];
                                            lds16(st + (t + 1) * pe + jj * VEC, x);
#pragma unroll
                                            for (int i = 0; i < VEC; i++) x[i] *= T(0.25);
                                            sts16(st + (t + 1) * pe + jj * VEC, x);
                                        }
                                    }
                                }
                            }
                        }
                        if (active) {
                            const T wb = rc.omega * (tab[(4 + ((o >> 2) & 1)) * nhp + rc.rz[q]] * tab[(2 + ((o >> 1) & 1)) * nhp + rc.ry[q]]);
                            double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
                            row_from_ring<T, NHX, NQ>(p, rc, q, wb, st, pe, tab + (o & 1) * nhp,
                                                      gcell + (int64_t)o * CH + (int64_t)(q * NRQ + r) * NHX, s0, s1, s2, s3);
                            fold_row_rt(o, s0, s1, s2, s3, rc.ay[q], rc.az[q], acc);
                        }
                        // a slot written with ordinary stores: order them before the bulk copy that refills it
                        if (mask) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&s.empty[slot]);
                    } else {
                        // Not this group's stage: observe and release its slots all the same.  Every warp then sees
                        // every phase of every slot, so a group can never run a lap ahead of a barrier it skipped
                        // (its parity test would pass on a slot that has not been filled yet).
                        int sl = slot;
                        uint32_t sp = ph;
                        for (int j = 0; j < (mask ? 4 : 1); j++) {
                            mbar_wait(&s.full[sl], sp, 7);
                            __syncwarp();
                            if (lane == 0) mbar_arrive(&s.empty[sl]);
                            if (++sl == NS) { sl = 0; sp ^= 1u; }
                        }
                    }
                    const int adv = mask ? 4 : 1;
                    slot += adv;
                    if (slot >= NS) { slot -= NS; ph ^= 1u; }
                } else if (mine && active) {
                    const T wb = rc.omega * (tab[(4 + ((o >> 2) & 1)) * nhp + rc.rz[q]] * tab[(2 + ((o >> 1) & 1)) * nhp + rc.ry[q]]);
                    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
                    row_from_gather<T, NHX, NQ>(p, rc, q, wb, o, CH, q * NRQ + r, rec, fin, cell, tab + (o & 1) * nhp,
                                                gcell + (int64_t)o * CH + (int64_t)(q * NRQ + r) * NHX, s0, s1, s2, s3);
                    fold_row_rt(o, s0, s1, s2, s3, rc.ay[q], rc.az[q], acc);
                }
            }
        }
        // the warp's partial sums; the warp that delivers last adds all of them up and writes the cell's sums
        double* red = s.red + ((size_t)cs * NW + warp) * SUMS_STRIDE;
        warp_store_sums(acc, red, lane);
        __threadfence_block();
        __syncwarp();
        int last = 0;
        if (lane == 0) last = atomicAdd(&s.cnt[cs], 1) == NW - 1;
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {
            __threadfence_block();
            if (lane < SUMS_STRIDE / 2) {
                double2 t = make_double2(0.0, 0.0);
                const double2* src = reinterpret_cast<const double2*>(s.red + (size_t)cs * NW * SUMS_STRIDE) + lane;
#pragma unroll
                for (int w = 0; w < NW; w++) {
                    const double2 v = src[w * (SUMS_STRIDE / 2)];
                    t.x += v.x; t.y += v.y;
                }
                reinterpret_cast<double2*>(p.sums_out + (int64_t)cell * SUMS_STRIDE)[lane] = t;
            }
            if (lane == 0) s.cnt[cs] = 0;
            __syncwarp();
        }
        if (lane == 0) mbar_arrive(&s.cempty[cs]);
    }
}

constexpr size_t ROWS_SMEM_MAX = 227 * 1024;

// the instantiations: (storage type, nh_x, warps per group, groups, row blocks per octant chunk)
struct RowsVariant { int storage, nhx, gw, ng, nq; };
constexpr RowsVariant ROWS_VARIANTS[] = {
    {UFS_STORE_F32, 12, 5, 3, 1},
    {UFS_STORE_F64, 12, 3, 5, 2},
    {UFS_STORE_F64, 6, 2, 4, 1},
};
const RowsVariant* rows_variant(int storage, const VelLayout& v) {
    if (!v.fast) return nullptr;
    const int nr = v.nh[1] * v.nh[2];
    for (const RowsVariant& rv : ROWS_VARIANTS)
        if (rv.storage == storage && rv.nhx == v.nh[0] && nr % rv.nq == 0 && nr / rv.nq <= rv.gw * 32) return &rv;
    return nullptr;
}

template <typename T, int NHX, int GW, int NG, int NQ>
cudaError_t launch_rows_t(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    auto k = k_rows<T, NHX, GW, NG, NQ>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    const int grid = p.n_kin < plan.grid ? p.n_kin : plan.grid;
    k<<<grid, (NG * GW + 1) * 32, plan.smem_bytes, st>>>(p);
    return cudaGetLastError();
}

}  // namespace

// Launch geometry of the row kernel for this storage type / velocity grid, or false if no instantiation fits (the
// one-vector-per-thread kernel of step_stream.cu, then the one-CTA-per-cell kernels of kernels.cu, take over).
bool rows_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan) {
    const RowsVariant* rv = rows_variant(storage, v);
    if (!rv) return false;
    for (int a = 0; a < 3; a++)
        if (v.nv[a] > 32) return false;
    StepLaunch base{};
    if (!stream_plan(storage, v, sm_count, &base)) return false;  // k_sums shares its thread mapping (vec, pieces)
    const size_t elem = storage == UFS_STORE_F32 ? 4 : 8;
    const int nr = v.nh[1] * v.nh[2];
    const size_t slot = (size_t)4 * (nr / rv->nq) * rv->nhx * elem;
    const int nw = rv->gw * rv->ng;
    const int32_t nh[3] = {v.nh[0], v.nh[1], v.nh[2]};
    const int tabn = tabn_of(nh);
    int ns = 16;
    while (ns >= 4 && rows_smem_bytes(elem, ns, slot, nw, tabn, nr) > ROWS_SMEM_MAX) ns--;
    if (ns < 4) return false;  // a 2:1 face needs four slots in flight at once
    *plan = base;
    plan->ring = 3;
    plan->stages = ns;
    plan->threads = (nw + 1) * 32;
    plan->smem_bytes = (int32_t)rows_smem_bytes(elem, ns, slot, nw, tabn, nr);
    plan->grid = sm_count;
    return true;
}

cudaError_t launch_rows(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    cudaError_t e = launch_prep(storage, p, st);
    if (e != cudaSuccess) return e;
    if (storage == UFS_STORE_F32) return launch_rows_t<float, 12, 5, 3, 1>(plan, p, st);
    if (p.nh[0] == 12) return launch_rows_t<double, 12, 3, 5, 2>(plan, p, st);
    return launch_rows_t<double, 6, 2, 4, 1>(plan, p, st);
}

}  // namespace ufs
#ifdef UFS_DEBUG_WAIT
extern "C" int ufs_dvm_debug_read(int* out) {
    return (int)cudaMemcpyFromSymbol(out, ufs::g_dbg, sizeof(int) * 8);
}
#endif
