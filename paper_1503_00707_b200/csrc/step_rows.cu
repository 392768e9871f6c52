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
constexpr int HDR_REC = 16;   // header ints: cell, level, kind, mbits, masks, -..., then the 32 words of the cell record
constexpr int HDR_INTS = 48;

// Shared-memory map of a CTA (byte offsets from the start of dynamic shared memory).
struct RowsSmem {
    uint32_t ring;    // [NS][slot_bytes]: 4 pieces
    uint32_t cells;   // [CELL_SLOTS][cell_bytes]: HDR_INTS ints, then the factor table
    uint32_t red;     // [CELL_SLOTS][NW][SUMS_STRIDE] doubles
    uint32_t ayz;     // [NR] double2: |xi_y|, |xi_z| of each row
    uint32_t full;    // [NS] mbarriers
    uint32_t empty;   // [NS]
    uint32_t cfull;   // [CELL_SLOTS]
    uint32_t cempty;  // [CELL_SLOTS]
    uint32_t cnt;     // [CELL_SLOTS] ints: warps that have delivered their partial sums
    uint32_t issued;  // int: ring slots armed by the producer so far
    uint32_t total;
};
__host__ __device__ inline size_t rows_cell_bytes(size_t elem, int tabn) {
    return ((size_t)HDR_INTS * 4 + (size_t)tabn * elem + 127) & ~(size_t)127;
}
__host__ __device__ inline RowsSmem rows_map(size_t elem, int ns, size_t slot_bytes, int nw, int tabn, int nr) {
    RowsSmem s;
    size_t off = 0;
    s.ring = (uint32_t)off; off += (size_t)ns * slot_bytes;
    s.cells = (uint32_t)off; off += CELL_SLOTS * rows_cell_bytes(elem, tabn);
    s.red = (uint32_t)off; off += (size_t)CELL_SLOTS * nw * SUMS_STRIDE * 8;
    s.ayz = (uint32_t)off; off += (size_t)nr * 16;
    s.full = (uint32_t)off; off += (size_t)ns * 8;
    s.empty = (uint32_t)off; off += (size_t)ns * 8;
    s.cfull = (uint32_t)off; off += CELL_SLOTS * 8;
    s.cempty = (uint32_t)off; off += CELL_SLOTS * 8;
    s.cnt = (uint32_t)off; off += CELL_SLOTS * 4;
    s.issued = (uint32_t)off; off += 8;
    s.total = (uint32_t)((off + 127) & ~(size_t)127);
    return s;
}
__host__ __device__ inline size_t rows_smem_bytes(size_t elem, int ns, size_t slot_bytes, int nw, int tabn, int nr) {
    return rows_map(elem, ns, slot_bytes, nw, tabn, nr).total;
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
};

// One row of values already in registers: transport + relaxation + store + the four x sums (a1, a4, a2').
template <typename T, int NHX, int NQ>
__device__ __forceinline__ void row_finish(const StepParams& p, const RowCtx<T, NQ>& rc, int q, T wb, int j, const T (&own)[V16<T>::N],
                                           const T (&X)[V16<T>::N], const T (&Y)[V16<T>::N], const T (&Z)[V16<T>::N],
                                           const T* gxrow, T* gdst, double& s0, double& s1, double& s2, double& s3) {
    constexpr int VEC = V16<T>::N;
    T out[VEC];
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
        const int k = j * VEC + i;
        const double d = (double)out[i];
        s0 += d;
        s1 = fma(p.xpow[0][k], d, s1);
        s2 = fma(p.xpow[1][k], d, s2);
        s3 = fma(p.xpow[2][k], d, s3);
    }
}

// Upwind values of a kinetic/fluid face (reading G13): the pointwise Maxwellian of the fluid leaf's frozen
// moments, from its separable factors; `code` is the source code of the direction, j the 16-byte vector of the row.
template <typename T>
__device__ __forceinline__ void fluid_vec(const StepParams& p, int code, int o, int j, int ry, int rz, T (&v)[V16<T>::N]) {
    constexpr int VEC = V16<T>::N;
    const FluidGhost* g = p.fluid + (code & SRC_INDEX_MASK);
    const int kz = ((o >> 2) & 1) ? p.nh[2] + rz : p.nh[2] - 1 - rz;
    const int ky = ((o >> 1) & 1) ? p.nh[1] + ry : p.nh[1] - 1 - ry;
    const double b = g->amp * g->g[2][kz] * g->g[1][ky];
#pragma unroll
    for (int i = 0; i < VEC; i++) {
        const int kx = (o & 1) ? p.nh[0] + j * VEC + i : p.nh[0] - 1 - j * VEC - i;
        v[i] = (T)(b * g->g[0][kx]);
    }
}
// what row_from_ring needs to know about the fluid streams of a stage (fm = 0: none)
struct FluidStreams { int fm, o, ry, rz; const int* rec; };
template <typename T>
__device__ __forceinline__ void apply_fluid(const StepParams& p, const FluidStreams& fs, int j, T (&X)[V16<T>::N], T (&Y)[V16<T>::N],
                                            T (&Z)[V16<T>::N]) {
    if (fs.fm & 1) fluid_vec<T>(p, fs.rec[(1 - (fs.o & 1)) * 4], fs.o, j, fs.ry, fs.rz, X);
    if (fs.fm & 2) fluid_vec<T>(p, fs.rec[(2 + 1 - ((fs.o >> 1) & 1)) * 4], fs.o, j, fs.ry, fs.rz, Y);
    if (fs.fm & 4) fluid_vec<T>(p, fs.rec[(4 + 1 - ((fs.o >> 2) & 1)) * 4], fs.o, j, fs.ry, fs.rz, Z);
}

// One row from the four streams of a ring slot.  EARLY: the whole row is read into registers first and the slot is
// handed back to the producer before the arithmetic (the ring then holds data in flight, not data in use).
// FLUID: streams whose source is a fluid leaf are not in the slot; they are computed (apply_fluid).
template <typename T, int NHX, int NQ, bool EARLY, bool FLUID>
__device__ __forceinline__ void row_from_ring(const StepParams& p, const RowCtx<T, NQ>& rc, int q, T wb, const T* st, int pe,
                                              const T* gxrow, T* gdst, bool active, int lane, uint32_t empty_bar,
                                              const FluidStreams& fs, double& s0, double& s1, double& s2, double& s3) {
    constexpr int VEC = V16<T>::N, RV = NHX / VEC;
    if (EARLY) {
        T own[RV][VEC], X[RV][VEC], Y[RV][VEC], Z[RV][VEC];
        if (active) {
#pragma unroll
            for (int j = 0; j < RV; j++) {
                lds16(st + j * VEC, own[j]);
                lds16(st + pe + j * VEC, X[j]);
                lds16(st + 2 * pe + j * VEC, Y[j]);
                lds16(st + 3 * pe + j * VEC, Z[j]);
                if (FLUID && fs.fm) apply_fluid<T>(p, fs, j, X[j], Y[j], Z[j]);
            }
        }
        __syncwarp();
        if (lane == 0) smbar_arrive(empty_bar);
        if (active) {
#pragma unroll
            for (int j = 0; j < RV; j++) row_finish<T, NHX, NQ>(p, rc, q, wb, j, own[j], X[j], Y[j], Z[j], gxrow, gdst, s0, s1, s2, s3);
        }
    } else {
        if (active) {
#pragma unroll
            for (int j = 0; j < RV; j++) {
                T own[VEC], X[VEC], Y[VEC], Z[VEC];
                lds16(st + j * VEC, own);
                lds16(st + pe + j * VEC, X);
                lds16(st + 2 * pe + j * VEC, Y);
                lds16(st + 3 * pe + j * VEC, Z);
                if (FLUID && fs.fm) apply_fluid<T>(p, fs, j, X, Y, Z);
                row_finish<T, NHX, NQ>(p, rc, q, wb, j, own, X, Y, Z, gxrow, gdst, s0, s1, s2, s3);
            }
        }
        __syncwarp();
        if (lane == 0) smbar_arrive(empty_bar);
    }
}

// The same row for a cell with a kinetic/fluid face: sources gathered with plain loads.
template <typename T, int NHX, int NQ>
__device__ __forceinline__ void row_from_gather(const StepParams& p, const RowCtx<T, NQ>& rc, int q, T wb, int o, int CH, int row,
                                                int ry, int rz, const int* rec, const T* fin, int cell, const T* gxrow, T* gdst,
                                                double& s0, double& s1, double& s2, double& s3) {
    constexpr int VEC = V16<T>::N, RV = NHX / VEC;
    const T* own_base = fin + (int64_t)cell * p.Nv + (int64_t)o * CH + (int64_t)row * NHX;
#pragma unroll 1
    for (int j = 0; j < RV; j++) {
        T own[VEC], X[VEC], Y[VEC], Z[VEC];
        const int e = row * NHX + j * VEC;
        ldg16(own_base + j * VEC, own);
        gather_axis<T>(p, rec, fin, 0, o, CH, e, j * VEC, ry, rz, X);
        gather_axis<T>(p, rec, fin, 1, o, CH, e, j * VEC, ry, rz, Y);
        gather_axis<T>(p, rec, fin, 2, o, CH, e, j * VEC, ry, rz, Z);
        row_finish<T, NHX, NQ>(p, rc, q, wb, j, own, X, Y, Z, gxrow, gdst, s0, s1, s2, s3);
    }
}

template <typename T, int NHX, int GW, int NG, int NQ, bool EARLY, bool FLUID>
__global__ void __launch_bounds__((NG * GW + 1) * 32, 1) k_rows(const StepParams p) {
    constexpr int VEC = V16<T>::N, RV = NHX / VEC, NW = NG * GW;
    constexpr int MAXST = (8 * NQ + NG - 1) / NG;  // stages of one cell that can fall to one group
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
    // the shared-memory map comes with the kernel parameters (constant bank): nothing of it has to live in registers
    RowsSmem s;
    s.ring = p.smap[0]; s.cells = p.smap[1]; s.red = p.smap[2]; s.ayz = p.smap[3]; s.full = p.smap[4]; s.empty = p.smap[5];
    s.cfull = p.smap[6]; s.cempty = p.smap[7]; s.cnt = p.smap[8]; s.issued = p.smap[9]; s.total = p.smap[10];
    const uint32_t sb = smem_u32(smem_raw);  // shared-space address of the map's origin
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) {
        for (int i = 0; i < NS; i++) {
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + s.full) + i, 1);
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + s.empty) + i, GW);
        }
        for (int i = 0; i < CELL_SLOTS; i++) {
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + s.cfull) + i, 1);
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + s.cempty) + i, NW);
            reinterpret_cast<int*>(smem_raw + s.cnt)[i] = 0;
        }
        reinterpret_cast<int*>(smem_raw + s.issued)[0] = reinterpret_cast<int*>(smem_raw + s.issued)[1] = 0;
        mbar_init_fence();
        if (blockIdx.x == 0) *p.counter_reset = 0;  // the other launch parity's cell counter
    }
    for (int r = tid; r < NR; r += blockDim.x)
        reinterpret_cast<double2*>(smem_raw + s.ayz)[r] =
            make_double2(p.vel->xi[1][p.nh[1] + r % p.nh[1]], p.vel->xi[2][p.nh[2] + r / p.nh[1]]);
    __syncthreads();
    const T* fin = reinterpret_cast<const T*>(p.f_in);

    if (warp == NW) {
        // ------------------------------------------------ producer warp: cell tickets, headers, factor tables, TMA copies
        const int o_l = lane >> 2, t_l = lane & 3;
        int slot = 0, gidx = 0;  // ring cursor and global index of the next slot (both producers count every slot)
        uint32_t ph = 0;
        auto skip = [&](int k) {
            gidx += k;
            slot += k;
            while (slot >= NS) { slot -= NS; ph ^= 1u; }
        };
        // arm the slot for `bytes` and publish it; the caller's lanes then issue the copies
        auto arm = [&](uint32_t bytes) {
            smbar_wait(sb + s.empty + 8u * slot, ph ^ 1u);
            if (lane == 0) {
                smbar_arrive_expect_tx(sb + s.full + 8u * slot, bytes);
                __threadfence_block();
                ssts_i32_volatile(sb + s.issued, gidx + 1);
            }
            __syncwarp();
        };
        // issue octants [o0, o1) of cell `cur`; rec = this lane's word of the cell record, masks = 3 bits per octant
        auto issue = [&](int cur, int rec, int masks, int fmasks, int o0, int o1) {
            // lane (o,t): stream t of octant o -- t = 0 own chunk, t = 1..3 the upwind chunk on axis t-1
            const int a = t_l > 0 ? t_l - 1 : 0;
            const int dir = 2 * a + (1 - ((o_l >> a) & 1));
            const int code = __shfl_sync(0xffffffffu, rec, dir * 4);
            const int kind = code >> SRC_SHIFT;
            const int64_t idx = code & SRC_INDEX_MASK;
            const T* ptr = (t_l == 0) ? fin + (int64_t)cur * p.Nv + (int64_t)o_l * CH
                                      : (kind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + idx * p.Nv
                                            + (int64_t)(kind == SRC_MIRROR ? (o_l ^ (1 << a)) : o_l) * CH;
            for (int o = o0; o < o1; o++) {
                const int mask = (masks >> (3 * o)) & 7;
                const int xdir = lane < 3 ? 2 * lane + (1 - ((o >> lane) & 1)) : 0;
#pragma unroll
                for (int q = 0; q < NQ; q++) {
                    // streams from a fluid leaf are not copied (the consumers compute them)
                    const int fm = FLUID ? (fmasks >> (3 * o)) & 7 : 0;
                    arm(slot_bytes - (uint32_t)__popc(fm) * piece_bytes);
                    if (o_l == o && !(t_l > 0 && ((fm >> (t_l - 1)) & 1)))
                        sbulk_g2s(sb + s.ring + slot * slot_bytes + t_l * piece_bytes, ptr + (size_t)q * pe, piece_bytes,
                                  sb + s.full + 8u * slot);
                    skip(1);
                    if (mask) {
                        // sources 1..3 of the axes in `mask` follow in three more slots (piece t = axis t)
#pragma unroll 1
                        for (int j = 1; j < 4; j++) {
                            const int xcode = __shfl_sync(0xffffffffu, rec, xdir * 4 + j);
                            arm((uint32_t)__popc(mask) * piece_bytes);
                            if (lane < 3 && ((mask >> lane) & 1)) {
                                const int xkind = xcode >> SRC_SHIFT;
                                const int64_t xidx = xcode & SRC_INDEX_MASK;
                                const T* xptr = (xkind == SRC_TABLE ? reinterpret_cast<const T*>(p.tables) : fin) + xidx * p.Nv
                                                + (int64_t)(xkind == SRC_MIRROR ? (o ^ (1 << lane)) : o) * CH;
                                sbulk_g2s(sb + s.ring + slot * slot_bytes + lane * piece_bytes, xptr + (size_t)q * pe, piece_bytes,
                                          sb + s.full + 8u * slot);
                            }
                            skip(1);
                        }
                    }
                }
            }
        };
        auto fetch_async = [&]() -> int { return lane == 0 ? atomicAdd(p.counter, 1) : 0; };
        auto load_rec = [&](int cell) -> int {
            return cell < p.n_kin ? __ldg(reinterpret_cast<const int*>(p.cells + cell) + lane) : 0;
        };
        int cur = __shfl_sync(0xffffffffu, fetch_async(), 0);
        int rec = load_rec(cur);
        for (int ncell = 0;; ncell++) {
            const int cs = ncell % CELL_SLOTS;
            int* hdr = reinterpret_cast<int*>(smem_raw + s.cells + (size_t)cs * cell_bytes);
            smbar_wait(sb + s.cempty + 8u * cs, (uint32_t)(((ncell / CELL_SLOTS) & 1) ^ 1));
            if (cur >= p.n_kin) {
                if (lane == 0) { hdr[2] = CK_STOP; smbar_arrive(sb + s.cfull + 8u * cs); }
                break;
            }
            // The next ticket is drawn now -- late enough that the cells in flight stay close in slab order, early
            // enough that the atomic and the record load (two dependent global round trips) hide behind the copies.
            const int nxt_raw = fetch_async();
            const int level = __shfl_sync(0xffffffffu, rec, 24), flags = __shfl_sync(0xffffffffu, rec, 25);
            const bool ringable = (flags & CELL_NOFLUID) != 0 || (FLUID && (flags & CELL_RINGFLUID) != 0);
            // which octants have a 2:1 upwind face, on which axes; which upwind sources are fluid leaves (computed by the
            // consumers, not copied): 3 bits per octant, precomputed by the flattener
            const int masks = ringable ? __shfl_sync(0xffffffffu, rec, 26) : 0;
            const int fmasks = FLUID && ringable ? __shfl_sync(0xffffffffu, rec, 27) : 0;
            const int mbits = (int)(__ballot_sync(0xffffffffu, lane < 8 && ((masks >> (3 * lane)) & 7) != 0) & 0xffu);
            hdr[HDR_REC + lane] = rec;
            if (lane == 0) { hdr[0] = cur; hdr[1] = level; hdr[2] = ringable ? CK_RING : CK_GATHER; hdr[3] = mbits; hdr[4] = masks; hdr[5] = fmasks; }
            __syncwarp();
            if (lane == 0) {
                const uint32_t cf = sb + s.cfull + 8u * cs;
                if (p.collide) {
                    smbar_arrive_expect_tx(cf, tab_bytes);
                    sbulk_g2s(sb + s.cells + cs * cell_bytes + HDR_INTS * 4, reinterpret_cast<const T*>(p.tabs) + (int64_t)cur * tabn,
                              tab_bytes, cf);
                } else {
                    smbar_arrive(cf);
                }
            }
            const int nxt = __shfl_sync(0xffffffffu, nxt_raw, 0);
            const int nrec = load_rec(nxt);  // in flight while this cell's copies are issued
            if (ringable) issue(cur, rec, masks, fmasks, 0, 8);
            cur = nxt;
            rec = nrec;
        }
        return;
    }

    // ---------------------------------------------------- consumer warps: group g takes stages n = g (mod NG)
    const int g = warp / GW;
    const int r = (warp % GW) * 32 + lane;  // row inside a stage
    const bool active = r < NRQ;
    // (|xi_y|, |xi_z| of the row are re-read from shared memory where needed: registers are what this kernel is short of)
    const double2* ayz = reinterpret_cast<const double2*>(smem_raw + s.ayz);
    int ry[NQ], rz[NQ];
#pragma unroll
    for (int q = 0; q < NQ; q++) {
        const int row = active ? q * NRQ + r : 0;
        ry[q] = row % p.nh[1]; rz[q] = row / p.nh[1];
    }
    const uint32_t inv_ns = (65536u + (uint32_t)NS - 1u) / (uint32_t)NS;  // x / NS = (x * inv_ns) >> 16 for x < 128
    int slot0 = 0, gslot0 = 0, turn0 = 0;  // ring cursor, slots consumed so far, stage counter mod NG at the cell's start
    uint32_t ph0 = 0;
    for (int ncell = 0;; ncell++) {
        const int cs = ncell % CELL_SLOTS;
        const uint32_t hdr = s.cells + cs * cell_bytes;
        smbar_wait(sb + s.cfull + 8u * cs, (uint32_t)((ncell / CELL_SLOTS) & 1));
        const int4 h0 = *reinterpret_cast<const int4*>(smem_raw + hdr);
        const int kind = h0.z;
        if (kind == CK_STOP) break;
        const int cell = h0.x;
        const T* tab = reinterpret_cast<const T*>(smem_raw + hdr + HDR_INTS * 4);
        const double dth = p.dt * p.inv_len * (double)(1 << h0.y);  // dt / h
        const int mbits = h0.w;  // 1 bit per octant: it has a 2:1 upwind face
        const int masks = *reinterpret_cast<const int*>(smem_raw + hdr + 16);  // 3 bits per octant: on which axes
        const int fmasks = FLUID ? *reinterpret_cast<const int*>(smem_raw + hdr + 20) : 0;  // ... the source is a fluid leaf
        RowCtx<T, NQ> rc;
        rc.omega = p.collide ? tab[6 * nhp] : T(0);
        const double om1 = 1.0 - (double)rc.omega;
        rc.sx = (T)(om1 * dth);
        const double omd = om1 * dth;
        if (NQ == 1) {  // one row per thread and cell: its coefficients are formed once per cell (else per stage, below)
            const double2 yz = ayz[active ? r : 0];
            rc.base[0] = (T)(om1 - omd * (yz.x + yz.y));
            rc.cy[0] = (T)(omd * yz.x);
            rc.cz[0] = (T)(omd * yz.y);
        }
        T* const gcell = reinterpret_cast<T*>(p.f_out) + (int64_t)cell * p.Nv;
        // this group's stages of the cell: first, first + NG, ...  (stage = octant * NQ + row block)
        int first = g - turn0;
        if (first < 0) first += NG;
        double S[MAXST][4];  // the row sums of this thread's stages (registers: the loops over them are unrolled)
#pragma unroll
        for (int i = 0; i < MAXST; i++) {
            const int stg = first + i * NG;
            S[i][0] = S[i][1] = S[i][2] = S[i][3] = 0.0;
            if (stg < 8 * NQ) {
                const int o = stg / NQ, q = stg % NQ;
                const int mask = (masks >> (3 * o)) & 7;
                const T* gxrow = tab + (o & 1) * nhp;
                T* const gdst = gcell + (int64_t)o * CH + (int64_t)(q * NRQ + r) * NHX;
                T wb = T(0);
                // this stage's row block: picked by selects, not by indexing (NQ <= 2; indexing would put the arrays in
                // local memory)
                RowCtx<T, 1> rq;
                if (NQ == 1) {
                    rq.base[0] = rc.base[0]; rq.cy[0] = rc.cy[0]; rq.cz[0] = rc.cz[0];
                } else {  // several row blocks: form the row's coefficients here rather than keep NQ sets in registers
                    const double2 yz = ayz[active ? q * NRQ + r : 0];
                    rq.base[0] = (T)(om1 - omd * (yz.x + yz.y));
                    rq.cy[0] = (T)(omd * yz.x);
                    rq.cz[0] = (T)(omd * yz.y);
                }
                rq.sx = rc.sx; rq.omega = rc.omega;
                const int ryq = NQ > 1 && q ? ry[NQ - 1] : ry[0], rzq = NQ > 1 && q ? rz[NQ - 1] : rz[0];
                if (p.collide) wb = rc.omega * (tab[(4 + ((o >> 2) & 1)) * nhp + rzq] * tab[(2 + ((o >> 1) & 1)) * nhp + ryq]);
                if (kind == CK_RING) {
                    // ring slots taken by the stages before this one: one each, four where the octant has a 2:1 face
                    const int before = stg + 3 * (NQ * __popc(mbits & ((1 << o) - 1)) + (mask ? q : 0));
                    const int lin = slot0 + before;
                    const int wraps = (int)(((uint32_t)lin * inv_ns) >> 16);
                    int slot = lin - wraps * NS;
                    uint32_t ph = ph0 ^ (uint32_t)(wraps & 1);
                    // the producer must have armed the stage's last slot before its barrier's parity means anything
                    const int need = gslot0 + before + (mask ? 4 : 1);
                    for (uint32_t spins = 0; slds_i32_volatile(sb + s.issued) < need; ) {
                        __nanosleep(64);
                        if (++spins > (1u << 24)) __trap();   // seconds without progress: a protocol bug must not hang the GPU
                    }
                    __threadfence_block();
                    smbar_wait(sb + s.full + 8u * slot, ph);
                    T* const st = reinterpret_cast<T*>(smem_raw + s.ring + (size_t)slot * slot_bytes) + (size_t)r * NHX;
                    if (mask) {
                        // 2:1 face (reading G3): the next three slots bring sources 1..3 of the axes in `mask`; they are
                        // added, in order, onto source 0 where it lies in this slot (a thread touches its own row only)
                        int sl = slot;
                        uint32_t sp = ph;
#pragma unroll 1
                        for (int j = 1; j < 4; j++) {
                            if (++sl == NS) { sl = 0; sp ^= 1u; }
                            smbar_wait(sb + s.full + 8u * sl, sp);
                            if (active) {
                                const T* se = reinterpret_cast<const T*>(smem_raw + s.ring + (size_t)sl * slot_bytes) + (size_t)r * NHX;
#pragma unroll 1
                                for (int t = 0; t < 3; t++) {
                                    if ((mask >> t) & 1) {
#pragma unroll
                                        for (int jj = 0; jj < RV; jj++) {
                                            T v[VEC], x[VEC];
                                            lds16(se + t * pe + jj * VEC, v);
                                            lds16(st + (t + 1) * pe + jj * VEC, x);
#pragma unroll
                                            for (int ii = 0; ii < VEC; ii++) x[ii] += v[ii];
                                            sts16(st + (t + 1) * pe + jj * VEC, x);
                                        }
                                    }
                                }
                            }
                            __syncwarp();
                            if (lane == 0) smbar_arrive(sb + s.empty + 8u * sl);
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
                                        for (int ii = 0; ii < VEC; ii++) x[ii] *= T(0.25);
                                        sts16(st + (t + 1) * pe + jj * VEC, x);
                                    }
                                }
                            }
                        }
                    }
                    // a slot written with ordinary stores: order them before the bulk copy that refills it
                    if (mask) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    FluidStreams fs;
                    fs.fm = FLUID ? (fmasks >> (3 * o)) & 7 : 0;
                    fs.o = o; fs.ry = ryq; fs.rz = rzq;
                    fs.rec = reinterpret_cast<const int*>(smem_raw + hdr + HDR_REC * 4);
                    row_from_ring<T, NHX, 1, EARLY, FLUID>(p, rq, 0, wb, st, pe, gxrow, gdst, active, lane, sb + s.empty + 8u * slot, fs,
                                                     S[i][0], S[i][1], S[i][2], S[i][3]);
                } else if (active) {
                    row_from_gather<T, NHX, 1>(p, rq, 0, wb, o, CH, q * NRQ + r, ryq, rzq, reinterpret_cast<const int*>(p.cells + cell),
                                                fin, cell, gxrow, gdst, S[i][0], S[i][1], S[i][2], S[i][3]);
                }
            }
        }
        if (kind == CK_RING) {
            const int total = 8 * NQ + 3 * NQ * __popc(mbits);
            const int lin = slot0 + total;
            const int wraps = (int)(((uint32_t)lin * inv_ns) >> 16);
            slot0 = lin - wraps * NS;
            ph0 ^= (uint32_t)(wraps & 1);
            gslot0 += total;
        }
        turn0 = (turn0 + 8 * NQ) % NG;
        // fold the y/z weights and signs into the row sums (a2'), then the warp's partial sums; the warp that delivers
        // last adds all of them up and writes the cell's sums
        double acc[35];
#pragma unroll
        for (int i = 0; i < 35; i++) acc[i] = 0.0;
#pragma unroll
        for (int i = 0; i < MAXST; i++) {
            const int stg = first + i * NG;
            if (stg < 8 * NQ && active) {
                const double2 yz = ayz[(stg % NQ) * NRQ + r];
                fold_row_rt(stg / NQ, S[i][0], S[i][1], S[i][2], S[i][3], yz.x, yz.y, acc);
            }
        }
        warp_store_sums(acc, reinterpret_cast<double*>(smem_raw + s.red) + ((size_t)cs * NW + warp) * SUMS_STRIDE, lane);
        __threadfence_block();
        __syncwarp();
        int last = 0;
        if (lane == 0) last = atomicAdd(reinterpret_cast<int*>(smem_raw + s.cnt) + cs, 1) == NW - 1;
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {
            __threadfence_block();
            if (lane < SUMS_STRIDE / 2) {
                double2 t = make_double2(0.0, 0.0);
                const double2* src = reinterpret_cast<const double2*>(smem_raw + s.red + (size_t)cs * NW * SUMS_STRIDE * 8) + lane;
#pragma unroll
                for (int w = 0; w < NW; w++) {
                    const double2 v = src[w * (SUMS_STRIDE / 2)];
                    t.x += v.x; t.y += v.y;
                }
                reinterpret_cast<double2*>(p.sums_out + (int64_t)cell * SUMS_STRIDE)[lane] = t;
            }
            if (lane == 0) reinterpret_cast<int*>(smem_raw + s.cnt)[cs] = 0;
            __syncwarp();
        }
        if (lane == 0) smbar_arrive(sb + s.cempty + 8u * cs);
    }
}

constexpr size_t ROWS_SMEM_MAX = 227 * 1024;

// the instantiations: (storage type, nh_x, warps per group, groups, row blocks per octant chunk, early release).
// Tried and slower on config 4 (fp32): two groups with early release (11.7 vs 9.6 ms on the quarter-size mesh), half
// chunks per stage with five groups (14.8 ms), the same with early release (18.6 ms).
struct RowsVariant { int storage, nhx, gw, ng, nq, early; };
constexpr RowsVariant ROWS_VARIANTS[] = {
    {UFS_STORE_F32, 12, 5, 3, 1, 0},
    {UFS_STORE_F64, 12, 3, 5, 2, 0},
    {UFS_STORE_F64, 6, 2, 4, 1, 1},
};
constexpr int N_ROWS_VARIANTS = sizeof(ROWS_VARIANTS) / sizeof(ROWS_VARIANTS[0]);
bool rows_variant_fits(const RowsVariant& rv, int storage, const VelLayout& v) {
    const int nr = v.nh[1] * v.nh[2];
    return rv.storage == storage && rv.nhx == v.nh[0] && nr % rv.nq == 0 && nr / rv.nq <= rv.gw * 32;
}
int rows_variant(int storage, const VelLayout& v) {
    if (!v.fast) return -1;
    for (int i = 0; i < N_ROWS_VARIANTS; i++)
        if (rows_variant_fits(ROWS_VARIANTS[i], storage, v)) return i;
    return -1;
}

template <typename T, int NHX, int GW, int NG, int NQ, bool EARLY, bool FLUID>
cudaError_t launch_rows_t2(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    auto k = k_rows<T, NHX, GW, NG, NQ, EARLY, FLUID>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    const int grid = p.n_kin < plan.grid ? p.n_kin : plan.grid;
    StepParams q = p;
    {
        const int nr = p.nh[1] * p.nh[2];
        const RowsSmem m = rows_map(sizeof(T), p.ring_stages, (size_t)4 * (nr / NQ) * NHX * sizeof(T), NG * GW, tabn_of(p.nh), nr);
        const uint32_t v[11] = {m.ring, m.cells, m.red, m.ayz, m.full, m.empty, m.cfull, m.cempty, m.cnt, m.issued, m.total};
        for (int i = 0; i < 11; i++) q.smap[i] = v[i];
    }
    if (plan.ev0) cudaEventRecord(plan.ev0, st);
    k<<<grid, (NG * GW + 1) * 32, plan.smem_bytes, st>>>(q);
    if (plan.ev1) cudaEventRecord(plan.ev1, st);
    return cudaGetLastError();
}

template <typename T, int NHX, int GW, int NG, int NQ, bool EARLY>
cudaError_t launch_rows_t(const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    return p.fluid ? launch_rows_t2<T, NHX, GW, NG, NQ, EARLY, true>(plan, p, st)
                   : launch_rows_t2<T, NHX, GW, NG, NQ, EARLY, false>(plan, p, st);
}

}  // namespace

// Launch geometry of the row kernel for this storage type / velocity grid, or false if no instantiation fits (the
// one-vector-per-thread kernel of step_stream.cu, then the one-CTA-per-cell kernels of kernels.cu, take over).
bool rows_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan) {
    const int vi = rows_variant(storage, v);
    if (vi < 0) return false;
    const RowsVariant* rv = &ROWS_VARIANTS[vi];
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
    plan->ncw = vi;            // which instantiation
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
    switch (plan.ncw) {
        // (meshes with fluid leaves get the instantiation that computes fluid streams; the others keep the leaner code)
        case 0: return launch_rows_t<float, 12, 5, 3, 1, false>(plan, p, st);
        case 1: return launch_rows_t<double, 12, 3, 5, 2, false>(plan, p, st);
        case 2: return launch_rows_t<double, 6, 2, 4, 1, true>(plan, p, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace ufs
