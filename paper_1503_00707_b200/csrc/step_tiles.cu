// step_tiles.cu -- k_tiles: the streaming pass of the DVM step (scheme: step_stream.cu) over TILES of up to eight
// consecutive slabs.
//
// Why tiles.  For one velocity octant (sign group) a cell reads four chunks: its own and the upwind
// cell's on each axis (first-order stencil records).  For the eight leaf children of one parent
// (consecutive in N-order) half of those upwind cells are siblings, so a tile that holds the octet needs
// 20 distinct chunks per octant instead of 32; a coarser neighbour serves four cells with one chunk.  The flattener
// lists the distinct chunks ("pieces") of every tile and octant (flatten.hpp); here they arrive once by cp.async.bulk
// and every consumer thread picks its four streams by index.
//
// Work decomposition.  A stage is (tile, row block q, octant o): NRP = 48 rows of every piece (a third of a 12x12-row
// chunk), 8 cells x 48 rows = one velocity row per consumer thread (12 warps).  Pieces live in a ring of NP piece
// slots allocated in stage order (a stage takes np <= pmax consecutive slots, modulo NP); stage k uses barrier pair
// k mod NSTG.  Four producer warps issue the copies of every stage together (piece i by lane i/4 of warp i%4), one of
// them also draws the tile tickets and publishes the tile header (cells, levels, Maxwellian factor tables of k_prep).
// A thread finishes its row exactly like k_rows:  f' = B f + Cx_k (fX - f) + Cy fY + Cz fZ + W gx_k  (Eq. 2,
// PAPER.md:103, with the BGK relaxation of PAPER.md:231 folded in), one store, four fp64 x sums of the row.  Over the
// eight octants of a row block the row sums are kept as 16 sign-weighted combinations (no octant-indexed registers);
// after the block they are expanded with the row's |xi_y|, |xi_z| to the cell's 35 velocity sums (stream_common.cuh),
// reduced over 16 lanes by a halving butterfly and added into shared memory; the last block writes them out.
//
// Partitioned mesh, fused ghost exchange (PUSH instantiation; include/ufs_dvm.h: ufs_dvm_halo_push_setup; PAPER.md:185-187 does
// this exchange as messages after the step): a thread that has formed a row of a cell some peer rank lists as a ghost cell
// stores the same registers a second time, into that peer's ghost slab of its next f (peer memory), and the thread that
// writes a cell's sums stores them into the peer's ghost row as well.  The flattener lists, per tile, one push entry per
// (cell, peer); tiles with entries come first and only they are stepped by this instantiation (launch_tiles).
#include <cmath>

#include "device_util.cuh"
#include "kernels.cuh"
#include "stream_common.cuh"

namespace ufs {
namespace {

constexpr int THX = 12;                 // values of a row (nh_x)
// Geometry of a piece by storage type.  fp32: 48 rows of 48 bytes, one consumer thread per row.  fp64: a row is 96 bytes,
// and one row per lane read with 16-byte loads hits only four distinct 16-byte offsets modulo 128 in a quarter-warp
// (96 r mod 128): a 2-way shared-memory bank conflict on every load, 46 % of the wavefronts (profiles/r2_full_config2.md).
// So fp64 takes 24 rows per piece and one thread per HALF row: lanes are 48 bytes apart as for fp32 (conflict-free), a
// piece is 2304 bytes for both types, and the ring is as many stages deep for fp64 as for fp32.
template <typename T> struct Geo { static constexpr int NRP = 48, HALVES = 1; };
template <> struct Geo<double> { static constexpr int NRP = 24, HALVES = 2; };
constexpr int PIECE_BYTES = 2304;       // = NRP * THX * sizeof(T) for both
constexpr int CELL_THREADS = 48;        // consumer threads of a cell = NRP * HALVES
__host__ __device__ constexpr int nrp_of(size_t elem) { return elem == 8 ? 24 : 48; }
constexpr int N_PROD = 4;               // producer warps: warps 0..3
constexpr int N_CONS = 12;              // consumer warps: warps 4..15
constexpr int NSTG = 8;                 // stage barrier pairs / stage descriptors
// Register re-allocation between the warp groups (setmaxnreg): the CTA starts with 128 registers per thread (512 threads,
// the whole file); the four producer warps give back down to REGS_PROD, the twelve consumer warps take REGS_CONS:
// 4 * 32 * 80 + 12 * 32 * 144 = 65 536.
constexpr int REGS_PROD = 80, REGS_CONS = 144;
constexpr int TSLOTS = 3;               // tile header slots
constexpr int DESC_BYTES = TILE_CELLS * CELLIDX_BYTES + 16;   // cell index tables, then the stage's first piece slot
constexpr int THDR_NEXT = 36;           // tile header: TileHdr (32 B), tile id (or -1: stop), next tile id,
constexpr int THDR_TAB = 64;            //   factor tables [8][tabn] of the storage type
constexpr int FLUID_PIECE_STRIDE = 64;               // ... padded to 512 bytes in the device table of all fluid pieces
constexpr int RED_DOUBLES = TILE_CELLS * 3 * SUMS_STRIDE;     // partial sums: [cell][16-lane group][36]

struct TilesSmem { uint32_t ring, desc, thdr, red, full, empty, tinfo, ttab, tempty, total, thdr_bytes; };
__host__ __device__ inline TilesSmem tiles_map(size_t elem, int np, int tabn) {
    TilesSmem s;
    size_t off = 0;
    s.ring = 0; off += (size_t)np * PIECE_BYTES;
    (void)elem;
    s.desc = (uint32_t)off; off += (size_t)NSTG * DESC_BYTES;
    off = (off + 127) & ~(size_t)127;
    s.thdr_bytes = (uint32_t)((THDR_TAB + (size_t)TILE_CELLS * tabn * elem + 127) & ~(size_t)127);
    s.thdr = (uint32_t)off; off += (size_t)TSLOTS * s.thdr_bytes;
    s.red = (uint32_t)off; off += (size_t)2 * RED_DOUBLES * 8;
    s.full = (uint32_t)off; off += NSTG * 8;
    s.empty = (uint32_t)off; off += NSTG * 8;
    s.tinfo = (uint32_t)off; off += TSLOTS * 8;
    s.ttab = (uint32_t)off; off += TSLOTS * 8;
    s.tempty = (uint32_t)off; off += TSLOTS * 8;
    s.total = (uint32_t)((off + 127) & ~(size_t)127);
    return s;
}

template <typename T> __device__ __forceinline__ T tx_of(const StepParams& p, int k);
template <> __device__ __forceinline__ float tx_of<float>(const StepParams& p, int k) { return p.xf[k]; }

// halving butterfly over the 16 lanes of a group: 36 -> 18 -> 9 -> 5 -> 3 values per lane (stream_common.cuh: halve)
__device__ __forceinline__ void group16_reduce(double (&v)[36], int lane) {
    halve<36, 8>(v, lane);
    halve<18, 4>(v, lane);
    halve<9, 2>(v, lane);
    halve<5, 1>(v, lane);
}

template <typename T, bool FLUID, bool SUMS_ONLY, bool PUSH = false>
__global__ void __launch_bounds__((N_PROD + N_CONS) * 32, 1) k_tiles(const StepParams p) {
    constexpr int NRP = Geo<T>::NRP, HALVES = Geo<T>::HALVES;
    constexpr int XT = THX / HALVES;                    // x ranks of a consumer thread: the whole row, or half of it
    constexpr int VEC = V16<T>::N, RV = XT / VEC;       // ... = three 16-byte vectors for both storage types
    static_assert(NRP * THX * sizeof(T) == PIECE_BYTES && NRP * HALVES == CELL_THREADS && RV == 3, "piece geometry");
    constexpr bool PACKED = sizeof(T) == 4 && !SUMS_ONLY;   // fp32 storage: packed two-value arithmetic in the row update
    constexpr uint32_t ROWB = THX * sizeof(T);          // bytes of a row
    constexpr uint32_t PB = NRP * ROWB;                 // bytes of a piece
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const uint32_t sb = smem_u32(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NP = p.ring_stages;                       // piece slots of the ring
    const int nhp = nhp_of(p.nh), tabn = tabn_of(p.nh);
    const int NR = p.nh[1] * p.nh[2];                   // rows of an octant chunk
    const int NQ = NR / NRP;                            // row blocks
    const int CH = NR * THX;                            // elements of an octant chunk
    // shared-memory map (kernel parameters: constant bank, no registers)
    const uint32_t o_desc = p.smap[1], o_thdr = p.smap[2], o_red = p.smap[3], o_full = p.smap[4], o_empty = p.smap[5],
                   o_tinfo = p.smap[6], o_ttab = p.smap[7], o_tempty = p.smap[8], thdr_bytes = p.smap[10];

    if (tid == 0) {
        for (int i = 0; i < NSTG; i++) {
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + o_full) + i, N_PROD);
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + o_empty) + i, N_CONS);
        }
        for (int i = 0; i < TSLOTS; i++) {
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + o_tinfo) + i, 1);
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + o_ttab) + i, 1);
            mbar_init(reinterpret_cast<uint64_t*>(smem_raw + o_tempty) + i, N_CONS + N_PROD - 1);
        }
        mbar_init_fence();
        if (blockIdx.x == 0) *p.counter_reset = 0;  // the other launch parity's ticket counter
    }
    __syncthreads();

    if (warp < N_PROD) {
        // =========================================================== producer warps
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_PROD));
        const int w = warp;
        const T* fin = reinterpret_cast<const T*>(p.f_in);
        const int my_piece = 4 * lane + w;          // the piece of every stage this lane copies
        uint32_t code[8], code_nx[8];               // its source chunk per octant: current / next tile
        int hw_nx = 0;                              // (warp 0, lanes 0..7) word `lane` of the next tile's TileHdr
        int tk_cur = 0, tk_nx_raw = 0;              // (warp 0) ticket of the current tile; lane 0: the next tile's (atomic in flight)
        // ring bookkeeping, identical in the four warps: pieces allocated / released so far, next stage to be released
        uint32_t alloc = 0, rel = 0;
        int head = 0;
        int k = 0, r = 0, rq = 0;                   // stage counters: next to issue, next to release, r within its tile
        bool r_prev = false;                        // stage r belongs to the previous tile
        unsigned long long np_cur = 0, np_prev = 0; // pieces per octant (8 bytes) of the current / previous tile
        auto load_codes = [&](int tile, uint32_t (&c)[8]) {
#pragma unroll
            for (int o = 0; o < 8; o++)
                c[o] = (!SUMS_ONLY && tile < p.n_tiles && my_piece < p.tile_pmax)
                           ? __ldg(p.tile_pieces + ((size_t)tile * 8 + o) * p.tile_pmax + my_piece) : 0u;
        };
        if (w == 0) {
            int t0 = 0, t1 = 0;
            if (lane == 0) { t0 = atomicAdd(p.counter, 1); t1 = atomicAdd(p.counter, 1); }
            tk_cur = __shfl_sync(0xffffffffu, t0, 0);
            tk_nx_raw = t1;
            hw_nx = (lane < 8 && tk_cur < p.n_tiles) ? __ldg(reinterpret_cast<const int*>(p.tile_hdr + tk_cur) + lane) : 0;
        }
        for (int n = 0;; n++) {
            const int ts = n % TSLOTS;
            const uint32_t tph = (uint32_t)((n / TSLOTS) & 1);
            const uint32_t hdr = sb + o_thdr + ts * thdr_bytes;
            int tile, next, s0, nc;
            if (w == 0) {
                // publish the header of tile n: its TileHdr came in a tile ago, the ticket of tile n + 1 as well
                smbar_wait(sb + o_tempty + 8u * ts, tph ^ 1u);
                tile = tk_cur < p.n_tiles ? tk_cur : -1;
                next = __shfl_sync(0xffffffffu, tk_nx_raw, 0);   // drawn a tile ago
                const int hw = hw_nx;
                if (lane < 8) ssts_i32(hdr + 4u * lane, hw);
                if (lane == 8) ssts_i32(hdr + 32u, tile);
                if (lane == 9) ssts_i32(hdr + THDR_NEXT, next);
                s0 = __shfl_sync(0xffffffffu, hw, 0);
                nc = __shfl_sync(0xffffffffu, hw, 1);
                np_prev = np_cur;
                np_cur = (unsigned long long)(uint32_t)__shfl_sync(0xffffffffu, hw, 2)
                         | ((unsigned long long)(uint32_t)__shfl_sync(0xffffffffu, hw, 3) << 32);
                __syncwarp();
                if (lane == 0) {
                    smbar_arrive(sb + o_tinfo + 8u * ts);
                    const uint32_t tb = sb + o_ttab + 8u * ts;
                    const uint32_t tab_bytes = (p.collide && !SUMS_ONLY && tile >= 0) ? (uint32_t)(nc * tabn) * (uint32_t)sizeof(T) : 0u;
                    if (tab_bytes) {
                        smbar_arrive_expect_tx(tb, tab_bytes);
                        sbulk_g2s(hdr + THDR_TAB, reinterpret_cast<const T*>(p.tabs) + (size_t)s0 * tabn, tab_bytes, tb);
                    } else {
                        smbar_arrive(tb);
                    }
                }
                if (tile < 0) break;
                // the ticket after the next (its result is read a tile from now) and the next tile's header words
                tk_cur = next;
                if (lane == 0) tk_nx_raw = atomicAdd(p.counter, 1);
                hw_nx = (lane < 8 && next < p.n_tiles) ? __ldg(reinterpret_cast<const int*>(p.tile_hdr + next) + lane) : 0;
            } else {
                smbar_wait(sb + o_tinfo + 8u * ts, tph);
                s0 = slds_i32(hdr + 0u);
                nc = slds_i32(hdr + 4u);
                np_prev = np_cur;
                np_cur = (unsigned long long)(uint32_t)slds_i32(hdr + 8u) | ((unsigned long long)(uint32_t)slds_i32(hdr + 12u) << 32);
                tile = slds_i32(hdr + 32u);
                next = slds_i32(hdr + THDR_NEXT);
                __syncwarp();
                if (lane == 0) smbar_arrive(sb + o_tempty + 8u * ts);   // everything needed is in registers
                if (tile < 0) break;
            }
            if (SUMS_ONLY) np_cur = (unsigned long long)nc * 0x0101010101010101ull;   // own chunks only
            if (n == 0) load_codes(tile, code);
            else {
#pragma unroll
                for (int o = 0; o < 8; o++) code[o] = code_nx[o];
            }
            load_codes(next, code_nx);   // in flight during this tile's stages
            r_prev = (r < k);            // stages not yet released belong to the tile that just ended (8 NQ >= NSTG)
            for (int q = 0; q < NQ; q++) {
#pragma unroll
                for (int o = 0; o < 8; o++) {
                    const int npk = (int)((np_cur >> (8 * o)) & 0xffull);
                    // ring space: piece slots and the barrier pair of stage k
                    while (k - r >= NSTG || alloc + (uint32_t)npk - rel > (uint32_t)NP) {
                        smbar_wait_relaxed(sb + o_empty + 8u * (r % NSTG), (uint32_t)((r / NSTG) & 1));
                        rel += (uint32_t)(((r_prev ? np_prev : np_cur) >> (8 * (rq & 7))) & 0xffull);
                        r++;
                        if (++rq == 8 * NQ) { rq = 0; r_prev = false; }
                    }
                    const int slot = k % NSTG;
                    const uint32_t fb = sb + o_full + 8u * slot;
                    const uint32_t dsc = sb + o_desc + slot * DESC_BYTES;
                    if constexpr (!FLUID) {
                        const int mine = npk > w ? (npk + 3 - w) >> 2 : 0;   // pieces this warp copies
                        // (test hook, UFS_DVM_TEST_STALL: one producer warp withholds its arrival on the fourth stage; the
                        // consumers' wait then runs into the watchdog, include/ufs_dvm.h)
                        if (lane == 0 && !(p.smap[11] && k == 3 && w == 1)) {
                            if (w == 0) ssts_i32(dsc + TILE_CELLS * CELLIDX_BYTES, head);
                            const uint32_t extra = (w == 0 && !SUMS_ONLY) ? (uint32_t)(TILE_CELLS * CELLIDX_BYTES) : 0u;
                            smbar_arrive_expect_tx(fb, (uint32_t)mine * PB + extra);
                            if (extra) sbulk_g2s(dsc, p.tile_cellidx + ((size_t)tile * 8 + o) * (TILE_CELLS * CELLIDX_BYTES), extra, fb);
                        }
                        __syncwarp();
                        if (my_piece < npk) {
                            const uint32_t c = SUMS_ONLY ? (uint32_t)((s0 + my_piece) * 8 + o) : code[o];
                            const T* src = ((c & PIECE_TABLE) ? reinterpret_cast<const T*>(p.tables) : fin)
                                           + (size_t)(c & PIECE_INDEX) * (size_t)CH + (size_t)q * (NRP * THX);
                            int ps = head + my_piece;
                            if (ps >= NP) ps -= NP;
                            sbulk_g2s(sb + (uint32_t)ps * PB, src, PB, fb);
                        }
                    } else {
                        // meshes with FLUID leaves: a piece is a bulk copy of a chunk's rows, or of a fluid ghost's factor rows
                        // for this sign group and row block (512 bytes from the table tiles_fluid_pieces() built)
                        const bool have = my_piece < npk;
                        const uint32_t c = have ? code[o] : 0u;
                        const bool is_fl = have && (c & PIECE_FLUID);
                        const int n_fl = __popc(__ballot_sync(0xffffffffu, is_fl));
                        const int n_copy = __popc(__ballot_sync(0xffffffffu, have && !is_fl));
                        if (lane == 0 && !(p.smap[11] && k == 3 && w == 1)) {   // (test hook: see the other branch)
                            if (w == 0) ssts_i32(dsc + TILE_CELLS * CELLIDX_BYTES, head);
                            const uint32_t extra = w == 0 ? (uint32_t)(TILE_CELLS * CELLIDX_BYTES) : 0u;
                            smbar_arrive_expect_tx(fb, (uint32_t)n_copy * PB + (uint32_t)n_fl * (uint32_t)(FLUID_PIECE_STRIDE * 8) + extra);
                            if (extra) sbulk_g2s(dsc, p.tile_cellidx + ((size_t)tile * 8 + o) * (TILE_CELLS * CELLIDX_BYTES), extra, fb);
                        }
                        __syncwarp();
                        if (have) {
                            int ps = head + my_piece;
                            if (ps >= NP) ps -= NP;
                            if (is_fl) {
                                const double* src = p.fluid_pieces + ((size_t)(c & PIECE_INDEX) * (size_t)NQ + (size_t)q) * FLUID_PIECE_STRIDE;
                                sbulk_g2s(sb + (uint32_t)ps * PB, src, (uint32_t)(FLUID_PIECE_STRIDE * 8), fb);
                            } else {
                                const T* src = ((c & PIECE_TABLE) ? reinterpret_cast<const T*>(p.tables) : fin)
                                               + (size_t)(c & PIECE_INDEX) * (size_t)CH + (size_t)q * (NRP * THX);
                                sbulk_g2s(sb + (uint32_t)ps * PB, src, PB, fb);
                            }
                        }
                    }
                    head += npk;
                    if (head >= NP) head -= NP;
                    alloc += (uint32_t)npk;
                    k++;
                }
            }
        }
        return;
    }

    // =============================================================== consumer warps: thread = (cell c, row r of the piece)
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_CONS));
    const int ct = tid - N_PROD * 32;
    const int c = ct / CELL_THREADS, hr = ct % CELL_THREADS;
    const int rr = hr / HALVES;                      // row of the piece
    const int k0 = (hr % HALVES) * XT;               // first x rank of this thread
    const int gi = hr >> 4;                          // 16-lane group of the cell
    const int ry = rr % p.nh[1], rzl = rr / p.nh[1]; // rank of |xi_y|; rank of |xi_z| inside the row block
    const double ay = p.yabs[ry];
    const uint32_t rowoff = (uint32_t)rr * ROWB + (uint32_t)k0 * (uint32_t)sizeof(T);   // = 48 hr: lanes 48 bytes apart
    const int triple = (warp - N_PROD) / 3;          // three warps share two cells: named barrier 1 + triple
    // fp64 (half rows): the thread's six x ranks are fixed for the whole run, |xi_x| of them stays in registers
    double txr[HALVES == 2 ? XT : 1];
    if constexpr (HALVES == 2) {
#pragma unroll
        for (int i = 0; i < XT; i++) {
            txr[i] = p.xpow[0][k0 + i];
            asm volatile("" : "+d"(txr[i]));
        }
    }
    int k = 0;
    for (int n = 0;; n++) {
        const int ts = n % TSLOTS;
        const uint32_t hdr = o_thdr + ts * thdr_bytes;   // offset from smem_raw
        smbar_wait(sb + o_ttab + 8u * ts, (uint32_t)((n / TSLOTS) & 1));
        const int tile = *reinterpret_cast<const int*>(smem_raw + hdr + 32);
        if (tile < 0) break;
        const int s0 = *reinterpret_cast<const int*>(smem_raw + hdr);
        const int nc = *reinterpret_cast<const int*>(smem_raw + hdr + 4);
        const bool active = c < nc;
        const int level = smem_raw[hdr + 16 + c];
        const T* tab = reinterpret_cast<const T*>(smem_raw + hdr + THDR_TAB) + c * tabn;
        const double dth = p.dt * p.inv_len * (double)(1 << level);   // dt / h
        const T omega = (p.collide && !SUMS_ONLY && active) ? tab[6 * nhp] : T(0);
        const double om1 = 1.0 - (double)omega, omd = om1 * dth;
        const T sxc = (T)omd;                         // times |xi_x,k| : the x coefficient
        const T cy = (T)(omd * ay);
        // fp32 storage: the x coefficients of the row, Cx_k = sxc |xi_x,k|, as six packed pairs kept for the whole tile
        float2 cx2[PACKED ? THX / 2 : 1];
        if constexpr (PACKED) {
#pragma unroll
            for (int k = 0; k < THX / 2; k++) {
                cx2[k] = make_float2(sxc * p.xf[2 * k], sxc * p.xf[2 * k + 1]);
                asm volatile("" : "+f"(cx2[k].x), "+f"(cx2[k].y));   // kept in registers, not recomputed per stage
            }
        }
        T* const gcell = reinterpret_cast<T*>(p.f_out) + (int64_t)(s0 + c) * p.Nv;
        // fused ghost exchange: the push entries of this thread's cell (flatten.hpp: PushEntry).  pinfo bits 0..7: the octants
        // some peer needs, bits 8..11: entries; a cell nobody needs (almost all of them) costs one predicate per store
        int pfirst = 0;
        uint32_t pinfo = 0u;
        if constexpr (PUSH) {
            const uint32_t cnts = *reinterpret_cast<const uint32_t*>(smem_raw + hdr + 28);
            if (cnts != 0u && active) {
                pfirst = *reinterpret_cast<const int*>(smem_raw + hdr + 24);
                for (int i = 0; i < c; i++) pfirst += (int)((cnts >> (4 * i)) & 15u);
                const uint32_t pcnt = (cnts >> (4 * c)) & 15u;
                for (uint32_t e = 0; e < pcnt; e++) pinfo |= __ldg(&p.tile_push[pfirst + e].info) & 0xffu;
                pinfo |= pcnt << 8;
            }
        }
        double* const red = reinterpret_cast<double*>(smem_raw + o_red) + (size_t)(n & 1) * RED_DOUBLES + (size_t)(c * 3 + gi) * SUMS_STRIDE;
        for (int q = 0; q < NQ; q++) {
            const int rz = q * (NRP / p.nh[1]) + rzl;
            const double az = p.zabs[rz];
            const T cz = (T)(omd * az);
            const T base = (T)(om1 - omd * (ay + az));
            // ... and the own-value coefficients B - Cx_k:  f' = (B - Cx_k) f + Cx_k fX + Cy fY + Cz fZ + W gx_k
            float2 bx2[PACKED ? THX / 2 : 1];
            float2 cy2, cz2;
            if constexpr (PACKED) {
#pragma unroll
                for (int k = 0; k < THX / 2; k++) {
                    bx2[k] = make_float2(base - cx2[k].x, base - cx2[k].y);
                    asm volatile("" : "+f"(bx2[k].x), "+f"(bx2[k].y));
                }
                cy2 = make_float2(cy, cy);
                cz2 = make_float2(cz, cz);
                asm volatile("" : "+f"(cy2.x), "+f"(cy2.y), "+f"(cz2.x), "+f"(cz2.y));
            }
            // relaxation weights of the row for the two signs of xi_y and of xi_z: W = omega gz[sz][rz] gy[sy][ry]
            T wgy[2] = {T(0), T(0)}, wgz[2] = {T(0), T(0)};
            if (p.collide && !SUMS_ONLY) {
                wgy[0] = omega * tab[2 * nhp + ry]; wgy[1] = omega * tab[3 * nhp + ry];
                wgz[0] = tab[4 * nhp + rz];         wgz[1] = tab[5 * nhp + rz];
            }
            const int row = q * NRP + rr;             // row of the octant chunk
            // the 16 sign-weighted combinations of the row sums s_k = sum_x |xi_x|^k f' over the eight octants
            double E0 = 0, Ey = 0, Ez = 0, Eyz = 0, F0 = 0, Fx = 0, Fy = 0, Fxy = 0, Fz = 0, Fxz = 0, G0 = 0, Gx = 0, Gy = 0, Gz = 0, K0 = 0, Kx = 0;
#pragma unroll 1
            for (int o = 0; o < 8; o++) {
                const int slot = k % NSTG;
                smbar_wait(sb + o_full + 8u * slot, (uint32_t)((k / NSTG) & 1));
                double s0_ = 0, s1_ = 0, s2_ = 0, s3_ = 0;
                // the row's x sums s_r += |xi_x,k|^r d.  fp32: powers from the constant bank (k is a compile-time index);
                // fp64 half rows: Horner with the thread's own |xi_x| (registers; `_dyn`: k known at run time only)
                auto row_sums = [&](double d, int kk) {
                    if constexpr (HALVES == 1) {
                        s0_ += d; s1_ = fma(p.xpow[0][kk], d, s1_); s2_ = fma(p.xpow[1][kk], d, s2_); s3_ = fma(p.xpow[2][kk], d, s3_);
                    } else {
                        const double x = txr[kk], t1 = x * d, t2 = x * t1;
                        s0_ += d; s1_ += t1; s2_ += t2; s3_ = fma(x, t2, s3_);
                    }
                };
                auto row_sums_dyn = [&](double d, int kk) {
                    if constexpr (HALVES == 1) {
                        s0_ += d; s1_ = fma(p.xpow[0][kk], d, s1_); s2_ = fma(p.xpow[1][kk], d, s2_); s3_ = fma(p.xpow[2][kk], d, s3_);
                    } else {
                        const double x = p.xpow[0][k0 + kk], t1 = x * d, t2 = x * t1;
                        s0_ += d; s1_ += t1; s2_ += t2; s3_ = fma(x, t2, s3_);
                    }
                };
                auto xk = [&](int kk) -> T { if constexpr (HALVES == 1) return tx_of<T>(p, kk); else return (T)txr[kk]; };
                auto xk_dyn = [&](int kk) -> T { if constexpr (HALVES == 1) return tx_of<T>(p, kk); else return (T)p.xpow[0][k0 + kk]; };
                if (active) {
                    const unsigned char* dsc = smem_raw + o_desc + slot * DESC_BYTES;
                    const int head = *reinterpret_cast<const int*>(dsc + TILE_CELLS * CELLIDX_BYTES);
                    uint4 ix;
                    if (SUMS_ONLY) ix = make_uint4((uint32_t)c, 0u, 0u, 0u);
                    else ix = *reinterpret_cast<const uint4*>(dsc + c * CELLIDX_BYTES);
                    auto addr_of = [&](uint32_t b) -> const T* {
                        int ps = head + (int)b;
                        if (ps >= NP) ps -= NP;
                        return reinterpret_cast<const T*>(smem_raw + (uint32_t)ps * PB + rowoff);
                    };
                    const T* a_own = addr_of(ix.x & 0xffu);
                    const uint32_t flags = (ix.x >> 8) & 0xffu;
                    T* const gdst = gcell + (int64_t)o * CH + (int64_t)row * THX + k0;
                    // the peers' ghost slabs that take this cell's chunk of octant o: the same row goes there as well
                    const bool po = PUSH && ((pinfo >> o) & 1u);
                    auto push_out = [&](int j, const T (&out)[VEC]) {
                        if constexpr (PUSH) {
                            if (po) {
                                const int pc = (int)(pinfo >> 8);
                                for (int e = 0; e < pc; e++) {
                                    const PushEntry* ent = p.tile_push + pfirst + e;
                                    if ((__ldg(&ent->info) >> o) & 1u)
                                        stg16(reinterpret_cast<T*>(__ldg(reinterpret_cast<const unsigned long long*>(ent->dst) + p.push_parity))
                                                  + (gdst - gcell) + j * VEC, out);
                                }
                            }
                        }
                    };
                    // unrolled row loops keep the row's vectors and push once, after the loop (one cold block per loop)
                    T outs[PUSH ? RV : 1][VEC];
                    auto keep_out = [&](int j, const T (&out)[VEC]) {
                        if constexpr (PUSH) {
#pragma unroll
                            for (int i = 0; i < VEC; i++) outs[j][i] = out[i];
                        }
                    };
                    auto push_row = [&]() {
                        if constexpr (PUSH) {
                            if (po) {
#pragma unroll
                                for (int j = 0; j < RV; j++) push_out(j, outs[j]);
                            }
                        }
                    };
                    T wb = T(0);
                    const T* gxrow = tab + (o & 1) * nhp + k0;
                    if (!SUMS_ONLY) wb = ((o & 4) ? wgz[1] : wgz[0]) * ((o & 2) ? wgy[1] : wgy[0]);
                    // packed path: the relaxation term is always added; with collisions off W = 0 multiplies the own row
                    // (finite values) instead of a factor table nobody wrote
                    const float* gxs = reinterpret_cast<const float*>(p.collide ? gxrow : a_own);
                    if (SUMS_ONLY) {
#pragma unroll
                        for (int j = 0; j < RV; j++) {
                            T own[VEC];
                            lds16(a_own + j * VEC, own);
#pragma unroll
                            for (int i = 0; i < VEC; i++) {
                                row_sums((double)own[i], j * VEC + i);
                            }
                        }
                    } else if (flags == 0) {
                        // every upwind source is one piece
                        const T* a_x = addr_of(ix.y & 0xffu);
                        const T* a_y = addr_of(ix.z & 0xffu);
                        const T* a_z = addr_of(ix.w & 0xffu);
#pragma unroll
                        for (int j = 0; j < RV; j++) {
                            T own[VEC], X[VEC], Y[VEC], Z[VEC], out[VEC];
                            lds16(a_own + j * VEC, own);
                            lds16(a_x + j * VEC, X);
                            lds16(a_y + j * VEC, Y);
                            lds16(a_z + j * VEC, Z);
                            if constexpr (PACKED) {
                                // two values per instruction (fma.rn.f32x2)
                                const float2 wb2 = make_float2(wb, wb);
                                float gx[4];
                                lds16(gxs + j * 4, gx);
#pragma unroll
                                for (int h = 0; h < 2; h++) {
                                    float2 m = __fmul2_rn(cx2[2 * j + h], make_float2(X[2 * h], X[2 * h + 1]));
                                    m = __ffma2_rn(bx2[2 * j + h], make_float2(own[2 * h], own[2 * h + 1]), m);
                                    m = __ffma2_rn(cy2, make_float2(Y[2 * h], Y[2 * h + 1]), m);
                                    m = __ffma2_rn(cz2, make_float2(Z[2 * h], Z[2 * h + 1]), m);
                                    m = __ffma2_rn(wb2, make_float2(gx[2 * h], gx[2 * h + 1]), m);
                                    out[2 * h] = m.x; out[2 * h + 1] = m.y;
                                }
                            } else {
#pragma unroll
                                for (int i = 0; i < VEC; i++) {
                                    const T cx = sxc * xk(j * VEC + i);
                                    out[i] = base * own[i] + cx * (X[i] - own[i]) + cy * Y[i] + cz * Z[i];
                                }
                                if (p.collide) {
                                    T gx[VEC];
                                    lds16(gxrow + j * VEC, gx);
#pragma unroll
                                    for (int i = 0; i < VEC; i++) out[i] += wb * gx[i];
                                }
                            }
                            stg16_cs(gdst + j * VEC, out);
                            keep_out(j, out);
#pragma unroll
                            for (int i = 0; i < VEC; i++) {
                                row_sums((double)out[i], j * VEC + i);
                            }
                        }
                        push_row();
                    } else if (FLUID && (flags & CIDX_FOUR) == 0u) {
                        // one source per axis, some of them fluid leaves (the common cell under a kinetic/fluid mask): a
                        // piece is read, a fluid source is row factor x x factor from its mini-piece (flatten.hpp)
                        const uint32_t fmask = ix.x >> 16;
                        const uint32_t bsrc[3] = {ix.y & 0xffu, ix.z & 0xffu, ix.w & 0xffu};
                        const bool isfl[3] = {(fmask & 0x001u) != 0u, (fmask & 0x010u) != 0u, (fmask & 0x100u) != 0u};
                        const T* ap[3];
                        const double* fq[3];
                        double bb[3];
#pragma unroll
                        for (int a = 0; a < 3; a++) {
                            int ps = head + (int)bsrc[a];
                            if (ps >= NP) ps -= NP;
                            fq[a] = reinterpret_cast<const double*>(smem_raw + (uint32_t)ps * PB);
                            ap[a] = reinterpret_cast<const T*>(smem_raw + (uint32_t)ps * PB + rowoff);
                            bb[a] = isfl[a] ? fq[a][FLUID_PIECE_B + rr] : 0.0;
                        }
#pragma unroll
                        for (int j = 0; j < RV; j++) {
                            T own[VEC], S[3][VEC], out[VEC];
                            lds16(a_own + j * VEC, own);
#pragma unroll
                            for (int a = 0; a < 3; a++) {
                                if (isfl[a]) {
#pragma unroll
                                    for (int i = 0; i < VEC; i++) S[a][i] = (T)(bb[a] * fq[a][FLUID_PIECE_GX + k0 + j * VEC + i]);
                                } else lds16(ap[a] + j * VEC, S[a]);
                            }
#pragma unroll
                            for (int i = 0; i < VEC; i++) {
                                const T cx = sxc * xk(j * VEC + i);
                                out[i] = base * own[i] + cx * (S[0][i] - own[i]) + cy * S[1][i] + cz * S[2][i];
                            }
                            if (p.collide) {
                                T gx[VEC];
                                lds16(gxrow + j * VEC, gx);
#pragma unroll
                                for (int i = 0; i < VEC; i++) out[i] += wb * gx[i];
                            }
                            stg16_cs(gdst + j * VEC, out);
                            keep_out(j, out);
#pragma unroll
                            for (int i = 0; i < VEC; i++) {
                                row_sums((double)out[i], j * VEC + i);
                            }
                        }
                        push_row();
                    } else {
                        // 2:1 faces towards finer leaves (four sources, each weighted 1/4: reading G3) and / or fluid leaves
                        const uint32_t words[3] = {ix.y, ix.z, ix.w};
                        const uint32_t fmask = FLUID ? (ix.x >> 16) : 0u;   // bit 4a + m: source m on axis a is a fluid ghost
                        // unrolled where every source is a piece (same-box A/B: config 4 -4 %, config 3' -3 %); kept rolled
                        // where fluid sources are formed from global factor tables (unrolled: config 5' +40 %)
#pragma unroll(FLUID ? 1 : RV)
                        for (int j = 0; j < RV; j++) {
                            T own[VEC], S[3][VEC], out[VEC];
                            lds16(a_own + j * VEC, own);
#pragma unroll
                            for (int a = 0; a < 3; a++) {
                                const int nsrc = (flags >> a) & 1u ? 4 : 1;
#pragma unroll
                                for (int i = 0; i < VEC; i++) S[a][i] = T(0);
                                for (int m = 0; m < nsrc; m++) {
                                    const uint32_t b = (words[a] >> (8 * m)) & 0xffu;
                                    T v[VEC];
                                    if (FLUID && ((fmask >> (4 * a + m)) & 1u)) {
                                        // the fluid leaf's Maxwellian at (row, rank) = row factor x x factor (flatten.hpp)
                                        int ps = head + (int)b;
                                        if (ps >= NP) ps -= NP;
                                        const double* fp = reinterpret_cast<const double*>(smem_raw + (uint32_t)ps * PB);
                                        const double bb = fp[FLUID_PIECE_B + rr];
#pragma unroll
                                        for (int i = 0; i < VEC; i++) v[i] = (T)(bb * fp[FLUID_PIECE_GX + k0 + j * VEC + i]);
                                    } else lds16(addr_of(b) + j * VEC, v);
#pragma unroll
                                    for (int i = 0; i < VEC; i++) S[a][i] += v[i];
                                }
                                if (nsrc == 4) {
#pragma unroll
                                    for (int i = 0; i < VEC; i++) S[a][i] *= T(0.25);
                                }
                            }
                            if constexpr (PACKED && !FLUID) {
                                // (j is a compile-time index here: the loop is unrolled)
                                const float2 wb2 = make_float2(wb, wb);
                                float gx[4];
                                lds16(gxs + j * 4, gx);
#pragma unroll
                                for (int h = 0; h < 2; h++) {
                                    float2 m = __fmul2_rn(cx2[2 * j + h], make_float2(S[0][2 * h], S[0][2 * h + 1]));
                                    m = __ffma2_rn(bx2[2 * j + h], make_float2(own[2 * h], own[2 * h + 1]), m);
                                    m = __ffma2_rn(cy2, make_float2(S[1][2 * h], S[1][2 * h + 1]), m);
                                    m = __ffma2_rn(cz2, make_float2(S[2][2 * h], S[2][2 * h + 1]), m);
                                    m = __ffma2_rn(wb2, make_float2(gx[2 * h], gx[2 * h + 1]), m);
                                    out[2 * h] = m.x; out[2 * h + 1] = m.y;
                                }
                            } else {
#pragma unroll
                                for (int i = 0; i < VEC; i++) {
                                    const T cx = sxc * (FLUID ? xk_dyn(j * VEC + i) : xk(j * VEC + i));   // (rolled loop in the fluid instantiation)
                                    out[i] = base * own[i] + cx * (S[0][i] - own[i]) + cy * S[1][i] + cz * S[2][i];
                                }
                                if (p.collide) {
                                    T gx[VEC];
                                    lds16(gxrow + j * VEC, gx);
#pragma unroll
                                    for (int i = 0; i < VEC; i++) out[i] += wb * gx[i];
                                }
                            }
                            stg16_cs(gdst + j * VEC, out);
                            if constexpr (FLUID) push_out(j, out); else keep_out(j, out);
#pragma unroll
                            for (int i = 0; i < VEC; i++) {
                                if constexpr (FLUID) row_sums_dyn((double)out[i], j * VEC + i); else row_sums((double)out[i], j * VEC + i);
                            }
                        }
                        if constexpr (!FLUID) push_row();
                    }
                }
                __syncwarp();
                if (lane == 0) smbar_arrive(sb + o_empty + 8u * slot);
                k++;
                // signs of the octant as doubles; fold the row sums into the 16 combinations
                const double sx = (o & 1) ? 1.0 : -1.0, sy = (o & 2) ? 1.0 : -1.0, sz = (o & 4) ? 1.0 : -1.0;
                const double sxy = sx * sy, sxz = sx * sz, syz = sy * sz;
                E0 += s0_; Ey = fma(sy, s0_, Ey); Ez = fma(sz, s0_, Ez); Eyz = fma(syz, s0_, Eyz);
                F0 += s1_; Fx = fma(sx, s1_, Fx); Fy = fma(sy, s1_, Fy); Fxy = fma(sxy, s1_, Fxy); Fz = fma(sz, s1_, Fz); Fxz = fma(sxz, s1_, Fxz);
                G0 += s2_; Gx = fma(sx, s2_, Gx); Gy = fma(sy, s2_, Gy); Gz = fma(sz, s2_, Gz);
                K0 += s3_; Kx = fma(sx, s3_, Kx);
            }
            // expand to the 35 sums of this row block (layout: stream_common.cuh) ...
            double v[36];
            const double r2 = fma(ay, ay, az * az);
            v[0] = E0; v[1] = Fx; v[2] = ay * Ey; v[3] = az * Ez; v[4] = fma(r2, E0, G0);
#pragma unroll
            for (int s = 0; s < 2; s++) {
                const double sp = s ? 1.0 : -1.0;     // sum over the octants with sign s on the axis: (all + sp * signed) / 2
                const double f0 = 0.5 * fma(sp, Fx, F0);
                v[g_index(0, s, 0)] = f0;
                v[g_index(0, s, 1)] = 0.5 * fma(sp, G0, Gx);
                v[g_index(0, s, 2)] = 0.5 * ay * fma(sp, Fxy, Fy);
                v[g_index(0, s, 3)] = 0.5 * az * fma(sp, Fxz, Fz);
                v[g_index(0, s, 4)] = fma(r2, f0, 0.5 * fma(sp, Kx, K0));
                const double ey = 0.5 * ay * fma(sp, Ey, E0);
                v[g_index(1, s, 0)] = ey;
                v[g_index(1, s, 1)] = 0.5 * ay * fma(sp, Fxy, Fx);
                v[g_index(1, s, 2)] = 0.5 * ay * ay * fma(sp, E0, Ey);
                v[g_index(1, s, 3)] = 0.5 * ay * az * fma(sp, Eyz, Ez);
                v[g_index(1, s, 4)] = fma(r2, ey, 0.5 * ay * fma(sp, Gy, G0));
                const double ez = 0.5 * az * fma(sp, Ez, E0);
                v[g_index(2, s, 0)] = ez;
                v[g_index(2, s, 1)] = 0.5 * az * fma(sp, Fxz, Fx);
                v[g_index(2, s, 2)] = 0.5 * az * ay * fma(sp, Eyz, Ey);
                v[g_index(2, s, 3)] = 0.5 * az * az * fma(sp, E0, Ez);
                v[g_index(2, s, 4)] = fma(r2, ez, 0.5 * az * fma(sp, Gz, G0));
            }
            v[35] = 0.0;
            // ... reduce over the 16 lanes of the group and add into the group's partial sums (one owner lane per entry)
            group16_reduce(v, lane);
            {
                const int b0 = lane & 1, b1 = (lane >> 1) & 1, b2 = (lane >> 2) & 1, b3 = (lane >> 3) & 1;
#pragma unroll
                for (int t = 0; t < 3; t++) {
                    const int l4 = t + 3 * b0;
                    if (l4 < (b1 ? 4 : 5)) {
                        const int j = l4 + 5 * b1 + 9 * b2 + 18 * b3;
                        if (q == 0) red[j] = v[t];
                        else red[j] += v[t];
                    }
                }
            }
        }
        // the three warps that share two cells meet; then the cells' sums go out
        asm volatile("bar.sync %0, %1;" ::"r"(1 + triple), "r"(96) : "memory");
        {
            const int u = ct - 96 * triple;
            if (u < 2 * SUMS_STRIDE) {
                const int cc = 2 * triple + u / SUMS_STRIDE, j = u % SUMS_STRIDE;
                if (cc < nc) {
                    const double* rp = reinterpret_cast<const double*>(smem_raw + o_red) + (size_t)(n & 1) * RED_DOUBLES + (size_t)cc * 3 * SUMS_STRIDE + j;
                    const double sum = rp[0] + rp[SUMS_STRIDE] + rp[2 * SUMS_STRIDE];
                    p.sums_out[(int64_t)(s0 + cc) * SUMS_STRIDE + j] = sum;
                    if constexpr (PUSH) {
                        // the peers that hold this cell as a ghost cell get its sums too (their k_prep reads them as an upwind source's)
                        const uint32_t cnts = *reinterpret_cast<const uint32_t*>(smem_raw + hdr + 28);
                        const int pc = (int)((cnts >> (4 * cc)) & 15u);
                        if (pc) {
                            int first = *reinterpret_cast<const int*>(smem_raw + hdr + 24);
                            for (int i = 0; i < cc; i++) first += (int)((cnts >> (4 * i)) & 15u);
                            for (int e = 0; e < pc; e++) {
                                const unsigned long long d = __ldg(reinterpret_cast<const unsigned long long*>(p.tile_push[first + e].sums_dst) + p.push_parity);
                                if (d) reinterpret_cast<double*>(d)[j] = sum;
                            }
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) smbar_arrive(sb + o_tempty + 8u * ts);
    }
}

constexpr size_t TILES_SMEM_MAX = 227 * 1024;

template <typename T, bool FLUID, bool SUMS_ONLY, bool PUSH = false>
cudaError_t launch_tiles_t(const StepLaunch& plan, const StepParams& p, cudaStream_t st, bool timed) {
    auto kfn = k_tiles<T, FLUID, SUMS_ONLY, PUSH>;
    cudaError_t e = cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    const int grid = p.n_tiles < plan.grid ? p.n_tiles : plan.grid;
    StepParams q = p;
    const TilesSmem m = tiles_map(sizeof(T), plan.stages, tabn_of(p.nh));
    const uint32_t v[11] = {m.ring, m.desc, m.thdr, m.red, m.full, m.empty, m.tinfo, m.ttab, m.tempty, m.total, m.thdr_bytes};
    for (int i = 0; i < 11; i++) q.smap[i] = v[i];
    q.smap[11] = plan.test_stall ? 1u : 0u;
    q.ring_stages = plan.stages;
    if (timed && plan.ev0) cudaEventRecord(plan.ev0, st);
    kfn<<<grid, (N_PROD + N_CONS) * 32, plan.smem_bytes, st>>>(q);
    if (timed && plan.ev1) cudaEventRecord(plan.ev1, st);
    return cudaGetLastError();
}

}  // namespace

// The fluid pieces of every fluid ghost: [ghost * 8 + octant][row block][FLUID_PIECE_STRIDE] doubles -- the 12 x factors of
// the sign group's x sign, then the NRP row factors amp g_z g_y of the block's rows (flatten.hpp; the product in the
// order in which the host forms the ghost's velocity sums, api.cu: ghost_state_sums).  12 KB per fluid ghost for 24^3.
void tiles_fluid_pieces(const FlatMesh& m, int storage, std::vector<double>& out) {
    const VelLayout& v = m.vel;
    const int NRP = nrp_of(storage == UFS_STORE_F32 ? 4 : 8);
    const int nq = v.nh[1] * v.nh[2] / NRP;
    out.assign(m.fluid.size() * 8 * (size_t)nq * FLUID_PIECE_STRIDE, 0.0);
#pragma omp parallel for schedule(static)
    for (int64_t gi = 0; gi < (int64_t)m.fluid.size(); gi++) {
        const FluidGhost& g = m.fluid[gi];
        for (int o = 0; o < 8; o++)
            for (int q = 0; q < nq; q++) {
                double* d = out.data() + (((size_t)gi * 8 + o) * nq + q) * FLUID_PIECE_STRIDE;
                for (int e = 0; e < THX; e++) d[FLUID_PIECE_GX + e] = g.g[0][(o & 1) ? v.nh[0] + e : v.nh[0] - 1 - e];
                for (int rr = 0; rr < NRP; rr++) {
                    const int row = q * NRP + rr, ry = row % v.nh[1], rz = row / v.nh[1];
                    const int kz = ((o >> 2) & 1) ? v.nh[2] + rz : v.nh[2] - 1 - rz;
                    const int ky = ((o >> 1) & 1) ? v.nh[1] + ry : v.nh[1] - 1 - ry;
                    d[FLUID_PIECE_B + rr] = g.amp * g.g[2][kz] * g.g[1][ky];
                }
            }
    }
}

// Launch geometry of the tile kernel, or false if the velocity grid does not fit it (12 x-ranks per row, whole row
// blocks of 48 rows, octant layout); *pmax = pieces a tile may list per octant (two stages must fit the ring).
bool tiles_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan, int* pmax) {
    if (!v.fast || v.nh[0] != THX) return false;
    const int nr = v.nh[1] * v.nh[2];
    const int NRP = nrp_of(storage == UFS_STORE_F32 ? 4 : 8);
    if (nr % NRP != 0 || NRP % v.nh[1] != 0 || (nr / NRP) * 8 < NSTG) return false;
    for (int a = 0; a < 3; a++)
        if (v.nv[a] > 32) return false;
    StepLaunch base{};
    if (!stream_plan(storage, v, sm_count, &base)) return false;   // k_prep / fallbacks share its checks
    const size_t elem = storage == UFS_STORE_F32 ? 4 : 8;
    const int32_t nh[3] = {v.nh[0], v.nh[1], v.nh[2]};
    const int tabn = tabn_of(nh);
    int np = 255;
    while (np >= 26 && tiles_map(elem, np, tabn).total > TILES_SMEM_MAX) np--;
    if (np < 26) return false;           // a single cell may need 13 pieces per octant; two stages must fit
    *plan = base;
    plan->ring = 4;
    plan->stages = np;                   // piece slots of the ring
    plan->threads = (N_PROD + N_CONS) * 32;
    plan->smem_bytes = (int32_t)tiles_map(elem, np, tabn).total;
    plan->grid = sm_count;
    *pmax = np / 2 < 40 ? np / 2 : 40;
    return true;
}

cudaError_t launch_tiles(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    cudaError_t e = launch_prep(storage, p, st);
    if (e != cudaSuccess) return e;
    if (plan.push_on) {
        // fused ghost exchange: first the tiles with cells some peer needs (their rows are also stored into the peers' ghost
        // slabs and travel while the rest is computed), then the plain pass over the other tiles.  Two launches, two ticket
        // counters: each launch draws from one and zeroes the other.
        const int nb = plan.push_tiles < p.n_tiles ? plan.push_tiles : p.n_tiles;
        StepLaunch pl = plan;
        cudaEvent_t ev1 = plan.ev1;
        if (nb > 0) {
            StepParams q = p;
            q.n_tiles = nb;
            if (nb < p.n_tiles) pl.ev1 = nullptr;
            if (storage == UFS_STORE_F32)
                e = p.tiles_have_fluid ? launch_tiles_t<float, true, false, true>(pl, q, st, true) : launch_tiles_t<float, false, false, true>(pl, q, st, true);
            else
                e = p.tiles_have_fluid ? launch_tiles_t<double, true, false, true>(pl, q, st, true) : launch_tiles_t<double, false, false, true>(pl, q, st, true);
            if (e != cudaSuccess || nb == p.n_tiles) return e;
            pl.ev0 = nullptr;
        }
        StepParams q = p;
        q.n_tiles = p.n_tiles - nb;
        q.tile_hdr = p.tile_hdr + nb;
        q.tile_pieces = p.tile_pieces + (size_t)nb * 8 * p.tile_pmax;
        q.tile_cellidx = p.tile_cellidx + (size_t)nb * 8 * TILE_CELLS * CELLIDX_BYTES;
        if (nb > 0) { q.counter = p.counter_reset; q.counter_reset = p.counter; }
        pl.ev1 = ev1;
        if (storage == UFS_STORE_F32)
            return p.tiles_have_fluid ? launch_tiles_t<float, true, false>(pl, q, st, true) : launch_tiles_t<float, false, false>(pl, q, st, true);
        return p.tiles_have_fluid ? launch_tiles_t<double, true, false>(pl, q, st, true) : launch_tiles_t<double, false, false>(pl, q, st, true);
    }
    if (storage == UFS_STORE_F32)
        return p.tiles_have_fluid ? launch_tiles_t<float, true, false>(plan, p, st, true) : launch_tiles_t<float, false, false>(plan, p, st, true);
    return p.tiles_have_fluid ? launch_tiles_t<double, true, false>(plan, p, st, true) : launch_tiles_t<double, false, false>(plan, p, st, true);
}

int tiles_launches_per_step(const StepLaunch& plan, const StepParams& p) {
    if (!plan.push_on) return 1;
    const int nb = plan.push_tiles < p.n_tiles ? plan.push_tiles : p.n_tiles;
    return (nb > 0 ? 1 : 0) + (nb < p.n_tiles ? 1 : 0);
}

// sums[n_kin][SUMS_STRIDE] of an f the caller has just written: the same kernel, own chunks only, no store
cudaError_t launch_tile_sums(int storage, const StepLaunch& plan, const StepParams& p, const void* f, double* sums, cudaStream_t st) {
    if (p.n_kin == 0) return cudaSuccess;
    StepParams q = p;
    q.f_in = f;
    q.sums_out = sums;
    if (storage == UFS_STORE_F32) return launch_tiles_t<float, false, true>(plan, q, st, false);
    return launch_tiles_t<double, false, true>(plan, q, st, false);
}

}  // namespace ufs
