// lbm.cu -- the lattice-Boltzmann variant of the kinetic step (include/ufs_lbm.h): the DVM solver's
// finite-volume transport on the octree with the 19 or 27 velocities of a 3x3x3 velocity grid, rho = sum f,
// rho u = sum c f, second-order polynomial equilibrium, BGK relaxation with a constant tau.
//
// Mapping.  The paper groups "each velocity grid in a spatial cell into a warp" (27 of 32 lanes busy, the
// moments by warp reductions) -- made for Fermi / Kepler.  Here that mapping measured 0.09 of the HBM peak, issue-bound
// (~400 warp instructions per cell, four fp64 shuffle reductions, 13 idle lanes for D3Q19).  On sm_100a the unit is one
// THREAD per cell and f is stored velocity-major, f[i][cell]: the 32 threads of a warp take 32 consecutive cells of the
// N-order curve, so every population's loads and stores are one contiguous run, the upwind neighbours of consecutive
// cells are mostly consecutive cells too, the moments are thread-local sums (no shuffles), and the lattice is a
// compile-time constant: the loop over the 19 / 27 populations unrolls completely, f* stays in registers.
// The upwind value of population i on axis a comes from the cell on the side c_i,a points away from: the same per-cell
// gather records as the DVM step (flatten.cpp; first-order form of the stencil records of PAPER.md:113-115), here
// compacted to 32 bytes per cell (a cell's f is only 76-216 bytes).  Everything in fp64 registers, one rounding at
// the store.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/ufs_lbm.h"
#include "device_util.cuh"
#include "flatten.hpp"

using namespace ufs;

namespace {

constexpr int32_t LBM_QUAD = 4;   // source kind of a compact record: four finer sources, index into the quad list

struct LbmRec {                   // 32 bytes per cell
    int32_t src[6];               // per direction 2*axis + side: SRC_SLAB / SRC_MIRROR / SRC_TABLE code, or LBM_QUAD
    int32_t level;
    int32_t pad;
};
static_assert(sizeof(LbmRec) == 32, "LbmRec must be 32 bytes");

struct LbmLattice {
    int32_t q;
    int8_t c[27][3];              // lattice velocities in column order
    int8_t mir[3][27];            // column of the velocity mirrored on axis a
    double w[27];
};

struct LbmParams {
    const void* f_in;
    void* f_out;
    const LbmRec* recs;
    const int32_t* quads;         // [n_quads][4] source codes
    const void* tables;           // [n_tables][Q] storage type: inflow equilibria
    int64_t n_cells;
    double dt, inv_len, omega;    // omega = dt / tau
    LbmLattice lat;
};

// second-order equilibrium, host and device
__host__ __device__ inline double lbm_feq(double w, double rho, double cu, double uu) {
    return w * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
}

// ---- the lattice as compile-time functions of (Q, column) ----------------------------------------------------------
// column i of D3Q27 is node k = i of the 3x3x3 grid ((kz*3 + ky)*3 + kx, c = k - 1); D3Q19 keeps the nodes with
// |c|^2 <= 2 in the same order
__host__ __device__ constexpr int lat_n2(int k) {
    return (k % 3 - 1) * (k % 3 - 1) + ((k / 3) % 3 - 1) * ((k / 3) % 3 - 1) + (k / 9 - 1) * (k / 9 - 1);
}
__host__ __device__ constexpr int lat_node(int q, int col) {
    if (q == 27) return col;
    int n = 0;
    for (int k = 0; k < 27; k++) {
        if (lat_n2(k) > 2) continue;
        if (n == col) return k;
        n++;
    }
    return -1;
}
__host__ __device__ constexpr int lat_col(int q, int k) {
    if (q == 27) return k;
    int n = 0;
    for (int kk = 0; kk < k; kk++) n += lat_n2(kk) <= 2 ? 1 : 0;
    return n;
}
__host__ __device__ constexpr int lat_c(int q, int col, int a) {
    const int k = lat_node(q, col);
    return a == 0 ? k % 3 - 1 : a == 1 ? (k / 3) % 3 - 1 : k / 9 - 1;
}
__host__ __device__ constexpr int lat_mirror(int q, int col, int a) {   // column of the velocity mirrored on axis a
    const int k = lat_node(q, col);
    const int kx = k % 3, ky = (k / 3) % 3, kz = k / 9;
    return lat_col(q, a == 0 ? (kz * 3 + ky) * 3 + (2 - kx) : a == 1 ? (kz * 3 + (2 - ky)) * 3 + kx : ((2 - kz) * 3 + ky) * 3 + kx);
}
__host__ __device__ constexpr double lat_w(int q, int col) {
    const int n2 = lat_n2(lat_node(q, col));
    return q == 19 ? (n2 == 0 ? 1.0 / 3.0 : n2 == 1 ? 1.0 / 18.0 : 1.0 / 36.0)
                   : (n2 == 0 ? 8.0 / 27.0 : n2 == 1 ? 2.0 / 27.0 : n2 == 2 ? 1.0 / 54.0 : 1.0 / 216.0);
}

void make_lattice(int q, LbmLattice& L) {   // the same lattice as run-time tables (layout accessor, inflow tables)
    L.q = q;
    for (int i = 0; i < q; i++) {
        for (int a = 0; a < 3; a++) { L.c[i][a] = (int8_t)lat_c(q, i, a); L.mir[a][i] = (int8_t)lat_mirror(q, i, a); }
        L.w[i] = lat_w(q, i);
    }
}

// upwind value of population I (compile time) on axis A from one source / from a record entry
template <typename T, int Q, int I, int A>
__device__ __forceinline__ double lbm_fetch1(const LbmParams& p, const T* __restrict__ fin, int32_t code) {
    const int kind = code >> SRC_SHIFT;
    const int64_t idx = code & SRC_INDEX_MASK;
    if (kind == SRC_SLAB) return (double)__ldg(fin + (int64_t)I * p.n_cells + idx);
    if (kind == SRC_MIRROR) return (double)__ldg(fin + (int64_t)lat_mirror(Q, I, A) * p.n_cells + idx);
    return (double)__ldg(reinterpret_cast<const T*>(p.tables) + idx * Q + I);   // SRC_TABLE
}
template <typename T, int Q, int I, int A>
__device__ __forceinline__ double lbm_fetch(const LbmParams& p, const T* __restrict__ fin, int32_t code) {
    if ((code >> SRC_SHIFT) != LBM_QUAD) return lbm_fetch1<T, Q, I, A>(p, fin, code);
    const int4 qd = __ldg(reinterpret_cast<const int4*>(p.quads) + (code & SRC_INDEX_MASK));
    // four sub-faces of a quarter of the face each (reading G3)
    return 0.25 * (lbm_fetch1<T, Q, I, A>(p, fin, qd.x) + lbm_fetch1<T, Q, I, A>(p, fin, qd.y)
                   + lbm_fetch1<T, Q, I, A>(p, fin, qd.z) + lbm_fetch1<T, Q, I, A>(p, fin, qd.w));
}

// f* of population I and its contribution to the moments
template <typename T, int Q, int I>
__device__ __forceinline__ void lbm_population(const LbmParams& p, const T* __restrict__ fin, int64_t cell, const int32_t (&src)[6],
                                               double dth, double (&fs)[Q], double& rho, double& mx, double& my, double& mz) {
    constexpr int cx = lat_c(Q, I, 0), cy = lat_c(Q, I, 1), cz = lat_c(Q, I, 2);
    constexpr int cabs = (cx < 0 ? -cx : cx) + (cy < 0 ? -cy : cy) + (cz < 0 ? -cz : cz);
    double acc = (double)__ldg(fin + (int64_t)I * p.n_cells + cell) * (1.0 - dth * (double)cabs);   // Eq. 2: what stays
    // c_a > 0: data comes from the low side (direction 2a), c_a < 0 from the high side
    if (cx != 0) acc += dth * lbm_fetch<T, Q, I, 0>(p, fin, src[cx > 0 ? 0 : 1]);
    if (cy != 0) acc += dth * lbm_fetch<T, Q, I, 1>(p, fin, src[cy > 0 ? 2 : 3]);
    if (cz != 0) acc += dth * lbm_fetch<T, Q, I, 2>(p, fin, src[cz > 0 ? 4 : 5]);
    fs[I] = acc;
    rho += acc;
    if (cx != 0) mx += (double)cx * acc;
    if (cy != 0) my += (double)cy * acc;
    if (cz != 0) mz += (double)cz * acc;
}
// the same for a cell whose six upwind sources are all plain cells of the same level or coarser (one slab each): no source
// kind to decode.  The arithmetic and its order are those of lbm_population.
template <typename T, int Q, int I>
__device__ __forceinline__ void lbm_population_simple(const LbmParams& p, const T* __restrict__ fin, int64_t cell, const int32_t (&src)[6],
                                                      double dth, double (&fs)[Q], double& rho, double& mx, double& my, double& mz) {
    constexpr int cx = lat_c(Q, I, 0), cy = lat_c(Q, I, 1), cz = lat_c(Q, I, 2);
    constexpr int cabs = (cx < 0 ? -cx : cx) + (cy < 0 ? -cy : cy) + (cz < 0 ? -cz : cz);
    const T* __restrict__ fi = fin + (int64_t)I * p.n_cells;
    double acc = (double)__ldg(fi + cell) * (1.0 - dth * (double)cabs);
    if (cx != 0) acc += dth * (double)__ldg(fi + src[cx > 0 ? 0 : 1]);
    if (cy != 0) acc += dth * (double)__ldg(fi + src[cy > 0 ? 2 : 3]);
    if (cz != 0) acc += dth * (double)__ldg(fi + src[cz > 0 ? 4 : 5]);
    fs[I] = acc;
    rho += acc;
    if (cx != 0) mx += (double)cx * acc;
    if (cy != 0) my += (double)cy * acc;
    if (cz != 0) mz += (double)cz * acc;
}
template <typename T, int Q, int I>
struct LbmUnroll {
    static __device__ __forceinline__ void transport_simple(const LbmParams& p, const T* __restrict__ fin, int64_t cell, const int32_t (&src)[6],
                                                            double dth, double (&fs)[Q], double& rho, double& mx, double& my, double& mz) {
        lbm_population_simple<T, Q, I>(p, fin, cell, src, dth, fs, rho, mx, my, mz);
        LbmUnroll<T, Q, I + 1>::transport_simple(p, fin, cell, src, dth, fs, rho, mx, my, mz);
    }
    static __device__ __forceinline__ void transport(const LbmParams& p, const T* __restrict__ fin, int64_t cell, const int32_t (&src)[6],
                                                     double dth, double (&fs)[Q], double& rho, double& mx, double& my, double& mz) {
        lbm_population<T, Q, I>(p, fin, cell, src, dth, fs, rho, mx, my, mz);
        LbmUnroll<T, Q, I + 1>::transport(p, fin, cell, src, dth, fs, rho, mx, my, mz);
    }
    static __device__ __forceinline__ void relax(const LbmParams& p, T* __restrict__ fout, int64_t cell, const double (&fs)[Q],
                                                 double rho, double ux, double uy, double uz, double uu) {
        constexpr int cx = lat_c(Q, I, 0), cy = lat_c(Q, I, 1), cz = lat_c(Q, I, 2);
        const double cu = (double)cx * ux + (double)cy * uy + (double)cz * uz;
        fout[(int64_t)I * p.n_cells + cell] = (T)(fs[I] + p.omega * (lbm_feq(lat_w(Q, I), rho, cu, uu) - fs[I]));
        LbmUnroll<T, Q, I + 1>::relax(p, fout, cell, fs, rho, ux, uy, uz, uu);
    }
    static __device__ __forceinline__ void moments(const LbmParams& p, const T* __restrict__ fin, int64_t cell, double& rho, double& mx,
                                                   double& my, double& mz) {
        const double f = (double)__ldg(fin + (int64_t)I * p.n_cells + cell);
        rho += f; mx += (double)lat_c(Q, I, 0) * f; my += (double)lat_c(Q, I, 1) * f; mz += (double)lat_c(Q, I, 2) * f;
        LbmUnroll<T, Q, I + 1>::moments(p, fin, cell, rho, mx, my, mz);
    }
};
template <typename T, int Q>
struct LbmUnroll<T, Q, Q> {
    static __device__ __forceinline__ void transport_simple(const LbmParams&, const T*, int64_t, const int32_t (&)[6], double, double (&)[Q],
                                                            double&, double&, double&, double&) {}
    static __device__ __forceinline__ void transport(const LbmParams&, const T*, int64_t, const int32_t (&)[6], double, double (&)[Q],
                                                     double&, double&, double&, double&) {}
    static __device__ __forceinline__ void relax(const LbmParams&, T*, int64_t, const double (&)[Q], double, double, double, double, double) {}
    static __device__ __forceinline__ void moments(const LbmParams&, const T*, int64_t, double&, double&, double&, double&) {}
};

// resident blocks per SM the register allocation aims at (same-box A/B of 4 / 6 / 8 for D3Q19 and 4 / 5 / 6 for D3Q27: the
// step is latency-bound, more warps win until the spills take over)
#ifndef LBM_MINB19
#define LBM_MINB19 8
#endif
#ifndef LBM_MINB27
#define LBM_MINB27 5
#endif
template <typename T, int Q>
__global__ void __launch_bounds__(128, Q == 19 ? LBM_MINB19 : LBM_MINB27) k_lbm_step(const LbmParams p) {
    const T* __restrict__ fin = reinterpret_cast<const T*>(p.f_in);
    T* __restrict__ fout = reinterpret_cast<T*>(p.f_out);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; cell < p.n_cells; cell += stride) {
        const int4 r0 = __ldg(reinterpret_cast<const int4*>(p.recs + cell)), r1 = __ldg(reinterpret_cast<const int4*>(p.recs + cell) + 1);
        const int32_t src[6] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y};
        const double dth = p.dt * p.inv_len * (double)(1 << r1.z);   // dt / h
        double fs[Q];
        double rho = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
        // SRC_SLAB is kind 0: the six codes are then the slab numbers themselves
        if (((r0.x | r0.y | r0.z | r0.w | r1.x | r1.y) >> SRC_SHIFT) == 0) LbmUnroll<T, Q, 0>::transport_simple(p, fin, cell, src, dth, fs, rho, mx, my, mz);
        else LbmUnroll<T, Q, 0>::transport(p, fin, cell, src, dth, fs, rho, mx, my, mz);
        const double ux = mx / rho, uy = my / rho, uz = mz / rho;
        LbmUnroll<T, Q, 0>::relax(p, fout, cell, fs, rho, ux, uy, uz, ux * ux + uy * uy + uz * uz);
    }
}

template <typename T, int Q>
__global__ void __launch_bounds__(128) k_lbm_moments(const LbmParams p, double* __restrict__ mom) {
    const T* __restrict__ fin = reinterpret_cast<const T*>(p.f_in);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; cell < p.n_cells; cell += stride) {
        double rho = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
        LbmUnroll<T, Q, 0>::moments(p, fin, cell, rho, mx, my, mz);
        mom[cell] = rho; mom[p.n_cells + cell] = mx; mom[2 * p.n_cells + cell] = my; mom[3 * p.n_cells + cell] = mz;
    }
}

template <typename T>
cudaError_t lbm_launch_step(int q, int grid, const LbmParams& p, cudaStream_t st) {
    if (q == 19) k_lbm_step<T, 19><<<grid, 128, 0, st>>>(p);
    else k_lbm_step<T, 27><<<grid, 128, 0, st>>>(p);
    return cudaGetLastError();
}
template <typename T>
cudaError_t lbm_launch_moments(int q, int grid, const LbmParams& p, double* mom, cudaStream_t st) {
    if (q == 19) k_lbm_moments<T, 19><<<grid, 128, 0, st>>>(p, mom);
    else k_lbm_moments<T, 27><<<grid, 128, 0, st>>>(p, mom);
    return cudaGetLastError();
}

}  // namespace

struct ufs_lbm_s {
    FlatMesh mesh;
    int storage = UFS_STORE_F64, q = 19;
    double tau = 1.0, domain_len = 1.0;
    LbmLattice lat{};
    std::vector<LbmRec> recs;
    std::vector<int32_t> quads;
    std::vector<double> tables;     // [n_tables][Q]
    bool device = false;
    void* f[2] = {nullptr, nullptr};
    int cur = 0;
    cudaStream_t stream = nullptr;
    LbmRec* d_recs = nullptr;
    int32_t* d_quads = nullptr;
    void* d_tables = nullptr;
    int grid = 0;
    int64_t launches = 0;
    int sticky = UFS_DVM_OK;
    std::string err;
};

namespace {

int lfail(ufs_lbm_t h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}
#define LCU(call, what)                                                              \
    do {                                                                             \
        cudaError_t e__ = (call);                                                    \
        if (e__ != cudaSuccess) {                                                    \
            h->sticky = UFS_DVM_ECUDA;                                               \
            return lfail(h, UFS_DVM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e__)); \
        }                                                                            \
    } while (0)

int lbm_create_common(const ufs_lbm_desc* desc, ufs_lbm_t* out) {
    if (!out) return UFS_DVM_EINVAL;
    *out = nullptr;
    if (!desc) return UFS_DVM_EINVAL;
    ufs_lbm_t h = new (std::nothrow) ufs_lbm_s();
    if (!h) return UFS_DVM_ENOMEM;
    *out = h;
    if (desc->lattice != 19 && desc->lattice != 27) return lfail(h, UFS_DVM_EINVAL, "lattice must be 19 (D3Q19) or 27 (D3Q27)");
    if (!(desc->tau > 0)) return lfail(h, UFS_DVM_EINVAL, "tau must be positive (+inf = no collisions)");
    if (desc->n_leaves <= 0 || !desc->kind) return lfail(h, UFS_DVM_EINVAL, "empty or NULL leaf list");
    for (int64_t j = 0; j < desc->n_leaves; j++)
        if (desc->kind[j] == UFS_CELL_FLUID) return lfail(h, UFS_DVM_EINVAL, "the LBM variant has no kinetic/fluid mask: no FLUID leaves");
    h->storage = desc->storage; h->q = desc->lattice; h->tau = desc->tau; h->domain_len = desc->domain_len;
    make_lattice(h->q, h->lat);
    // the DVM flattener on the 3x3x3 velocity grid with nodes -1, 0, 1
    ufs_dvm_desc dd{};
    dd.n_leaves = desc->n_leaves; dd.level = desc->level; dd.ijk = desc->ijk; dd.kind = desc->kind;
    dd.domain_len = desc->domain_len;
    for (int s = 0; s < 6; s++) {
        dd.bc[s] = desc->bc[s];
        dd.inflow[s][0] = 1.0; dd.inflow[s][4] = 1.0;   // (the flattener's own Maxwellian tables are not used here)
        if (desc->bc[s] == UFS_BC_INFLOW && !(desc->inflow[s][0] > 0)) return lfail(h, UFS_DVM_EINVAL, "inflow state needs rho > 0");
    }
    for (int a = 0; a < 3; a++) { dd.nv[a] = 3; dd.vmin[a] = -1.5; dd.vmax[a] = 1.5; }
    dd.kn = INFINITY; dd.visc_exp = 0.5; dd.nu_prefactor = 1.0; dd.storage = desc->storage;
    try {
        std::string err;
        const int rc = flatten(dd, h->mesh, err);
        if (rc) return lfail(h, rc, err);
        const FlatMesh& m = h->mesh;
        // compact records
        h->recs.assign(m.n_kin, LbmRec{});
        for (int64_t s = 0; s < m.n_kin; s++) {
            const CellRec& r = m.recs[s];
            LbmRec& o = h->recs[s];
            o.level = r.level;
            for (int d = 0; d < 6; d++) {
                if (r.src[d][1] < 0) { o.src[d] = r.src[d][0]; continue; }
                if (h->quads.size() / 4 >= (size_t)SRC_INDEX_MASK) return lfail(h, UFS_DVM_EINVAL, "too many 2:1 faces");
                o.src[d] = (LBM_QUAD << SRC_SHIFT) | (int32_t)(h->quads.size() / 4);
                for (int k = 0; k < 4; k++) h->quads.push_back(r.src[d][k]);
            }
        }
        // inflow equilibria, one table per INFLOW side in the flattener's table order
        h->tables.assign((size_t)m.n_tables * h->q, 0.0);
        for (int s = 0; s < 6; s++) {
            const int t = m.table_of_side[s];
            if (t < 0) continue;
            const double rho = desc->inflow[s][0], ux = desc->inflow[s][1], uy = desc->inflow[s][2], uz = desc->inflow[s][3];
            for (int i = 0; i < h->q; i++) {
                const double cu = h->lat.c[i][0] * ux + h->lat.c[i][1] * uy + h->lat.c[i][2] * uz;
                h->tables[(size_t)t * h->q + i] = lbm_feq(h->lat.w[i], rho, cu, ux * ux + uy * uy + uz * uz);
            }
        }
    } catch (const std::bad_alloc&) {
        return lfail(h, UFS_DVM_ENOMEM, "out of host memory while flattening");
    } catch (...) {
        return lfail(h, UFS_DVM_EINVAL, "unexpected failure while flattening");
    }
    return UFS_DVM_OK;
}

LbmParams lbm_params(ufs_lbm_t h, double dt) {
    LbmParams p{};
    p.f_in = h->f[h->cur]; p.f_out = h->f[h->cur ^ 1];
    p.recs = h->d_recs; p.quads = h->d_quads; p.tables = h->d_tables;
    p.n_cells = h->mesh.n_kin;
    p.dt = dt; p.inv_len = 1.0 / h->domain_len;
    p.omega = std::isinf(h->tau) ? 0.0 : dt / h->tau;
    p.lat = h->lat;
    return p;
}

}  // namespace

extern "C" {

int ufs_lbm_create_host(const ufs_lbm_desc* desc, ufs_lbm_t* out) { return lbm_create_common(desc, out); }

int ufs_lbm_create(const ufs_lbm_desc* desc, void* f_dev[2], void* cuda_stream, ufs_lbm_t* out) {
    int rc = lbm_create_common(desc, out);
    if (rc) return rc;
    ufs_lbm_t h = *out;
    const int64_t n = h->mesh.n_kin;
    if (!f_dev || ((!f_dev[0] || !f_dev[1]) && n > 0)) return lfail(h, UFS_DVM_EINVAL, "f_dev[0] and f_dev[1] must be device buffers");
    if (n > 0 && (f_dev[0] == f_dev[1] || ((uintptr_t)f_dev[0] & 15) || ((uintptr_t)f_dev[1] & 15)))
        return lfail(h, UFS_DVM_EINVAL, "the two f buffers must be distinct and 16-byte aligned");
    h->f[0] = f_dev[0]; h->f[1] = f_dev[1];
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    h->device = true;
    auto up = [&](void** dst, const void* src, size_t bytes, const char* what) -> int {
        *dst = nullptr;
        if (!bytes) return UFS_DVM_OK;
        LCU(cudaMalloc(dst, bytes), what);
        LCU(cudaMemcpyAsync(*dst, src, bytes, cudaMemcpyHostToDevice, h->stream), what);
        return UFS_DVM_OK;
    };
    if ((rc = up(reinterpret_cast<void**>(&h->d_recs), h->recs.data(), h->recs.size() * sizeof(LbmRec), "upload cell records"))) return rc;
    if ((rc = up(reinterpret_cast<void**>(&h->d_quads), h->quads.data(), h->quads.size() * 4, "upload 2:1 source lists"))) return rc;
    std::vector<float> t32;
    const void* tab = h->tables.data();
    size_t tb = h->tables.size() * 8;
    if (h->storage == UFS_STORE_F32) { t32.assign(h->tables.begin(), h->tables.end()); tab = t32.data(); tb = t32.size() * 4; }
    if ((rc = up(&h->d_tables, tab, tb, "upload inflow tables"))) return rc;
    const int64_t want = (n + 127) / 128;
    // one cell per thread (the kernels' grid-stride loop only serves meshes beyond 2^31 threads): with 32 blocks per SM and a
    // second trip for 40 % of the threads D3Q19 took 0.130 instead of 0.124 ms, D3Q27 0.268 instead of 0.250 (same box)
    h->grid = (int)std::max<int64_t>(1, std::min<int64_t>(want, (int64_t)1 << 24));
    LCU(cudaStreamSynchronize(h->stream), "upload");
    return UFS_DVM_OK;
}

int ufs_lbm_step(ufs_lbm_t h, double dt, int nsteps) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return lfail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (!(dt > 0) || nsteps < 0) return lfail(h, UFS_DVM_EINVAL, "dt must be positive and nsteps >= 0");
    if (h->mesh.n_kin == 0) return UFS_DVM_OK;
    for (int s = 0; s < nsteps; s++) {
        const LbmParams p = lbm_params(h, dt);
        LCU(h->storage == UFS_STORE_F32 ? lbm_launch_step<float>(h->q, h->grid, p, h->stream) : lbm_launch_step<double>(h->q, h->grid, p, h->stream),
            "step kernel launch");
        h->cur ^= 1;
        h->launches++;
    }
    return UFS_DVM_OK;
}

int ufs_lbm_moments(ufs_lbm_t h, double* mom_dev) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return lfail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (h->mesh.n_kin == 0) return UFS_DVM_OK;
    if (!mom_dev) return lfail(h, UFS_DVM_EINVAL, "mom_dev is NULL");
    const LbmParams p = lbm_params(h, 1.0);
    LCU(h->storage == UFS_STORE_F32 ? lbm_launch_moments<float>(h->q, h->grid, p, mom_dev, h->stream)
                                    : lbm_launch_moments<double>(h->q, h->grid, p, mom_dev, h->stream), "moments kernel launch");
    h->launches++;
    return UFS_DVM_OK;
}

int ufs_lbm_sync(ufs_lbm_t h) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return lfail(h, UFS_DVM_EINVAL, "host-only handle");
    LCU(cudaStreamSynchronize(h->stream), "stream synchronize");
    return h->sticky;
}

int ufs_lbm_destroy(ufs_lbm_t h) {
    if (!h) return UFS_DVM_OK;
    int rc = UFS_DVM_OK;
    if (h->device) {
        if (cudaStreamSynchronize(h->stream) != cudaSuccess) rc = UFS_DVM_ECUDA;
        cudaFree(h->d_recs); cudaFree(h->d_quads); cudaFree(h->d_tables);
    }
    delete h;
    return rc;
}

int ufs_lbm_current(ufs_lbm_t h) { return h ? h->cur : UFS_DVM_EINVAL; }

int ufs_lbm_layout(ufs_lbm_t h, int64_t* n_cells, int64_t* cell_of_row, int32_t* q, int8_t* c, double* w) {
    if (!h) return UFS_DVM_EINVAL;
    if (n_cells) *n_cells = h->mesh.n_kin;
    if (cell_of_row) std::memcpy(cell_of_row, h->mesh.cell_of_slab.data(), (size_t)h->mesh.n_kin * 8);
    if (q) *q = h->q;
    if (c) for (int i = 0; i < h->q; i++) for (int a = 0; a < 3; a++) c[3 * i + a] = h->lat.c[i][a];
    if (w) for (int i = 0; i < h->q; i++) w[i] = h->lat.w[i];
    return UFS_DVM_OK;
}

int64_t ufs_lbm_launch_count(ufs_lbm_t h) { return h ? h->launches : 0; }

const char* ufs_lbm_last_error(ufs_lbm_t h) { return h ? h->err.c_str() : "null handle"; }

}  // extern "C"
