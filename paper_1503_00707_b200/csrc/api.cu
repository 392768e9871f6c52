// api.cu -- the C ABI of libufs_dvm.so (include/ufs_dvm.h): handle life cycle, uploads of what the
// flattener built, and the enqueue calls.  No torch types, no exceptions across the boundary.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/ufs_dvm.h"
#include "flatten.hpp"
#include "kernels.cuh"

using namespace ufs;

struct ufs_dvm_s {
    FlatMesh mesh;
    int storage = UFS_STORE_F64;
    double kn = 0, visc_exp = 0.5, nu_pref = 1, domain_len = 1;
    bool device = false;
    void* f[2] = {nullptr, nullptr};
    int cur = 0;
    cudaStream_t stream = nullptr;
    CellRec* d_cells = nullptr;
    void* d_tables = nullptr;
    FluidGhost* d_fluid = nullptr;
    VelDev* d_vel = nullptr;
    uchar4* d_slot_k = nullptr;
    int32_t* d_mirror = nullptr;
    int32_t* d_flags = nullptr;
    int32_t* d_counter = nullptr;  // [2] cell counters of the ring kernel, one per launch parity
    // streaming step: velocity sums of f[0] / f[1], of the ghost states, and the per-step factor tables
    double* d_sums[2] = {nullptr, nullptr};
    bool sums_are_callers = false;   // ufs_dvm_sums_use: the two arrays belong to the caller (not freed at destroy)
    double* d_ghost_sums = nullptr;
    void* d_tabs = nullptr;
    // tile kernel: the flattener's tile records
    TileHdr* d_tile_hdr = nullptr;
    uint32_t* d_tile_pieces = nullptr;
    uint8_t* d_tile_cellidx = nullptr;
    double* d_fluid_pieces = nullptr;
    PushEntry* d_tile_push = nullptr;   // fused ghost exchange (ufs_dvm_halo_push_setup)
    TileHdr* d_ghost_tiles = nullptr;   // partitioned mesh, tile kernel: the ghost slabs in runs of eight (their sums pass)
    int64_t n_ghost_tiles = 0;
    // partitioned mesh: per peer the chunk lists (slab * 8 + octant) to send / to receive, on the device
    std::vector<int32_t*> d_send_chunks, d_recv_chunks;
    std::vector<int64_t> n_send_chunks, n_recv_chunks;
    std::vector<int32_t*> d_send_slabs, d_recv_slabs;   // ... and the slab lists themselves (the cells' sums travel too)
    bool check = false;            // UFS_DVM_CHECK: every step call verifies the carried sums of a few cells against f
    double* d_check = nullptr;     // scratch of the check
    uint64_t check_rng = 0x9E3779B97F4A7C15ull;
    bool push_sums = false;        // fused exchange: the peers' step kernels also write the ghost cells' sums
    bool ghost_sums_pushed = false; // the ghost rows of the sums hold the owners' sums of the current f (unpacked, or pushed)
    bool ghosts_fresh = false;     // the ghost slabs of f[cur] and their sums are those of the peers' current f
    bool sums_valid = false;       // d_sums[cur] describes f[cur]
    int parity = 0;
    StepLaunch plan{};
    int64_t launches = 0;
    // optional timing of the main kernel of each step (ufs_dvm_profile)
    static constexpr int MAX_PROF = 64;
    cudaEvent_t prof_ev[MAX_PROF][2] = {};
    int prof_n = 0;
    bool prof_on = false;
    int sticky = UFS_DVM_OK;
    std::string err;
};

namespace {

int fail(ufs_dvm_t h, int code, const std::string& msg) {
    if (h) h->err = msg;
    return code;
}
int cuda_fail(ufs_dvm_t h, cudaError_t e, const char* what) {
    h->sticky = UFS_DVM_ECUDA;
    return fail(h, UFS_DVM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call, what)                                        \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(h, e__, what); \
    } while (0)

template <typename T>
int upload(ufs_dvm_t h, T** dst, const void* src, size_t bytes, const char* what) {
    *dst = nullptr;
    if (bytes == 0) return UFS_DVM_OK;
    CU(cudaMalloc(reinterpret_cast<void**>(dst), bytes), what);
    CU(cudaMemcpyAsync(*dst, src, bytes, cudaMemcpyHostToDevice, h->stream), what);
    return UFS_DVM_OK;
}

StepParams make_params(ufs_dvm_t h, double dt) {
    StepParams p{};
    const VelLayout& v = h->mesh.vel;
    p.f_in = h->f[h->cur];
    p.f_out = h->f[h->cur ^ 1];
    p.cells = h->d_cells;
    p.tables = h->d_tables;
    p.fluid = h->d_fluid;
    p.vel = h->d_vel;
    p.slot_k = h->d_slot_k;
    p.mirror_slot = h->d_mirror;
    p.flags = h->d_flags;
    p.Nv = v.Nv;
    p.n_kin = (int32_t)h->mesh.n_kin;
    for (int a = 0; a < 3; a++) { p.nv[a] = v.nv[a]; p.nh[a] = v.nh[a]; }
    p.collide = std::isinf(h->kn) ? 0 : 1;
    p.dt = dt;
    p.w = v.w;
    p.inv_len = 1.0 / h->domain_len;
    p.inv_kn = p.collide ? 1.0 / h->kn : 0.0;
    p.visc_exp = h->visc_exp;
    p.nu_pref = h->nu_pref;
    p.counter = h->d_counter + h->parity;
    p.counter_reset = h->d_counter + (h->parity ^ 1);
    p.ring_stages = h->plan.stages;
    p.sums_in = h->d_sums[h->cur];
    p.sums_out = h->d_sums[h->cur ^ 1];
    p.ghost_sums = h->d_ghost_sums;
    p.tabs = h->d_tabs;
    p.n_tables = h->mesh.n_tables;
    p.tile_hdr = h->d_tile_hdr;
    p.tile_pieces = h->d_tile_pieces;
    p.tile_cellidx = h->d_tile_cellidx;
    p.tiles_have_fluid = h->mesh.tiles_have_fluid ? 1 : 0;
    p.fluid_pieces = h->d_fluid_pieces;
    p.n_tiles = (int32_t)h->mesh.tiles.size();
    p.tile_pmax = h->mesh.tile_pmax;
    p.tile_push = h->d_tile_push;
    p.push_parity = h->cur ^ 1;
    if (v.fast) {
        for (int r = 0; r < v.nh[0] && r < 16; r++) {
            const double x = v.xi[0][v.nh[0] + r];
            p.xpow[0][r] = x; p.xpow[1][r] = x * x; p.xpow[2][r] = x * x * x;
            p.xf[r] = (float)x;
        }
        for (int r = 0; r < 16; r++) {
            p.yabs[r] = r < v.nh[1] ? v.xi[1][v.nh[1] + r] : 0.0;
            p.zabs[r] = r < v.nh[2] ? v.xi[2][v.nh[2] + r] : 0.0;
        }
    }
    return p;
}

// The 35 velocity sums (layout of step_stream.cu: H[5], then G[axis][sign][5]) of one ghost state given by its
// values in slot order, exactly as the step kernel sees them (storage-type rounding included).
template <typename F>
void ghost_state_sums(const VelLayout& v, F value_of_slot, double* out) {
    for (int i = 0; i < SUMS_STRIDE; i++) out[i] = 0.0;
    for (int64_t sl = 0; sl < v.Nv; sl++) {
        const double x[3] = {v.xi[0][v.slot_k[sl * 4]], v.xi[1][v.slot_k[sl * 4 + 1]], v.xi[2][v.slot_k[sl * 4 + 2]]};
        const double m[5] = {1.0, x[0], x[1], x[2], x[0] * x[0] + x[1] * x[1] + x[2] * x[2]};
        const double f = value_of_slot(sl);
        for (int k = 0; k < 5; k++) out[k] += m[k] * f;
        for (int a = 0; a < 3; a++) {
            if (x[a] == 0.0) continue;
            const int s = x[a] > 0.0 ? 1 : 0;
            for (int k = 0; k < 5; k++) out[5 + (2 * a + s) * 5 + k] += m[k] * std::fabs(x[a]) * f;
        }
    }
}

int create_common(const ufs_dvm_desc* desc, ufs_dvm_t* out, const int32_t* rank_of_leaf = nullptr, int my_rank = 0, int n_ranks = 1) {
    if (!out) return UFS_DVM_EINVAL;
    *out = nullptr;
    if (!desc) return UFS_DVM_EINVAL;
    ufs_dvm_t h = new (std::nothrow) ufs_dvm_s();
    if (!h) return UFS_DVM_ENOMEM;
    *out = h;  // returned even on failure so that the caller can read last_error, then destroy
    h->storage = desc->storage;
    h->kn = desc->kn; h->visc_exp = desc->visc_exp; h->nu_pref = desc->nu_prefactor; h->domain_len = desc->domain_len;
    try {
        std::string err;
        int rc = flatten(*desc, h->mesh, err);
        if (rc) return fail(h, rc, err);
        if (rank_of_leaf) {
            if (!h->mesh.vel.fast) return fail(h, UFS_DVM_EINVAL, "a partitioned mesh needs the octant layout (even, symmetric velocity grid)");
            rc = restrict_to_rank(h->mesh, rank_of_leaf, my_rank, n_ranks, err);
            if (rc) return fail(h, rc, err);
        }
    } catch (const std::bad_alloc&) {
        return fail(h, UFS_DVM_ENOMEM, "out of host memory while flattening");
    } catch (...) {
        return fail(h, UFS_DVM_EINVAL, "unexpected failure while flattening");
    }
    const char* why = "";
    int rc = step_plan(h->storage, h->mesh.vel, &h->plan, &why);
    if (rc) return fail(h, rc, why);
    // Kernel choice: the tile kernel (step_tiles.cu) where the velocity grid fits it, else the streaming step with one
    // row per thread (step_rows.cu), else one vector per thread (step_stream.cu), else one CTA per cell (kernels.cu).
    // UFS_DVM_KERNEL = rows | stream | cell forces the later ones (A/B timing, tests of the fallbacks).  The grid size
    // (one CTA per SM) is filled in by ufs_dvm_create once the device is known.
    const char* force = std::getenv("UFS_DVM_KERNEL");
    const bool want_cell = force && std::strcmp(force, "cell") == 0;
    const bool want_vec = force && std::strcmp(force, "stream") == 0;
    const bool want_rows = force && std::strcmp(force, "rows") == 0;
    if (!want_cell) {
        int pmax = 0;
        StepLaunch cand{};
        // (piece codes keep 30 bits for (slab or fluid ghost) * 8 + octant)
        const bool codes_fit = h->mesh.n_slabs < (int64_t(1) << 27) && (int64_t)h->mesh.fluid.size() < (int64_t(1) << 27);
        if (!want_vec && !want_rows && codes_fit && tiles_plan(h->storage, h->mesh.vel, 1, &cand, &pmax)) {
            h->plan = cand;
            try {
                build_tiles(h->mesh, pmax);
            } catch (const std::bad_alloc&) {
                return fail(h, UFS_DVM_ENOMEM, "out of host memory while building the tile records");
            }
        } else if (!want_vec && rows_plan(h->storage, h->mesh.vel, 1, &cand)) h->plan = cand;
        else if (stream_plan(h->storage, h->mesh.vel, 1, &cand)) h->plan = cand;
    }
    h->plan.test_stall = std::getenv("UFS_DVM_TEST_STALL") ? 1 : 0;
    h->check = std::getenv("UFS_DVM_CHECK") != nullptr;
    return UFS_DVM_OK;
}

}  // namespace

extern "C" {

int ufs_dvm_create_host(const ufs_dvm_desc* desc, ufs_dvm_t* out) { return create_common(desc, out); }

static int create_device(ufs_dvm_t h, void* f_dev[2], void* cuda_stream);

int ufs_dvm_create(const ufs_dvm_desc* desc, void* f_dev[2], void* cuda_stream, ufs_dvm_t* out) {
    int rc = create_common(desc, out);
    if (rc) return rc;
    return create_device(*out, f_dev, cuda_stream);
}

int ufs_dvm_partition(const ufs_dvm_desc* desc, int32_t n_ranks, double w_kinetic, double w_fluid, int32_t* rank_of_leaf) {
    if (!desc) return UFS_DVM_EINVAL;
    std::string err;
    try {
        return partition_leaves(*desc, n_ranks, w_kinetic, w_fluid, rank_of_leaf, err);
    } catch (...) {
        return UFS_DVM_ENOMEM;
    }
}

int ufs_dvm_create_part_host(const ufs_dvm_desc* desc, const int32_t* rank_of_leaf, int32_t my_rank, int32_t n_ranks, ufs_dvm_t* out) {
    if (!rank_of_leaf) { if (out) *out = nullptr; return UFS_DVM_EINVAL; }
    return create_common(desc, out, rank_of_leaf, my_rank, n_ranks);
}

int ufs_dvm_create_part(const ufs_dvm_desc* desc, const int32_t* rank_of_leaf, int32_t my_rank, int32_t n_ranks, void* f_dev[2],
                        void* cuda_stream, ufs_dvm_t* out) {
    int rc = ufs_dvm_create_part_host(desc, rank_of_leaf, my_rank, n_ranks, out);
    if (rc) return rc;
    ufs_dvm_t h = *out;
    if ((rc = create_device(h, f_dev, cuda_stream))) return rc;
    // the ghost slabs start finite (chunks that never arrive are never used, but their sums are formed)
    const FlatMesh& m = h->mesh;
    const size_t elem = h->storage == UFS_STORE_F32 ? 4 : 8;
    const size_t off = (size_t)m.n_kin * m.vel.Nv * elem, len = (size_t)(m.n_slabs - m.n_kin) * m.vel.Nv * elem;
    if (len)
        for (int b = 0; b < 2; b++) CU(cudaMemsetAsync(static_cast<char*>(h->f[b]) + off, 0, len, h->stream), "clear ghost slabs");
    // chunk lists per peer
    h->d_send_chunks.assign(m.n_ranks, nullptr); h->d_recv_chunks.assign(m.n_ranks, nullptr);
    h->n_send_chunks.assign(m.n_ranks, 0); h->n_recv_chunks.assign(m.n_ranks, 0);
    h->d_send_slabs.assign(m.n_ranks, nullptr); h->d_recv_slabs.assign(m.n_ranks, nullptr);
    for (int pr = 0; pr < m.n_ranks; pr++)
        for (int dir = 0; dir < 2; dir++) {
            const std::vector<int32_t>& slab = dir ? m.recv_slab[pr] : m.send_slab[pr];
            if ((rc = upload(h, dir ? &h->d_recv_slabs[pr] : &h->d_send_slabs[pr], slab.data(), slab.size() * 4, "upload halo slab lists"))) return rc;
            const std::vector<uint8_t>& mask = dir ? m.recv_mask[pr] : m.send_mask[pr];
            std::vector<int32_t> chunks;
            for (size_t i = 0; i < slab.size(); i++)
                for (int o = 0; o < 8; o++)
                    if (mask[i] & (1u << o)) chunks.push_back(slab[i] * 8 + o);
            (dir ? h->n_recv_chunks : h->n_send_chunks)[pr] = (int64_t)chunks.size();
            if ((rc = upload(h, dir ? &h->d_recv_chunks[pr] : &h->d_send_chunks[pr], chunks.data(), chunks.size() * 4, "upload halo chunk lists"))) return rc;
            CU(cudaStreamSynchronize(h->stream), "upload");   // `chunks` dies here
        }
    if (h->plan.ring == 4 && m.n_slabs > m.n_kin) {
        // the ghost slabs as tiles of up to eight consecutive slabs: ufs_dvm_halo_done sums them with the tile kernel's
        // sums-only pass (a tile's header is all that pass reads)
        std::vector<TileHdr> gt;
        for (int64_t s = m.n_kin; s < m.n_slabs; s += TILE_CELLS) {
            TileHdr t{};
            t.s0 = (int32_t)s;
            t.nc = (int32_t)std::min<int64_t>(TILE_CELLS, m.n_slabs - s);
            gt.push_back(t);
        }
        h->n_ghost_tiles = (int64_t)gt.size();
        if ((rc = upload(h, &h->d_ghost_tiles, gt.data(), gt.size() * sizeof(TileHdr), "upload ghost tiles"))) return rc;
        CU(cudaStreamSynchronize(h->stream), "upload");   // `gt` dies here
    }
    h->ghosts_fresh = m.n_slabs == m.n_kin;
    return UFS_DVM_OK;
}

static int create_device(ufs_dvm_t h, void* f_dev[2], void* cuda_stream) {
    int rc = UFS_DVM_OK;
    if (!f_dev || ((!f_dev[0] || !f_dev[1]) && h->mesh.n_kin > 0)) return fail(h, UFS_DVM_EINVAL, "f_dev[0] and f_dev[1] must be device buffers");
    if (h->mesh.n_kin > 0 && (f_dev[0] == f_dev[1] || ((uintptr_t)f_dev[0] & 15) || ((uintptr_t)f_dev[1] & 15)))
        return fail(h, UFS_DVM_EINVAL, "the two f buffers must be distinct and 16-byte aligned");
    h->f[0] = f_dev[0]; h->f[1] = f_dev[1];
    h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    h->device = true;
    const FlatMesh& m = h->mesh;
    const VelLayout& v = m.vel;
    if ((rc = upload(h, &h->d_cells, m.recs.data(), m.recs.size() * sizeof(CellRec), "upload cell records"))) return rc;
    if ((rc = upload(h, &h->d_fluid, m.fluid.data(), m.fluid.size() * sizeof(FluidGhost), "upload fluid ghosts"))) return rc;
    VelDev vd{};
    std::memcpy(vd.xi, v.xi, sizeof vd.xi);
    for (int a = 0; a < 3; a++) { vd.nv[a] = v.nv[a]; vd.nh[a] = v.nh[a]; }
    if ((rc = upload(h, &h->d_vel, &vd, sizeof vd, "upload velocity grid"))) return rc;
    if ((rc = upload(h, &h->d_slot_k, v.slot_k.data(), v.slot_k.size(), "upload slot table"))) return rc;
    std::vector<int32_t> mir((size_t)3 * v.Nv);
    for (int a = 0; a < 3; a++) std::memcpy(mir.data() + (size_t)a * v.Nv, v.mirror_slot[a].data(), (size_t)v.Nv * 4);
    if ((rc = upload(h, &h->d_mirror, mir.data(), mir.size() * 4, "upload mirror table"))) return rc;
    // inflow ghost tables in the storage type
    std::vector<float> tab32;
    const void* tab = m.tables.data();
    size_t tab_bytes = m.tables.size() * 8;
    if (h->storage == UFS_STORE_F32) {
        tab32.assign(m.tables.begin(), m.tables.end());
        tab = tab32.data();
        tab_bytes = tab32.size() * 4;
    }
    if ((rc = upload(h, &h->d_tables, tab, tab_bytes, "upload inflow tables"))) return rc;
    CU(cudaMalloc(reinterpret_cast<void**>(&h->d_flags), 4), "allocate flags");
    CU(cudaMemsetAsync(h->d_flags, 0, 4, h->stream), "clear flags");
    CU(cudaMalloc(reinterpret_cast<void**>(&h->d_counter), 8), "allocate cell counters");
    CU(cudaMemsetAsync(h->d_counter, 0, 8, h->stream), "clear cell counters");
    if (h->plan.ring >= 2) {
        int dev = 0, sms = 0;
        CU(cudaGetDevice(&dev), "get device");
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "query SM count");
        h->plan.grid = sms;   // persistent kernels: one CTA per SM
    }
    if (h->plan.ring == 4) {
        if ((rc = upload(h, &h->d_tile_hdr, m.tiles.data(), m.tiles.size() * sizeof(TileHdr), "upload tile headers"))) return rc;
        if ((rc = upload(h, &h->d_tile_pieces, m.tile_pieces.data(), m.tile_pieces.size() * 4, "upload tile piece lists"))) return rc;
        if ((rc = upload(h, &h->d_tile_cellidx, m.tile_cellidx.data(), m.tile_cellidx.size(), "upload tile index tables"))) return rc;
        if (m.tiles_have_fluid) {
            std::vector<double> fp;
            tiles_fluid_pieces(m, h->storage, fp);
            if ((rc = upload(h, &h->d_fluid_pieces, fp.data(), fp.size() * sizeof(double), "upload fluid pieces"))) return rc;
            CU(cudaStreamSynchronize(h->stream), "upload");   // fp dies here
        }
    }
    if (h->plan.ring >= 2 && m.n_kin > 0) {
        const size_t elem = h->storage == UFS_STORE_F32 ? 4 : 8;
        const size_t sums_bytes = (size_t)m.n_slabs * SUMS_STRIDE * sizeof(double);   // ghost cells carry sums too
        for (int b = 0; b < 2; b++) CU(cudaMalloc(reinterpret_cast<void**>(&h->d_sums[b]), sums_bytes), "allocate velocity sums");
        CU(cudaMalloc(&h->d_tabs, (size_t)m.n_kin * stream_tabn(v) * elem), "allocate factor tables");
        // sums of the ghost states (inflow tables, fluid leaves), from the values the kernel will read
        const size_t ng = (size_t)m.n_tables + m.fluid.size();
        std::vector<double> gs(ng * SUMS_STRIDE);
        const bool f32 = h->storage == UFS_STORE_F32;
        for (int t = 0; t < m.n_tables; t++) {
            const double* tb = m.tables.data() + (size_t)t * v.Nv;
            ghost_state_sums(v, [&](int64_t sl) { return f32 ? (double)(float)tb[sl] : tb[sl]; }, gs.data() + (size_t)t * SUMS_STRIDE);
        }
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t g = 0; g < (int64_t)m.fluid.size(); g++) {
            const FluidGhost& fg = m.fluid[g];
            ghost_state_sums(v, [&](int64_t sl) {
                const double b = fg.amp * fg.g[2][v.slot_k[sl * 4 + 2]] * fg.g[1][v.slot_k[sl * 4 + 1]];
                const double val = b * fg.g[0][v.slot_k[sl * 4]];
                return f32 ? (double)(float)val : val;
            }, gs.data() + ((size_t)m.n_tables + g) * SUMS_STRIDE);
        }
        if ((rc = upload(h, &h->d_ghost_sums, gs.data(), gs.size() * sizeof(double), "upload ghost sums"))) return rc;
        CU(cudaStreamSynchronize(h->stream), "upload");  // gs dies at the end of this block
    }
    CU(cudaStreamSynchronize(h->stream), "upload");  // the host vectors above die at return
    return UFS_DVM_OK;
}

// The 35 velocity sums of the current f, which nobody has summed yet (first step, or the caller rewrote f).
static int enqueue_sums(ufs_dvm_t h, const StepParams& p) {
    if (h->plan.ring == 4) {
        CU(launch_tile_sums(h->storage, h->plan, p, h->f[h->cur], h->d_sums[h->cur], h->stream), "sums kernel launch");
        h->parity ^= 1;   // the pass drew its tile tickets from this parity's counter and zeroed the other one
    } else {
        CU(launch_sums(h->storage, h->plan, p, h->f[h->cur], h->d_sums[h->cur], h->stream), "sums kernel launch");
    }
    h->sums_valid = true;
    h->launches++;
    return UFS_DVM_OK;
}

int ufs_dvm_step(ufs_dvm_t h, double dt, int nsteps) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (!(dt > 0) || nsteps < 0) return fail(h, UFS_DVM_EINVAL, "dt must be positive and nsteps >= 0");
    const bool has_ghosts = h->mesh.n_slabs > h->mesh.n_kin;
    if (has_ghosts && nsteps > 1) return fail(h, UFS_DVM_EINVAL, "a partitioned mesh is stepped one step at a time (ghost exchange in between)");
    if (has_ghosts && nsteps == 1 && !h->ghosts_fresh)
        return fail(h, UFS_DVM_EINVAL, "ghost cells are stale: exchange them (ufs_dvm_halo_pack / unpack) and call ufs_dvm_halo_done before the step");
    const bool stream = h->plan.ring >= 2 && h->mesh.n_kin > 0;
    if (h->check && stream && h->sums_valid && nsteps > 0) {
        // check mode: the carried sums must still describe f (a caller that rewrote f and forgot ufs_dvm_f_changed gets
        // UFS_DVM_EINVAL at the next ufs_dvm_sync instead of Maxwellians from stale sums)
        if (!h->d_check) CU(cudaMalloc(reinterpret_cast<void**>(&h->d_check), SUMS_STRIDE * sizeof(double)), "allocate check scratch");
        const StepParams p = make_params(h, dt);
        for (int i = 0; i < 8; i++) {
            h->check_rng = h->check_rng * 6364136223846793005ull + 1442695040888963407ull;
            const int64_t cell = (int64_t)((h->check_rng >> 33) % (uint64_t)h->mesh.n_kin);
            CU(launch_check_sums(h->storage, h->plan, p, h->f[h->cur], h->d_sums[h->cur], cell, h->d_check, h->d_flags, h->stream), "check kernel launch");
            h->launches += 2;
        }
    }
    for (int s = 0; s < nsteps; s++) {
        if (stream && !h->sums_valid) {
            const int rc = enqueue_sums(h, make_params(h, dt));
            if (rc) return rc;
        }
        const StepParams p = make_params(h, dt);
        StepLaunch plan = h->plan;
        plan.ev0 = plan.ev1 = nullptr;
        if (h->prof_on && h->prof_n < ufs_dvm_s::MAX_PROF) {
            for (int e = 0; e < 2; e++)
                if (!h->prof_ev[h->prof_n][e]) CU(cudaEventCreate(&h->prof_ev[h->prof_n][e]), "create event");
            plan.ev0 = h->prof_ev[h->prof_n][0];
            plan.ev1 = h->prof_ev[h->prof_n][1];
            h->prof_n++;
        }
        CU(launch_step(h->storage, plan, p, h->stream), "step kernel launch");
        h->cur ^= 1;
        // every streaming launch draws its tickets from one counter and zeroes the other (the fused exchange has two per step)
        const int nl = h->plan.ring == 4 ? tiles_launches_per_step(plan, p) : 1;
        if (nl & 1) h->parity ^= 1;
        if (has_ghosts) h->ghosts_fresh = false;
        h->ghost_sums_pushed = h->plan.push_on && h->push_sums;   // by the peers' step kernels of this round (protocol: ufs_dvm.h)
        if (h->mesh.n_kin > 0) h->launches += ((stream && p.collide) ? 1 : 0) + nl;
    }
    return UFS_DVM_OK;
}

int ufs_dvm_moments(ufs_dvm_t h, double* mom_dev) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (!mom_dev && h->mesh.n_kin > 0) return fail(h, UFS_DVM_EINVAL, "mom_dev is NULL");
    if (h->plan.ring >= 2 && h->mesh.n_kin > 0) {
        if (!h->sums_valid) {
            const int rc = enqueue_sums(h, make_params(h, 1.0));
            if (rc) return rc;
        }
        const StepParams p = make_params(h, 1.0);
        CU(launch_moments_from_sums(p, h->d_sums[h->cur], mom_dev, h->stream), "moments kernel launch");
        h->launches++;
        return UFS_DVM_OK;
    }
    const StepParams p = make_params(h, 1.0);
    CU(launch_moments(h->storage, p, h->f[h->cur], mom_dev, h->stream), "moments kernel launch");
    if (h->mesh.n_kin > 0) h->launches++;
    return UFS_DVM_OK;
}

int ufs_dvm_sync(ufs_dvm_t h) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    CU(cudaStreamSynchronize(h->stream), "stream synchronize");
    int32_t flags = 0;
    CU(cudaMemcpy(&flags, h->d_flags, 4, cudaMemcpyDeviceToHost), "read flags");
    if ((flags & 2) && h->sticky == UFS_DVM_OK) {
        h->sticky = UFS_DVM_EINVAL;
        h->err = "UFS_DVM_CHECK: the carried velocity sums no longer describe f: f was rewritten without ufs_dvm_f_changed";
    }
    if ((flags & 1) && h->sticky == UFS_DVM_OK) {
        h->sticky = UFS_DVM_ENEWTON;
        h->err = "Newton iteration for the discrete Maxwellian failed in at least one cell (n <= 0, T <= 0 or no convergence)";
    }
    return h->sticky;
}

int ufs_dvm_destroy(ufs_dvm_t h) {
    if (!h) return UFS_DVM_OK;
    int rc = UFS_DVM_OK;
    if (h->device) {
        if (cudaStreamSynchronize(h->stream) != cudaSuccess) rc = UFS_DVM_ECUDA;
        cudaFree(h->d_cells); cudaFree(h->d_tables); cudaFree(h->d_fluid); cudaFree(h->d_vel);
        cudaFree(h->d_slot_k); cudaFree(h->d_mirror); cudaFree(h->d_flags); cudaFree(h->d_counter);
        if (!h->sums_are_callers) { cudaFree(h->d_sums[0]); cudaFree(h->d_sums[1]); }
        cudaFree(h->d_ghost_sums); cudaFree(h->d_tabs);
        cudaFree(h->d_tile_hdr); cudaFree(h->d_tile_pieces); cudaFree(h->d_tile_cellidx); cudaFree(h->d_fluid_pieces);
        cudaFree(h->d_check); cudaFree(h->d_tile_push); cudaFree(h->d_ghost_tiles);
        for (int32_t* q : h->d_send_chunks) cudaFree(q);
        for (int32_t* q : h->d_recv_chunks) cudaFree(q);
        for (int32_t* q : h->d_send_slabs) cudaFree(q);
        for (int32_t* q : h->d_recv_slabs) cudaFree(q);
        for (auto& pr : h->prof_ev) for (cudaEvent_t e : pr) if (e) cudaEventDestroy(e);
    }
    delete h;
    return rc;
}

int ufs_dvm_current(ufs_dvm_t h) { return h ? h->cur : UFS_DVM_EINVAL; }

int ufs_dvm_f_changed(ufs_dvm_t h) {
    if (!h) return UFS_DVM_EINVAL;
    h->sums_valid = false;
    return UFS_DVM_OK;
}

int ufs_dvm_layout(ufs_dvm_t h, int64_t* n_kinetic, int64_t* cell_of_slab, int32_t* vel_of_slot) {
    if (!h) return UFS_DVM_EINVAL;
    if (n_kinetic) *n_kinetic = h->mesh.n_kin;
    if (cell_of_slab) std::memcpy(cell_of_slab, h->mesh.cell_of_slab.data(), (size_t)h->mesh.n_kin * 8);
    if (vel_of_slot) std::memcpy(vel_of_slot, h->mesh.vel.vel_of_slot.data(), (size_t)h->mesh.vel.Nv * 4);
    return UFS_DVM_OK;
}

int ufs_dvm_faces(ufs_dvm_t h, int64_t* n_faces, int64_t* owner, int64_t* neigh, double* area, int8_t* axis, int8_t* ratio) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    const size_t n = m.f_owner.size();
    if (n_faces) *n_faces = (int64_t)n;
    if (owner) std::memcpy(owner, m.f_owner.data(), n * 8);
    if (neigh) std::memcpy(neigh, m.f_neigh.data(), n * 8);
    if (area) std::memcpy(area, m.f_area.data(), n * 8);
    if (axis) std::memcpy(axis, m.f_axis.data(), n);
    if (ratio) std::memcpy(ratio, m.f_ratio.data(), n);
    return UFS_DVM_OK;
}

int ufs_dvm_boundary_faces(ufs_dvm_t h, int64_t* n_faces, int64_t* cell, int8_t* axis, int8_t* side, double* area,
                           int8_t* kind, int64_t* state) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    const size_t n = m.b_cell.size();
    if (n_faces) *n_faces = (int64_t)n;
    if (cell) std::memcpy(cell, m.b_cell.data(), n * 8);
    if (axis) std::memcpy(axis, m.b_axis.data(), n);
    if (side) std::memcpy(side, m.b_side.data(), n);
    if (area) std::memcpy(area, m.b_area.data(), n * 8);
    if (kind) std::memcpy(kind, m.b_kind.data(), n);
    if (state) std::memcpy(state, m.b_state.data(), n * 8);
    return UFS_DVM_OK;
}

int ufs_dvm_run_host(ufs_dvm_t h, const void* f_host_in, void* f_host_out, double* mom_dev_scratch, double* mom_host,
                     double dt, int nsteps) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (!f_host_in || !mom_dev_scratch || !mom_host) return fail(h, UFS_DVM_EINVAL, "NULL buffer");
    if (h->mesh.partial) return fail(h, UFS_DVM_EINVAL, "ufs_dvm_run_host does not drive a partitioned mesh (ghost exchange between steps)");
    const size_t bytes = (size_t)h->mesh.n_kin * (size_t)h->mesh.vel.Nv * (h->storage == UFS_STORE_F32 ? 4 : 8);
    CU(cudaMemcpyAsync(h->f[h->cur], f_host_in, bytes, cudaMemcpyHostToDevice, h->stream), "copy f to the device");
    h->sums_valid = false;
    int rc = ufs_dvm_step(h, dt, nsteps);
    if (rc) return rc;
    if ((rc = ufs_dvm_moments(h, mom_dev_scratch))) return rc;
    CU(cudaMemcpyAsync(mom_host, mom_dev_scratch, (size_t)h->mesh.n_kin * 40, cudaMemcpyDeviceToHost, h->stream), "copy moments to the host");
    if (f_host_out) CU(cudaMemcpyAsync(f_host_out, h->f[h->cur], bytes, cudaMemcpyDeviceToHost, h->stream), "copy f to the host");
    return ufs_dvm_sync(h);
}

int ufs_dvm_tiles(ufs_dvm_t h, int64_t* n_tiles, int32_t* pmax, int32_t* hdr, uint32_t* pieces, uint8_t* cellidx,
                  int64_t* n_fluid_ghosts, int64_t* fluid_leaf) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    if (n_tiles) *n_tiles = (int64_t)m.tiles.size();
    if (pmax) *pmax = m.tile_pmax;
    if (hdr) std::memcpy(hdr, m.tiles.data(), m.tiles.size() * sizeof(TileHdr));
    if (pieces) std::memcpy(pieces, m.tile_pieces.data(), m.tile_pieces.size() * 4);
    if (cellidx) std::memcpy(cellidx, m.tile_cellidx.data(), m.tile_cellidx.size());
    if (n_fluid_ghosts) *n_fluid_ghosts = (int64_t)m.fluid_leaf.size();
    if (fluid_leaf) std::memcpy(fluid_leaf, m.fluid_leaf.data(), m.fluid_leaf.size() * 8);
    return UFS_DVM_OK;
}

int ufs_dvm_remap_plan(ufs_dvm_t old_h, ufs_dvm_t new_h, int64_t* n_entries, int64_t* off, int32_t* src, double* wgt,
                       int64_t* n_ghosts, int64_t* ghost_leaf) {
    if (!old_h || !new_h) return UFS_DVM_EINVAL;
    if (old_h->mesh.partial || new_h->mesh.partial) return fail(new_h, UFS_DVM_EINVAL, "mesh change of a partitioned mesh is not supported");
    RemapPlan plan;
    std::string err;
    const int rc = build_remap(old_h->mesh, new_h->mesh, plan, err);
    if (rc) return fail(new_h, rc, err);
    if (n_entries) *n_entries = (int64_t)plan.src.size();
    if (off) std::memcpy(off, plan.off.data(), plan.off.size() * 8);
    if (src) std::memcpy(src, plan.src.data(), plan.src.size() * 4);
    if (wgt) std::memcpy(wgt, plan.wgt.data(), plan.wgt.size() * 8);
    if (n_ghosts) *n_ghosts = (int64_t)plan.ghost_leaf.size();
    if (ghost_leaf) std::memcpy(ghost_leaf, plan.ghost_leaf.data(), plan.ghost_leaf.size() * 8);
    return UFS_DVM_OK;
}

int ufs_dvm_remesh(ufs_dvm_t old_h, const ufs_dvm_desc* new_desc, void* f_new_dev[2], void* cuda_stream, ufs_dvm_t* out,
                   int64_t counts[4]) {
    if (!out) return UFS_DVM_EINVAL;
    *out = nullptr;
    if (!old_h || !old_h->device) return UFS_DVM_EINVAL;
    if (old_h->sticky) return old_h->sticky;
    if (old_h->mesh.partial) return UFS_DVM_EINVAL;
    int rc = ufs_dvm_create(new_desc, f_new_dev, cuda_stream, out);
    if (rc) return rc;
    ufs_dvm_t h = *out;   // errors below are reported on the new handle
    if (h->storage != old_h->storage) return fail(h, UFS_DVM_EINVAL, "mesh change: the storage type must not change");
    for (int b = 0; b < 2; b++)
        if (h->mesh.n_kin > 0 && f_new_dev[0] == old_h->f[old_h->cur])
            return fail(h, UFS_DVM_EINVAL, "mesh change: f_new_dev[0] must not be the old handle's current buffer");
    RemapPlan plan;
    try {
        std::string err;
        rc = build_remap(old_h->mesh, h->mesh, plan, err);
        if (rc) return fail(h, rc, err);
    } catch (const std::bad_alloc&) {
        return fail(h, UFS_DVM_ENOMEM, "out of host memory while building the mesh-change map");
    }
    if (counts) { counts[0] = plan.n_copy; counts[1] = plan.n_prolong; counts[2] = plan.n_restrict; counts[3] = plan.n_from_fluid; }
    if (h->mesh.n_kin == 0) return UFS_DVM_OK;
    // the old handle's stream may differ: order the map after everything it has enqueued
    if (old_h->stream != h->stream) {
        cudaEvent_t ev;
        CU(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "create event");
        CU(cudaEventRecord(ev, old_h->stream), "record event");
        CU(cudaStreamWaitEvent(h->stream, ev, 0), "wait event");
        CU(cudaEventDestroy(ev), "destroy event");
    }
    int64_t* d_off = nullptr; int32_t* d_src = nullptr; double* d_wgt = nullptr; FluidGhost* d_gh = nullptr;
    if ((rc = upload(h, &d_off, plan.off.data(), plan.off.size() * 8, "upload remap offsets"))) return rc;
    if ((rc = upload(h, &d_src, plan.src.data(), plan.src.size() * 4, "upload remap sources"))) return rc;
    if ((rc = upload(h, &d_wgt, plan.wgt.data(), plan.wgt.size() * 8, "upload remap weights"))) return rc;
    if ((rc = upload(h, &d_gh, plan.ghosts.data(), plan.ghosts.size() * sizeof(FluidGhost), "upload remap ghosts"))) return rc;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev), "get device");
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "query SM count");
    CU(launch_remap(h->storage, old_h->f[old_h->cur], h->f[0], d_off, d_src, d_wgt, d_gh, h->d_slot_k, h->mesh.n_kin, h->mesh.vel.Nv, sms, h->stream),
       "remap kernel launch");
    h->launches++;
    h->cur = 0;
    h->sums_valid = false;
    // the map is read by that one launch only (the host vectors of `plan` die at return: wait for the uploads too)
    CU(cudaStreamSynchronize(h->stream), "mesh change");
    cudaFree(d_off); cudaFree(d_src); cudaFree(d_wgt); cudaFree(d_gh);
    return UFS_DVM_OK;
}

int ufs_dvm_part_layout(ufs_dvm_t h, int64_t* n_inner, int64_t* n_ghost, int64_t* first_global_slab, int64_t* leaf_of_slab, int32_t* owner_of_ghost) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    if (n_inner) *n_inner = m.n_kin;
    if (n_ghost) *n_ghost = m.n_slabs - m.n_kin;
    if (first_global_slab) *first_global_slab = m.first_global_slab;
    if (leaf_of_slab) std::memcpy(leaf_of_slab, m.cell_of_slab.data(), (size_t)m.n_slabs * 8);
    if (owner_of_ghost && !m.ghost_owner.empty()) std::memcpy(owner_of_ghost, m.ghost_owner.data(), m.ghost_owner.size() * 4);
    return UFS_DVM_OK;
}

int ufs_dvm_halo(ufs_dvm_t h, int32_t peer, int64_t* n_send, int32_t* send_slab, uint8_t* send_mask, int64_t* n_recv,
                 int32_t* recv_slab, uint8_t* recv_mask) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    if (!m.partial || peer < 0 || peer >= m.n_ranks) return fail(h, UFS_DVM_EINVAL, "not a partitioned mesh, or no such peer");
    if (n_send) *n_send = (int64_t)m.send_slab[peer].size();
    if (n_recv) *n_recv = (int64_t)m.recv_slab[peer].size();
    if (send_slab && !m.send_slab[peer].empty()) std::memcpy(send_slab, m.send_slab[peer].data(), m.send_slab[peer].size() * 4);
    if (send_mask && !m.send_mask[peer].empty()) std::memcpy(send_mask, m.send_mask[peer].data(), m.send_mask[peer].size());
    if (recv_slab && !m.recv_slab[peer].empty()) std::memcpy(recv_slab, m.recv_slab[peer].data(), m.recv_slab[peer].size() * 4);
    if (recv_mask && !m.recv_mask[peer].empty()) std::memcpy(recv_mask, m.recv_mask[peer].data(), m.recv_mask[peer].size());
    return UFS_DVM_OK;
}

static int64_t chunk_bytes_of(ufs_dvm_t h) {
    const VelLayout& v = h->mesh.vel;
    return (int64_t)v.nh[0] * v.nh[1] * v.nh[2] * (h->storage == UFS_STORE_F32 ? 4 : 8);
}

int ufs_dvm_halo_bytes(ufs_dvm_t h, int32_t peer, int64_t* send_bytes, int64_t* recv_bytes) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    if (!m.partial || peer < 0 || peer >= m.n_ranks) return fail(h, UFS_DVM_EINVAL, "not a partitioned mesh, or no such peer");
    int64_t ns = 0, nr = 0;
    for (uint8_t mk : m.send_mask[peer]) ns += __builtin_popcount(mk);
    for (uint8_t mk : m.recv_mask[peer]) nr += __builtin_popcount(mk);
    // behind the chunks: the 36 carried sums of every listed cell (streaming kernels; the one-CTA-per-cell kernels carry none)
    const int64_t tail = h->plan.ring >= 2 ? (int64_t)(SUMS_STRIDE * sizeof(double)) : 0;
    if (send_bytes) *send_bytes = ns * chunk_bytes_of(h) + (int64_t)m.send_slab[peer].size() * tail;
    if (recv_bytes) *recv_bytes = nr * chunk_bytes_of(h) + (int64_t)m.recv_slab[peer].size() * tail;
    return UFS_DVM_OK;
}

static int halo_copy(ufs_dvm_t h, int32_t peer, void* buf, bool pack) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    const FlatMesh& m = h->mesh;
    if (!m.partial || peer < 0 || peer >= m.n_ranks) return fail(h, UFS_DVM_EINVAL, "not a partitioned mesh, or no such peer");
    const int64_t n = pack ? h->n_send_chunks[peer] : h->n_recv_chunks[peer];
    if (n == 0) return UFS_DVM_OK;
    if (!buf || ((uintptr_t)buf & 15)) return fail(h, UFS_DVM_EINVAL, "the halo buffer must be a 16-byte aligned device buffer");
    CU(launch_halo_copy(pack, pack ? h->d_send_chunks[peer] : h->d_recv_chunks[peer], n, h->f[h->cur], buf, chunk_bytes_of(h), h->stream),
       "halo copy kernel launch");
    h->launches++;
    if (h->plan.ring >= 2) {
        // the cells' carried sums behind the chunks (a sender that has not summed its f yet does so now)
        if (pack && !h->sums_valid) {
            const int rc = enqueue_sums(h, make_params(h, 1.0));
            if (rc) return rc;
        }
        const int64_t n_slabs = (int64_t)(pack ? m.send_slab[peer].size() : m.recv_slab[peer].size());
        CU(launch_halo_sums(pack, pack ? h->d_send_slabs[peer] : h->d_recv_slabs[peer], n_slabs, h->d_sums[h->cur],
                            static_cast<char*>(buf) + n * chunk_bytes_of(h), h->stream), "halo sums kernel launch");
        h->launches++;
        if (!pack) h->ghost_sums_pushed = true;   // the ghost rows hold the owners' sums: nothing for ufs_dvm_halo_done to form
    }
    return UFS_DVM_OK;
}
int ufs_dvm_halo_pack(ufs_dvm_t h, int32_t peer, void* buf_dev) { return halo_copy(h, peer, buf_dev, true); }
int ufs_dvm_halo_unpack(ufs_dvm_t h, int32_t peer, const void* buf_dev) { return halo_copy(h, peer, const_cast<void*>(buf_dev), false); }

int ufs_dvm_halo_done(ufs_dvm_t h) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    const FlatMesh& m = h->mesh;
    const int64_t n_gh = m.n_slabs - m.n_kin;
    if (n_gh > 0 && h->plan.ring >= 2 && !h->ghost_sums_pushed) {
        // the velocity sums of the ghost cells, from the chunks that have just arrived (the step's Maxwellian needs
        // the upwind flux moments of every source; entries of chunks that never arrive are never read)
        StepParams p = make_params(h, 1.0);
        if (h->plan.ring == 4) {
            // the tile kernel's sums-only pass over the ghost tiles (slab numbers are those of the whole buffer)
            p.tile_hdr = h->d_ghost_tiles;
            p.n_tiles = (int32_t)h->n_ghost_tiles;
            CU(launch_tile_sums(h->storage, h->plan, p, h->f[h->cur], h->d_sums[h->cur], h->stream), "ghost sums kernel launch");
            h->parity ^= 1;   // the pass drew its tile tickets from this parity's counter and zeroed the other one
        } else {
            p.n_kin = (int32_t)n_gh;
            const size_t elem = h->storage == UFS_STORE_F32 ? 4 : 8;
            const char* f = static_cast<const char*>(h->f[h->cur]) + (size_t)m.n_kin * m.vel.Nv * elem;
            CU(launch_sums(h->storage, h->plan, p, f, h->d_sums[h->cur] + (size_t)m.n_kin * SUMS_STRIDE, h->stream), "ghost sums kernel launch");
        }
        h->launches++;
    }
    h->ghosts_fresh = true;
    return UFS_DVM_OK;
}

int ufs_dvm_sums_dev(ufs_dvm_t h, void** sums0, void** sums1) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (sums0) *sums0 = h->d_sums[0];
    if (sums1) *sums1 = h->d_sums[1];
    return UFS_DVM_OK;
}

int ufs_dvm_sums_use(ufs_dvm_t h, void* sums0, void* sums1) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (h->plan.ring < 2 || !h->d_sums[0]) return fail(h, UFS_DVM_EINVAL, "this handle carries no velocity sums");
    if (!sums0 || !sums1 || sums0 == sums1 || ((uintptr_t)sums0 & 15) || ((uintptr_t)sums1 & 15))
        return fail(h, UFS_DVM_EINVAL, "sums0 and sums1 must be two distinct 16-byte aligned device arrays");
    // what the library's arrays hold (sums of the current f, ghost rows) moves over; then they are released
    const size_t bytes = (size_t)h->mesh.n_slabs * SUMS_STRIDE * sizeof(double);
    void* mine[2] = {sums0, sums1};
    for (int b = 0; b < 2; b++) CU(cudaMemcpyAsync(mine[b], h->d_sums[b], bytes, cudaMemcpyDeviceToDevice, h->stream), "copy the sums");
    CU(cudaStreamSynchronize(h->stream), "copy the sums");
    if (!h->sums_are_callers) { cudaFree(h->d_sums[0]); cudaFree(h->d_sums[1]); }
    h->d_sums[0] = static_cast<double*>(sums0);
    h->d_sums[1] = static_cast<double*>(sums1);
    h->sums_are_callers = true;
    return UFS_DVM_OK;
}

int ufs_dvm_halo_push_setup(ufs_dvm_t h, void* const* peer_f0, void* const* peer_f1, const int32_t* const* dest_slab,
                            void* const* peer_sums0, void* const* peer_sums1) {
    if (!h) return UFS_DVM_EINVAL;
    if (h->sticky) return h->sticky;
    if (!h->mesh.partial) return fail(h, UFS_DVM_EINVAL, "not a partitioned mesh");
    if (h->plan.ring != 4) return fail(h, UFS_DVM_EINVAL, "the fused ghost exchange needs the tile kernel (k_tiles)");
    if (!peer_f0 || !peer_f1 || !dest_slab) return fail(h, UFS_DVM_EINVAL, "peer_f0, peer_f1 and dest_slab must be arrays of n_ranks entries");
    FlatMesh& m = h->mesh;
    const size_t elem = h->storage == UFS_STORE_F32 ? 4 : 8;
    std::string err;
    int rc;
    try {
        if ((peer_sums0 == nullptr) != (peer_sums1 == nullptr)) return fail(h, UFS_DVM_EINVAL, "peer_sums0 and peer_sums1: both or neither");
        rc = build_push(m, peer_f0, peer_f1, dest_slab, (int64_t)(m.vel.Nv * elem), peer_sums0, peer_sums1,
                        (int64_t)(SUMS_STRIDE * sizeof(double)), err);
    } catch (const std::bad_alloc&) {
        return fail(h, UFS_DVM_ENOMEM, "out of host memory");
    }
    if (rc) return fail(h, rc, err);
    h->plan.push_on = 1;
    h->plan.push_tiles = (int32_t)m.n_push_tiles;
    h->push_sums = peer_sums0 != nullptr;
    h->ghost_sums_pushed = false;
    if (!h->device) return UFS_DVM_OK;   // host-only handle: the records are built (ufs_dvm_push_entries), nothing to upload
    CU(cudaStreamSynchronize(h->stream), "stream synchronize");   // no step in flight reads the old headers
    cudaFree(h->d_tile_push);
    h->d_tile_push = nullptr;
    if ((rc = upload(h, &h->d_tile_push, m.tile_push.data(), m.tile_push.size() * sizeof(PushEntry), "upload push entries"))) return rc;
    // build_push has moved the tiles with push entries to the front: all three tile arrays go up again
    CU(cudaMemcpyAsync(h->d_tile_hdr, m.tiles.data(), m.tiles.size() * sizeof(TileHdr), cudaMemcpyHostToDevice, h->stream), "upload tile headers");
    CU(cudaMemcpyAsync(h->d_tile_pieces, m.tile_pieces.data(), m.tile_pieces.size() * 4, cudaMemcpyHostToDevice, h->stream), "upload tile piece lists");
    CU(cudaMemcpyAsync(h->d_tile_cellidx, m.tile_cellidx.data(), m.tile_cellidx.size(), cudaMemcpyHostToDevice, h->stream), "upload tile index tables");
    CU(cudaStreamSynchronize(h->stream), "upload");
    return UFS_DVM_OK;
}

int ufs_dvm_push_entries(ufs_dvm_t h, int64_t* n_entries, int64_t* n_push_tiles, int32_t* slab, uint8_t* mask, uint64_t* dst0, uint64_t* dst1,
                         uint64_t* sums0, uint64_t* sums1) {
    if (!h) return UFS_DVM_EINVAL;
    const FlatMesh& m = h->mesh;
    if (!h->plan.push_on) return fail(h, UFS_DVM_EINVAL, "ufs_dvm_halo_push_setup has not been called");
    if (n_entries) *n_entries = (int64_t)m.tile_push.size();
    if (n_push_tiles) *n_push_tiles = m.n_push_tiles;
    for (const TileHdr& t : m.tiles) {
        int64_t e = t.pad[0];
        for (int c = 0; c < t.nc; c++)
            for (uint32_t k = 0; k < (((uint32_t)t.pad[1] >> (4 * c)) & 15u); k++, e++) {
                if (slab) slab[e] = t.s0 + c;
                if (mask) mask[e] = (uint8_t)(m.tile_push[e].info & 0xffu);
                if (dst0) dst0[e] = m.tile_push[e].dst[0];
                if (dst1) dst1[e] = m.tile_push[e].dst[1];
                if (sums0) sums0[e] = m.tile_push[e].sums_dst[0];
                if (sums1) sums1[e] = m.tile_push[e].sums_dst[1];
            }
    }
    return UFS_DVM_OK;
}

int64_t ufs_dvm_launch_count(ufs_dvm_t h) { return h ? h->launches : 0; }

int ufs_dvm_profile(ufs_dvm_t h, int enable) {
    if (!h) return UFS_DVM_EINVAL;
    h->prof_on = enable != 0;
    h->prof_n = 0;
    return UFS_DVM_OK;
}

int ufs_dvm_kernel_ms(ufs_dvm_t h, double* mean_ms, int32_t* n_launches) {
    if (!h || !mean_ms || !n_launches) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    CU(cudaStreamSynchronize(h->stream), "stream synchronize");
    double sum = 0.0;
    for (int i = 0; i < h->prof_n; i++) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, h->prof_ev[i][0], h->prof_ev[i][1]), "event elapsed time");
        sum += ms;
    }
    *n_launches = h->prof_n;
    *mean_ms = h->prof_n ? sum / h->prof_n : 0.0;
    return UFS_DVM_OK;
}

int ufs_dvm_kernel_info(ufs_dvm_t h, int32_t* threads, int32_t* smem_bytes, int32_t* vec, int32_t* fast) {
    if (!h) return UFS_DVM_EINVAL;
    if (threads) *threads = h->plan.threads;
    if (smem_bytes) *smem_bytes = h->plan.smem_bytes;
    if (vec) *vec = h->plan.vec;
    if (fast) *fast = h->plan.fast;
    return UFS_DVM_OK;
}

const char* ufs_dvm_kernel_name(ufs_dvm_t h) {
    if (!h) return "";
    return h->plan.ring == 4 ? "k_tiles" : h->plan.ring == 3 ? "k_rows" : h->plan.ring == 2 ? "k_stream"
                             : (h->plan.fast ? "k_step_fast" : "k_step_generic");
}

const char* ufs_dvm_last_error(ufs_dvm_t h) { return h ? h->err.c_str() : "null handle"; }

}  // extern "C"

// ---------------------------------------------------------------- ufs_dvm_moments_static: moments without any allocation
// For callers that cannot allocate (CUDA graph capture, tight serving loops): the sums pass (k_sums) writes the 35
// velocity sums of every cell of the caller's f into a FIXED array in the library's device image instead of a
// cudaMalloc'ed buffer, and k_moments_from_sums reads them from there.  Every device that loads the library holds the
// array (UFS_DVM_STATIC_MAX_CELLS * 36 doubles = 2.25 MiB) until the process exits.  All calls on a device share it:
// calls that overlap on the GPU (different streams) race.  Nothing in it has to start at zero: k_sums writes all 36
// numbers of each cell before k_moments_from_sums, later on the same stream, reads them.
static __device__ __align__(256) double g_static_sums[(size_t)UFS_DVM_STATIC_MAX_CELLS * SUMS_STRIDE];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
double* g_static_sums_ptr[STATIC_MAX_DEVICES] = {};   // the array's DEVICE address, per device ordinal
std::mutex g_static_mu;

// In host code `g_static_sums` is only a stand-in for the symbol: its device address comes from the runtime, once per
// device, with that device current.
cudaError_t static_sums_address(int dev, double** out) {
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_sums_ptr[dev]) {
        double* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_static_sums);
        if (e != cudaSuccess) return e;
        g_static_sums_ptr[dev] = ptr;
    }
    *out = g_static_sums_ptr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" int ufs_dvm_moments_static(ufs_dvm_t h, const void* f_dev, double* mom_dev) {
    if (!h) return UFS_DVM_EINVAL;
    if (!h->device) return fail(h, UFS_DVM_EINVAL, "host-only handle");
    if (h->sticky) return h->sticky;
    if (h->mesh.n_kin == 0) return UFS_DVM_OK;
    if (!mom_dev) return fail(h, UFS_DVM_EINVAL, "mom_dev is NULL");
    if (h->plan.ring < 2)
        return fail(h, UFS_DVM_EINVAL, "ufs_dvm_moments_static needs the octant layout of the streaming kernels (even, symmetric velocity grid)");
    if (h->mesh.n_kin > UFS_DVM_STATIC_MAX_CELLS)
        return fail(h, UFS_DVM_EINVAL, "ufs_dvm_moments_static: " + std::to_string(h->mesh.n_kin) + " kinetic cells exceed the fixed scratch of UFS_DVM_STATIC_MAX_CELLS = "
                                           + std::to_string(UFS_DVM_STATIC_MAX_CELLS) + " cells; use ufs_dvm_moments");
    int dev = -1;
    CU(cudaGetDevice(&dev), "get device");
    cudaPointerAttributes attr{};
    CU(cudaPointerGetAttributes(&attr, h->d_flags), "pointer attributes");
    if (attr.device != dev || dev < 0 || dev >= STATIC_MAX_DEVICES)
        return fail(h, UFS_DVM_EINVAL, "ufs_dvm_moments_static: the handle's device (" + std::to_string(attr.device) + ") must be the current device (" + std::to_string(dev) + ")");
    double* scratch = nullptr;
    CU(static_sums_address(dev, &scratch), "address of the static scratch");
    const StepParams p = make_params(h, 1.0);
    CU(launch_sums(h->storage, h->plan, p, f_dev ? f_dev : h->f[h->cur], scratch, h->stream), "sums kernel launch");
    CU(launch_moments_from_sums(p, scratch, mom_dev, h->stream), "moments kernel launch");
    h->launches += 2;
    return UFS_DVM_OK;
}
