// kernels.cuh -- device-side parameter block and launchers of the DVM step kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <vector>

#include "flatten.hpp"

namespace ufs {

// Velocity-grid tables in device memory (one per handle).
struct VelDev {
    double xi[3][NV_MAX];  // node values, canonical index
    int32_t nv[3];
    int32_t nh[3];
};

// Everything a step launch needs.  Passed by value (kernel parameter space).
struct StepParams {
    const void* f_in;           // [n_kin][Nv] storage type, current f
    void* f_out;                // [n_kin][Nv] next f
    const CellRec* cells;       // [n_kin]
    const void* tables;         // [n_tables][Nv] storage type, slot order (inflow ghosts)
    const FluidGhost* fluid;    // [n_fluid_ghosts]
    const VelDev* vel;
    const uchar4* slot_k;       // [Nv] (kx,ky,kz,0) of each slot          (generic path, moments)
    const int32_t* mirror_slot; // [3][Nv]                                  (generic path)
    int32_t* flags;             // bit 0: a Newton solve failed
    int64_t Nv;
    int32_t n_kin;
    int32_t nv[3], nh[3];
    int32_t collide;            // 0: Kn = inf, pure transport
    double dt, w, inv_len, inv_kn, visc_exp, nu_pref;
    int32_t* counter;           // streaming kernels: cell-ticket counter of this launch (zero at launch)
    int32_t* counter_reset;     // the other launch parity's counter, zeroed by this launch
    int32_t ring_stages;        // slots in the shared-memory ring
    // streaming step (step_stream.cu)
    const double* sums_in;      // [n_kin][SUMS_STRIDE] velocity sums of f_in
    double* sums_out;           // [n_kin][SUMS_STRIDE] velocity sums of f_out
    const double* ghost_sums;   // [n_tables + n_fluid_ghosts][SUMS_STRIDE] the same sums of the ghost states
    void* tabs;                 // [n_kin][tabn] storage type: Maxwellian factor tables + dt*nu of this step
    int32_t n_tables;
    // row kernel (step_rows.cu): |xi_x| of the x ranks and its powers (uniform operands, constant bank)
    double xpow[3][16];         // [r-1][rank] = |xi_x|^r, r = 1..3
    float xf[16];               // |xi_x| in fp32
    double yabs[16], zabs[16];  // tile kernel: |xi_y|, |xi_z| by rank (constant bank: with 225 KB of shared memory L1 is ~3 KB)
    uint32_t smap[12];          // row / tile kernel: its shared-memory map (byte offsets), computed by the launcher
    // tile kernel (step_tiles.cu): the tile records of the flattener
    const TileHdr* tile_hdr;        // [n_tiles]
    const uint32_t* tile_pieces;    // [n_tiles][8][tile_pmax]
    const uint8_t* tile_cellidx;    // [n_tiles][8][TILE_CELLS][CELLIDX_BYTES]
    int32_t tiles_have_fluid;       // some piece is a fluid ghost (k_tiles' FLUID instantiation)
    const double* fluid_pieces;     // [n_fluid_ghosts * 8][row blocks][64] the fluid ghosts' factor rows (tiles_fluid_pieces)
    int32_t n_tiles, tile_pmax;
    // fused ghost exchange (k_tiles' PUSH instantiation): the tiles' push entries; which of PushEntry::dst[] is the NEXT f
    const PushEntry* tile_push;
    int32_t push_parity;
};

constexpr int SUMS_STRIDE = 36;  // doubles per cell in the sums arrays (35 used)

struct StepLaunch {
    int32_t threads, smem_bytes, vec, fast;
    int32_t ring;                  // 4: tile kernel (step_tiles.cu), 3: streaming step, one row per thread (step_rows.cu),
                                   // 2: streaming step, one vector per thread (step_stream.cu), 0: one CTA per cell (kernels.cu)
    int32_t grid, ncw, pieces, stages;  // ring kernel: CTAs, consumer warps, pieces per octant chunk, ring depth
    cudaEvent_t ev0, ev1;          // if set: recorded on the stream right before / after the main kernel of the step
    int32_t test_stall;            // UFS_DVM_TEST_STALL was set at creation: k_tiles stalls on purpose (watchdog test)
    int32_t push_on;               // ufs_dvm_halo_push_setup was called: the first push_tiles tiles are stepped by k_tiles' PUSH
    int32_t push_tiles;            //   instantiation (boundary cells also stored into the peers' ghost slabs), then the rest
};

// per-axis table stride (nodes rounded up to a multiple of 4)
__host__ __device__ inline int nvp_of(const int32_t nv[3]) {
    int m = nv[0] > nv[1] ? nv[0] : nv[1];
    m = m > nv[2] ? m : nv[2];
    return (m + 3) & ~3;
}

// Chooses the kernel variant for this storage type / grid and returns its launch geometry, or an
// error (negative) if the slab does not fit on chip.
int step_plan(int storage, const VelLayout& v, StepLaunch* plan, const char** why);

// step_stream.cu: the streaming step (k_prep + k_stream), the sums of a freshly written f, moments from sums.
bool stream_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan);
int stream_tabn(const VelLayout& v);
cudaError_t launch_stream(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t stream);
cudaError_t launch_prep(int storage, const StepParams& p, cudaStream_t stream);   // k_prep alone
// step_rows.cu: the same step with one velocity row per thread
bool rows_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan);
cudaError_t launch_rows(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t stream);
cudaError_t launch_sums(int storage, const StepLaunch& plan, const StepParams& p, const void* f, double* sums, cudaStream_t stream);
cudaError_t launch_moments_from_sums(const StepParams& p, const double* sums, double* mom, cudaStream_t stream);
// check mode: re-sum one cell of f and compare with its carried sums (flags bit 1 on mismatch)
cudaError_t launch_check_sums(int storage, const StepLaunch& plan, const StepParams& p, const void* f, const double* carried, int64_t cell,
                              double* scratch, int32_t* flags, cudaStream_t stream);

// step_tiles.cu: the same step over tiles of up to eight consecutive slabs (shared upwind chunks on chip)
bool tiles_plan(int storage, const VelLayout& v, int sm_count, StepLaunch* plan, int* pmax);
void tiles_fluid_pieces(const FlatMesh& m, int storage, std::vector<double>& out);   // host: the table behind StepParams::fluid_pieces
cudaError_t launch_tiles(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t stream);
int tiles_launches_per_step(const StepLaunch& plan, const StepParams& p);   // streaming launches of one step (1, or 2 with the fused exchange)
cudaError_t launch_tile_sums(int storage, const StepLaunch& plan, const StepParams& p, const void* f, double* sums, cudaStream_t stream);

// remap.cu: f of a new mesh from f of the old one (weighted sums of old slabs / frozen fluid Maxwellians)
cudaError_t launch_remap(int storage, const void* f_old, void* f_new, const int64_t* off, const int32_t* src, const double* wgt,
                         const FluidGhost* ghosts, const uchar4* slot_k, int64_t n_new, int64_t Nv, int sm_count, cudaStream_t stream);

// halo.cu: ghost-cell exchange of a partitioned mesh: chunk list -> contiguous buffer (pack) or back (unpack)
cudaError_t launch_halo_copy(bool pack, const int32_t* chunks, int64_t n_chunks, void* f, void* buf, int64_t chunk_bytes, cudaStream_t stream);
// ... and the listed cells' carried sums <-> the tail of the buffer ([n_slabs][SUMS_STRIDE] doubles)
cudaError_t launch_halo_sums(bool pack, const int32_t* slabs, int64_t n_slabs, double* sums, void* tail, cudaStream_t stream);

// Enqueue one fused step (transport + moments + discrete Maxwellian + relaxation) on `stream`.
cudaError_t launch_step(int storage, const StepLaunch& plan, const StepParams& p, cudaStream_t stream);

// Enqueue the moments kernel: mom[5][n_kin] = (n, n u, E) of f.
cudaError_t launch_moments(int storage, const StepParams& p, const void* f, double* mom, cudaStream_t stream);

}  // namespace ufs
