// flatten.hpp -- host-side octree flattener of the DVM step.
//
// Turns the caller's leaf list into what the device kernels consume:
//   * Morton ("N-order") numbering of the leaves, slabs = kinetic leaves in that order;
//   * the sorted interior face list (owner, neighbour, area, axis, level ratio) and the boundary-face
//     list (PAPER.md:51 boundary cells; PAPER.md:207 kinetic/fluid interface);
//   * per kinetic cell the upwind gather record derived from those faces -- the first-order form of the
//     paper's per-cell, per-sign-group stencil records m, alpha, a;
//   * the velocity-slot layout: the 8 sign groups ("octants") stored contiguously.
// Pure C++, no CUDA.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/ufs_dvm.h"

namespace ufs {

// How a source of upwind data is encoded in a gather record (one int32 per source).
// code < 0: unused.  Otherwise bits 28..30 = kind, bits 0..27 = index.
enum SrcKind : int32_t {
    SRC_SLAB = 0,    // slab `index` of the current f buffer, same velocity slot
    SRC_MIRROR = 1,  // slab `index` (the cell itself), slot of the velocity mirrored on this axis (specular)
    SRC_TABLE = 2,   // ghost table `index` (inflow Maxwellian), same slot
    SRC_FLUID = 3    // fluid ghost `index`: pointwise Maxwellian of frozen moments
};
constexpr int32_t SRC_SHIFT = 28;
constexpr int32_t SRC_INDEX_MASK = (1 << SRC_SHIFT) - 1;
inline int32_t src_code(SrcKind k, int64_t idx) { return (int32_t)((k << SRC_SHIFT) | (int32_t)idx); }

// One kinetic cell, 128 bytes: for each direction d = 2*axis + side (side 0 = low) up to 4 sources
// (1 = same level or coarser neighbour / ghost, 4 = finer neighbours, each weighted 1/4).
struct CellRec {
    int32_t src[6][4];
    int32_t level;
    int32_t flags;  // bit 0: every direction has exactly one source and none is SRC_FLUID; bit 1: no source is SRC_FLUID; bit 2: CELL_RINGFLUID
    int32_t masks;   // 3 bits per velocity octant o (bit a): the upwind face of o on axis a has four finer sources
    int32_t fmasks;  // 3 bits per octant: the upwind source on axis a is a fluid leaf (single source)
    int32_t pad[4];
};
static_assert(sizeof(CellRec) == 128, "CellRec must be 128 bytes");
constexpr int32_t CELL_SIMPLE = 1;
constexpr int32_t CELL_NOFLUID = 2;
constexpr int32_t CELL_RINGFLUID = 4;  // some source is SRC_FLUID, and every direction with one has that source alone

constexpr int NV_MAX = 64;  // per-axis node limit (tables live in shared memory)

struct VelLayout {
    int nv[3];
    int64_t Nv;
    double xi[3][NV_MAX];        // node values, canonical index
    double w;                    // quadrature weight dvx*dvy*dvz (midpoint rule)
    bool symmetric[3];           // vmin = -vmax on the axis
    bool fast;                   // every axis: even nv, symmetric => 8 equal octant chunks
    int nh[3];                   // nv/2 (fast path)
    int ncls[3][3];              // nodes per sign class (0: xi<0, 1: xi>0, 2: xi==0)
    std::vector<int32_t> vel_of_slot;      // [Nv] canonical index stored at each slot
    std::vector<int32_t> slot_of_vel;      // inverse
    std::vector<int32_t> mirror_slot[3];   // [Nv] slot of the velocity mirrored on axis a (if symmetric[a])
    std::vector<uint8_t> slot_k;           // [Nv][4] (kx,ky,kz,0) of each slot
};

struct FluidGhost {          // frozen Maxwellian of a FLUID leaf, separable factors
    double amp;              // n / (2 pi T)^{3/2}
    double g[3][NV_MAX];     // exp(-(xi_k - u_a)^2 / 2T), canonical index
};

// ---- tiles (step_tiles.cu): up to TILE_CELLS consecutive slabs stepped together, so that a chunk that is the upwind
// source of several cells of the tile (siblings of a Morton octet) is brought on chip once.  For each tile
// and velocity octant (sign group) the flattener lists the distinct source chunks ("pieces") and, per
// cell, which piece is its own chunk and which pieces are its upwind sources on each axis -- the first-order stencil
// records of PAPER.md:113-115, deduplicated per tile.
constexpr int TILE_CELLS = 8;
constexpr uint32_t PIECE_TABLE = 0x80000000u;  // piece code: bit 31 = inflow ghost table, bits 0..29 = (slab, table or fluid ghost) * 8 + octant
constexpr uint32_t PIECE_FLUID = 0x40000000u;  // ... bit 30 = a fluid ghost: the producer warps write its factor rows, nothing is copied
constexpr uint32_t PIECE_INDEX = 0x3fffffffu;
constexpr uint8_t IDX_NONE = 0xFF;             // cell index table: unused source
constexpr int CELLIDX_BYTES = 16;              // per (tile, octant, cell): [0] own piece, [1] flags, [2..3] fluid mask, [4+4a+k] source k on axis a
constexpr uint8_t CIDX_FOUR = 0x07;            // flags bits 0..2: axis a has four (finer) sources, each weighted 1/4
constexpr uint8_t CIDX_FLUID = 0x08;           // flags bit 3: some source of the cell is a fluid leaf (which: bit 4a + k of bytes [2..3])
// A fluid piece holds, as doubles, the 12 x factors g_x[rank] of the octant's x sign, then the row factors
// b[row] = amp g_z g_y of the stage's NRP rows: the leaf's Maxwellian at (row, rank) is b[row] g_x[rank] (separable, G13).
constexpr int FLUID_PIECE_GX = 0, FLUID_PIECE_B = 12;
struct TileHdr {                               // 32 bytes
    int32_t s0, nc;                            // first slab, cells
    uint8_t np[8];                             // pieces per octant
    uint8_t level[TILE_CELLS];
    int32_t pad[2];
};
static_assert(sizeof(TileHdr) == 32, "TileHdr must be 32 bytes");

// Fused ghost exchange (build_push): a cell whose chunks a peer rank needs is stored a second time by k_tiles, straight
// into that peer's ghost slab of the NEXT f.  One entry per (cell, peer); a tile's entries are consecutive, ordered by
// cell: TileHdr::pad[0] = index of the tile's first entry, pad[1] = eight 4-bit counts (entries of cell c in bits 4c..4c+3).
constexpr int PUSH_PER_CELL_MAX = 4;           // peers that may need one cell (more: the pack / unpack exchange serves)
struct PushEntry {                             // 48 bytes
    uint64_t dst[2];                           // address of the peer's ghost slab in its f buffer 0 / 1 (peer memory)
    uint64_t sums_dst[2];                      // address of that ghost cell's 36 velocity sums in the peer's sums array 0 / 1, or 0
    uint32_t info;                             // bits 0..7: octant mask of the chunks the peer needs
    uint32_t pad[3];
};
static_assert(sizeof(PushEntry) == 48, "PushEntry must be 48 bytes");

struct FlatMesh {
    int64_t n_leaves = 0, n_kin = 0;
    // ---- one rank's part of a partitioned mesh (restrict_to_rank).  n_kin counts the rank's own
    // ("inner") kinetic leaves, stored first; the ghost cells -- kinetic leaves of other ranks that are upwind sources of
    // inner cells -- follow ("inner cells are stored before ghost cells").  Unpartitioned: n_slabs = n_kin.
    int64_t n_slabs = 0;
    bool partial = false;
    int32_t my_rank = 0, n_ranks = 1;
    int64_t first_global_slab = 0;             // inner slab s is slab first_global_slab + s of the whole mesh
    std::vector<int32_t> ghost_owner;          // [n_slabs - n_kin] rank that owns each ghost cell
    // per peer rank: the chunks to send (inner slab, octant mask) and to receive (ghost slab, octant mask), both in
    // ascending order of the cell's global slab number, so that the k-th entry sent is the k-th entry the peer expects
    std::vector<std::vector<int32_t>> send_slab, recv_slab;
    std::vector<std::vector<uint8_t>> send_mask, recv_mask;
    int lmax = 0;
    std::vector<int64_t> order;         // Morton rank -> leaf
    std::vector<int64_t> rank;          // leaf -> Morton rank
    std::vector<int64_t> cell_of_slab;  // slab -> leaf
    std::vector<int64_t> slab_of_leaf;  // leaf -> slab or -1
    // interior faces (between non-SOLID leaves), sorted by (rank of owner, axis)
    std::vector<int64_t> f_owner, f_neigh;
    std::vector<double> f_area;
    std::vector<int8_t> f_axis, f_ratio;
    // boundary faces of non-SOLID leaves
    std::vector<int64_t> b_cell, b_state;
    std::vector<double> b_area;
    std::vector<int8_t> b_axis, b_side, b_kind;
    // device-bound data
    std::vector<CellRec> recs;          // [n_kin]
    std::vector<int64_t> fluid_leaf;    // fluid ghost index -> leaf
    std::vector<FluidGhost> fluid;      // [n fluid ghosts]
    int table_of_side[6];               // inflow side -> ghost table index or -1
    int n_tables = 0;
    std::vector<double> tables;         // [n_tables][Nv] inflow Maxwellians, SLOT order, fp64
    int64_t n_simple = 0;
    VelLayout vel;
    // the leaf list itself and its Morton start keys (depth lmax), kept for mesh changes (build_remap)
    std::vector<uint8_t> leaf_level, leaf_kind;
    std::vector<double> leaf_fluid;         // [n_leaves][5] or empty
    std::vector<uint64_t> start_keys;       // [n_leaves] Morton-sorted (position r = leaf order[r])
    // tiles (filled by build_tiles)
    std::vector<uint8_t> octet_start;       // [n_kin] 1: slabs s..s+7 are the eight leaf children of one parent, all kinetic
    int tile_pmax = 0;                      // piece-list stride
    std::vector<TileHdr> tiles;
    std::vector<uint32_t> tile_pieces;      // [n_tiles][8 octants][tile_pmax]
    std::vector<uint8_t> tile_cellidx;      // [n_tiles][8 octants][TILE_CELLS][CELLIDX_BYTES]
    bool tiles_have_fluid = false;          // some piece is a fluid ghost: the kernel's FLUID instantiation
    std::vector<PushEntry> tile_push;       // fused ghost exchange (build_push): the tiles' push entries
    int64_t n_push_tiles = 0;               // ... and how many tiles have some (build_push moves them to the front)
};

// Returns UFS_DVM_OK or an error code with a message in `err`.
int flatten(const ufs_dvm_desc& d, FlatMesh& out, std::string& err);

// Mesh change (reading G20): every slab of the new mesh as a weighted sum of sources of
// the old one -- one source of weight 1 where an old leaf covers the new one (unchanged leaf, or refinement: injection),
// the old leaves inside it with their volume fractions where the new leaf is coarser (restriction).  A source is an old
// slab (src >= 0) or the frozen Maxwellian of an old FLUID leaf (src = -1 - ghost index).
struct RemapPlan {
    std::vector<int64_t> off;          // [n_new_kin + 1]
    std::vector<int32_t> src;
    std::vector<double> wgt;
    std::vector<FluidGhost> ghosts;    // factors of the old FLUID leaves that became KINETIC
    std::vector<int64_t> ghost_leaf;   // ... and which old leaves they are
    int64_t n_copy = 0, n_prolong = 0, n_restrict = 0, n_from_fluid = 0;
};
int build_remap(const FlatMesh& old_mesh, const FlatMesh& new_mesh, RemapPlan& plan, std::string& err);

// Space-filling-curve partition (Fig. 3): the leaves in N-order, each weighted by its cost (w_kinetic for
// KINETIC, w_fluid for FLUID, 0 for SOLID), cut into n_ranks consecutive ranges of equal weight: leaf number r of the
// curve goes to rank floor(W_before(r) * n_ranks / W_total), so every rank's weight is within one leaf of the mean.
int partition_leaves(const ufs_dvm_desc& d, int n_ranks, double w_kinetic, double w_fluid, int32_t* rank_of_leaf, std::string& err);

// Turns the flattened WHOLE mesh into rank `my_rank`'s part: the rank's kinetic leaves (one range of consecutive slabs)
// first, then its ghost cells; gather records renumbered; the halo lists of every peer.  Face lists, ghost-state tables
// and the leaf arrays stay those of the whole mesh.
int restrict_to_rank(FlatMesh& m, const int32_t* rank_of_leaf, int my_rank, int n_ranks, std::string& err);

// Groups the slabs into tiles whose piece lists hold at most `pmax` pieces per octant (complete sibling octets where
// the mesh has them, else runs of consecutive slabs) and fills the tile arrays of `m`.
void build_tiles(FlatMesh& m, int pmax);

// Fused ghost exchange of a partitioned mesh: moves the tiles with cells some peer needs to the front of the tile arrays
// (m.n_push_tiles of them) and fills m.tile_push and the pad words of m.tiles from the send lists.  Per peer
// rank p: peer_f[b][p] = address (as this device reaches it) of rank p's f buffer b, dest_slab[p][i] = the ghost slab of
// rank p that takes this rank's i-th send slab (rank p's recv_slab list for this rank), slab_bytes = Nv * element size.
// peer_sums[b] (may be NULL): per peer the address of its velocity-sums array b ([slabs][sums_stride] doubles): the owner's
// sums of a pushed cell then go to the peer's ghost row as well.
int build_push(FlatMesh& m, const void* const* peer_f0, const void* const* peer_f1, const int32_t* const* dest_slab, int64_t slab_bytes,
               const void* const* peer_sums0, const void* const* peer_sums1, int64_t sums_row_bytes, std::string& err);

}  // namespace ufs
