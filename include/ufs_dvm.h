/*
 * ufs_dvm.h -- C ABI of the B200-native DVM step (libufs_dvm.so).
 *
 * One explicit time step of the discrete-velocity-method Boltzmann solver of the Unified Flow
 * Solver's kinetic module (arxiv 1503.00707; citations are lines of the paper text PAPER.md):
 *
 *   Eq. 1   df/dt + xi . grad_x f = (1/Kn) I(f,f), non-dimensional, velocity unit sqrt(R T0)
 *   PAPER.md:93           f lives at the cell centres of a uniform Cartesian velocity grid (nv[0] x nv[1] x nv[2])
 *                         and of an adaptive octree Cartesian mesh in physical space
 *   Eq. 2  explicit finite-volume advection; here first-order upwind over every leaf face,
 *                         2:1 level-jump faces included
 *   PAPER.md:45           octree rules: levels of direct and of diagonal neighbours differ by at most one
 *   PAPER.md:51           boundary cells carry the boundary conditions (ghost states)
 *   PAPER.md:145-163,179  per-cell 5x5 system from the moments of f (here: Newton for the discrete Maxwellian)
 *   PAPER.md:231          BGK relaxation  -(f - f_eq)/tau
 *   PAPER.md:81, 207      per-cell kinetic/fluid flag; Maxwellian of the fluid cell at kinetic/fluid faces
 *
 * One step, for every KINETIC leaf j and velocity node i (readings in DESIGN.md):
 *   f*   = f - dt sum_F (A_F/V_j) (xi_i . n_F) f_up          f_up = own value if xi.n > 0, else across F
 *   rho  = w sum_i (1, xi, |xi|^2) f*                        (fp64 accumulation for either storage type)
 *   M    = exp(alpha . (1, xi, |xi|^2)),  w sum_i m M = rho  (discrete Maxwellian, Newton)
 *   f'   = f* + dt nu (M - f*),  nu = nu_prefactor * n * T^(1-visc_exp) / kn
 *
 * Conventions.  Every function returns a status code (0 = OK, negative = error); nothing throws,
 * exits or prints.  "host" / "device" is stated per pointer.  All device work is enqueued on the
 * CUDA stream given at creation and the calls do not synchronise unless stated; errors of
 * asynchronous work (including UFS_DVM_ENEWTON) surface at ufs_dvm_sync, ufs_dvm_destroy or, if
 * already known, at the next call.  The library never allocates f: the two f buffers, the moments
 * buffer and the stream belong to the caller (PyTorch tensors in the Python binding).
 */
#ifndef UFS_DVM_H
#define UFS_DVM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ufs_dvm_s *ufs_dvm_t; /* opaque handle, owned by the library */

enum { UFS_DVM_OK = 0,
       UFS_DVM_EINVAL = -1,  /* bad argument, unsupported velocity grid, host-only handle used for device work */
       UFS_DVM_EMESH = -2,   /* leaves do not tile the cube, overlap, or violate 2:1 balance (faces or diagonals) */
       UFS_DVM_ECUDA = -3,   /* a CUDA call failed; see ufs_dvm_last_error */
       UFS_DVM_ENOMEM = -4,
       UFS_DVM_ENEWTON = -5  /* some cell's Newton solve did not converge (or had n <= 0 or T <= 0) */ };
enum { UFS_BC_PERIODIC = 0, UFS_BC_SPECULAR = 1, UFS_BC_INFLOW = 2, UFS_BC_OUTFLOW = 3 };
enum { UFS_CELL_KINETIC = 0, UFS_CELL_FLUID = 1, UFS_CELL_SOLID = 2 }; /* SOLID: removed, specular at its faces */
enum { UFS_STORE_F64 = 0, UFS_STORE_F32 = 1 };
/* kinds in the boundary-face list */
enum { UFS_BF_SPECULAR = 1, UFS_BF_INFLOW = 2, UFS_BF_OUTFLOW = 3, UFS_BF_SOLID = 4, UFS_BF_FLUID = 5 };

/* Problem statement.  All arrays are HOST memory, caller-owned, read during create only. */
typedef struct {
    int64_t n_leaves;
    const uint8_t *level;        /* [n]    octree level of each leaf (edge h = domain_len / 2^level), <= 18 */
    const uint32_t *ijk;         /* [n][3] integer coordinates of the leaf at its own level                 */
    const uint8_t *kind;         /* [n]    UFS_CELL_*                                                       */
    double domain_len;           /* cube edge L                                                             */
    int32_t bc[6];               /* UFS_BC_* for the sides -x,+x,-y,+y,-z,+z (periodic must be set on both) */
    double inflow[6][5];         /* (n,ux,uy,uz,T) of the Maxwellian entering through INFLOW sides          */
    const double *fluid_moments; /* [n][5] (n,ux,uy,uz,T); read for FLUID leaves only; NULL if there are none */
    int32_t nv[3];               /* velocity nodes per axis; node k: xi = vmin + (k+1/2)(vmax-vmin)/nv      */
    double vmin[3], vmax[3];
    double kn;                   /* Knudsen number; +inf switches collisions off                            */
    double visc_exp;             /* omega in nu ~ T^(1-omega); 0.5 = hard spheres                           */
    double nu_prefactor;         /* c_nu                                                                     */
    int32_t storage;             /* UFS_STORE_*: element type of the f buffers                              */
} ufs_dvm_desc;

/* Flatten the mesh (Morton order, face lists, per-cell upwind gather records, ghost tables), upload it,
 * and bind the two caller-owned DEVICE buffers f_dev[0], f_dev[1], each n_kinetic * Nv elements of the
 * storage type, 16-byte aligned, and the CUDA stream (cudaStream_t cast to void*; NULL = default stream).
 * The buffers are recorded, not read: before the first step the caller fills f_dev[0] with f at t = 0 in
 * the library's layout, slab s = leaf cell_of_slab[s], slot t = velocity node vel_of_slot[t]
 * (ufs_dvm_layout).  Validates the tree (EMESH) and the grid (EINVAL: specular sides and SOLID leaves
 * need vmin = -vmax on the wall-normal axis; where only the one-CTA-per-cell kernels apply, Nv * sizeof(element)
 * must fit their on-chip slab buffer). */
int ufs_dvm_create(const ufs_dvm_desc *desc, void *f_dev[2], void *cuda_stream, ufs_dvm_t *out);

/* Same flattening and validation without touching CUDA: the handle answers ufs_dvm_layout,
 * ufs_dvm_faces, ufs_dvm_boundary_faces and ufs_dvm_destroy; device calls return EINVAL. */
int ufs_dvm_create_host(const ufs_dvm_desc *desc, ufs_dvm_t *out);

/* Enqueue nsteps explicit steps of size dt (transport -> moments -> discrete Maxwellian -> BGK relaxation).
 * f ping-pongs between the two buffers.  A step is two launches: k_prep (per cell: the moments of f* from the carried
 * velocity sums, Newton for the discrete Maxwellian) and the streaming pass that reads f once and writes f once
 * (k_tiles where the velocity grid has 12 positive nodes on x and whole 48-row blocks, e.g. 24^3; else k_rows,
 * k_stream, or the one-CTA-per-cell kernels, which need no k_prep); one more pass (the velocity sums of f) before
 * the first step and after ufs_dvm_f_changed.  The environment variable UFS_DVM_KERNEL = rows | stream | cell (read at
 * creation) forces the later kernels of that list (A/B timing, tests of the fallbacks).
 * Every wait inside the persistent kernels has a wall-clock watchdog (2 s without progress): a protocol bug or a faulted
 * copy ends the kernel with a trap, reported as UFS_DVM_ECUDA by ufs_dvm_sync (the CUDA context is then lost, as after
 * any device fault), never a hung GPU.  UFS_DVM_TEST_STALL (read at creation) makes k_tiles withhold one barrier arrival on
 * purpose so that tests can see exactly that. */
int ufs_dvm_step(ufs_dvm_t h, double dt, int nsteps);

/* Enqueue the moments of the current f: mom_dev is DEVICE memory, [5][n_kinetic] doubles in slab order:
 * n, n*ux, n*uy, n*uz, E = (w/2) sum |xi|^2 f  (PAPER.md:237 for the first two). */
int ufs_dvm_moments(ufs_dvm_t h, double *mom_dev);

/* The same moments of ANY f in this handle's layout, without allocating anything: for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops).  f_dev: DEVICE, [n_kinetic][Nv] elements of the storage type in slab
 * and slot order (NULL = the current f); mom_dev: DEVICE, [5][n_kinetic] doubles as above; both caller-owned.  The 35
 * velocity sums per cell that ufs_dvm_moments keeps in a cudaMalloc'ed buffer go, here, through a fixed array in the
 * library's device image: UFS_DVM_STATIC_MAX_CELLS * 36 doubles = 2.25 MiB, held by every device that loads the library
 * until the process exits.  More than UFS_DVM_STATIC_MAX_CELLS kinetic cells, a handle whose device is not the current
 * device, or a velocity grid without the octant layout (odd or asymmetric): UFS_DVM_EINVAL with the reason in
 * ufs_dvm_last_error, nothing enqueued.  Calls no cudaMalloc / cudaFree and no allocating library routine; two launches on
 * the handle's stream.  All calls on one device share the array (it keeps the last call's sums; nothing in it has to start
 * at zero: every number read is written first by the same call), so calls that OVERLAP on the GPU -- handles on different
 * streams -- race; calls on one stream are ordered.  The carried sums of the step are neither read nor changed. */
#define UFS_DVM_STATIC_MAX_CELLS 8192
int ufs_dvm_moments_static(ufs_dvm_t h, const void *f_dev, double *mom_dev);

/* Wait for the stream and report sticky asynchronous errors (ECUDA, ENEWTON). */
int ufs_dvm_sync(ufs_dvm_t h);

/* Frees everything the library built (host and device).  The f buffers are not touched. */
int ufs_dvm_destroy(ufs_dvm_t h);

/* 0 or 1: which of f_dev[] holds the current f. */
int ufs_dvm_current(ufs_dvm_t h);

/* Tell the library that the caller has (re)written the current f buffer on the device.  The streaming step keeps,
 * per cell, 35 velocity sums of the current f (the moments of Eq. 2's upwind fluxes, that the next
 * step's Maxwellian needs) from one step to the next; after this call they are recomputed from f by one extra
 * pass at the next ufs_dvm_step / ufs_dvm_moments.  Not needed after ufs_dvm_create (nothing is cached yet) nor
 * with ufs_dvm_run_host (it does this itself).  Host-side flag only; returns UFS_DVM_OK.
 * A caller that rewrites f and forgets this call gets Maxwellians from stale sums.  Check mode guards against it: with the
 * environment variable UFS_DVM_CHECK set at creation, every ufs_dvm_step call first re-sums eight pseudo-random cells of
 * the current f on the device and compares them with the carried sums; a mismatch makes the next ufs_dvm_sync return
 * UFS_DVM_EINVAL (sixteen small launches per call: for debugging, not for timing). */
int ufs_dvm_f_changed(ufs_dvm_t h);

/* Layout of the f buffers (HOST outputs, any may be NULL): *n_kinetic; cell_of_slab[n_kinetic] = index into
 * the caller's leaf list; vel_of_slot[Nv] = canonical velocity index (kz*nv[1] + ky)*nv[0] + kx stored at
 * each slab slot.  Slabs are in Morton order, slots grouped by velocity octant. */
int ufs_dvm_layout(ufs_dvm_t h, int64_t *n_kinetic, int64_t *cell_of_slab, int32_t *vel_of_slot);

/* Interior faces between two non-SOLID leaves (HOST outputs; pass NULL arrays to get the count):
 * owner = leaf on the low side, neigh = leaf on the high side (leaf-list indices), area = min(h)^2,
 * axis 0/1/2, ratio = level(neigh) - level(owner) in {-1,0,+1}.  Sorted by (Morton rank of owner, axis). */
int ufs_dvm_faces(ufs_dvm_t h, int64_t *n_faces, int64_t *owner, int64_t *neigh, double *area,
                  int8_t *axis, int8_t *ratio);

/* Boundary faces of non-SOLID leaves (HOST outputs; NULL arrays for the count): cell (leaf-list index),
 * axis, side (0 = low, 1 = high), area, kind UFS_BF_*, state = domain side 0..5 for SPECULAR / INFLOW /
 * OUTFLOW, the SOLID or FLUID leaf's index otherwise. */
int ufs_dvm_boundary_faces(ufs_dvm_t h, int64_t *n_faces, int64_t *cell, int8_t *axis, int8_t *side,
                           double *area, int8_t *kind, int64_t *state);

/* End-to-end convenience with HOST buffers (pinned or pageable): copy f_host_in (n_kinetic*Nv elements of
 * the storage type, library layout) to the current device buffer, run nsteps, compute the moments into
 * mom_dev_scratch (DEVICE, [5][n_kinetic]) and copy them to mom_host ([5][n_kinetic] doubles); if
 * f_host_out is not NULL also copy the final f back.  Synchronises the stream before returning. */
int ufs_dvm_run_host(ufs_dvm_t h, const void *f_host_in, void *f_host_out, double *mom_dev_scratch,
                     double *mom_host, double dt, int nsteps);

/* Mesh change on the device (the arrays of f and of the stencil records "are redone each time the
 * spatial mesh is changed"; PAPER.md:199 names host preparation and transfer as the bottleneck).  Creates the handle of
 * the new mesh exactly like ufs_dvm_create (new_desc, f_new_dev[2], cuda_stream, *out: same meaning, same errors) and
 * fills f_new_dev[0] from the old handle's current f without leaving the device: an unchanged leaf keeps its f, a leaf
 * created by refinement takes the f of the old leaf that covers it, a leaf created by coarsening the volume-weighted
 * mean of the old leaves inside it (the volume average of the old piecewise-constant field: conservative, first
 * order like the scheme), and a KINETIC leaf over an old FLUID leaf the Maxwellian of that leaf's frozen moments
 * (PAPER.md:207).  Any refinement depth; velocity grid and storage type must not change (EINVAL); a new KINETIC leaf
 * over an old SOLID leaf is EINVAL.  f_new_dev[0] must differ from the old handle's current buffer; f_new_dev[1] may
 * be any buffer of the right size, e.g. the old handle's other one if it is large enough.  counts (HOST, may be
 * NULL): new kinetic leaves copied / refined / coarsened, and sources that were FLUID leaves.  Synchronises the
 * stream before returning; the old handle stays valid (destroy it when done).  On error *out may hold a handle whose
 * ufs_dvm_last_error explains; destroy it. */
int ufs_dvm_remesh(ufs_dvm_t old_handle, const ufs_dvm_desc *new_desc, void *f_new_dev[2], void *cuda_stream,
                   ufs_dvm_t *out, int64_t counts[4]);

/* The map ufs_dvm_remesh applies, for two existing handles (host-only handles will do; HOST outputs, NULL arrays for
 * the sizes): new slab s = sum over k in [off[s], off[s+1]) of wgt[k] * source src[k], a source being slab src[k] of
 * the old mesh if src[k] >= 0, else the frozen Maxwellian of the old FLUID leaf ghost_leaf[-1 - src[k]].
 * off has n_kinetic(new) + 1 entries.  Errors are reported on new_handle. */
int ufs_dvm_remap_plan(ufs_dvm_t old_handle, ufs_dvm_t new_handle, int64_t *n_entries, int64_t *off, int32_t *src,
                       double *wgt, int64_t *n_ghosts, int64_t *ghost_leaf);

/* ---- Partitioned mesh: one GPU (process) per rank (PAPER.md:57 space-filling-curve partition, Fig. 3; PAPER.md:185-187
 * multi-GPU advection, Fig. 5: "inner cells are stored before ghost cells", ghost cells gathered before the kernel runs;
 * the collision part is local).
 *
 * ufs_dvm_partition: rank_of_leaf[n_leaves] (HOST output).  The leaves in N-order (Morton), each weighted by its cost
 * (w_kinetic for KINETIC, w_fluid for FLUID, 0 for SOLID leaves; "weight proportional to the CPU time"),
 * are cut into n_ranks consecutive ranges of equal weight: every rank's weight is within one leaf's weight of the mean.
 * No handle, no CUDA. */
int ufs_dvm_partition(const ufs_dvm_desc *desc, int32_t n_ranks, double w_kinetic, double w_fluid,
                      int32_t *rank_of_leaf);

/* Rank my_rank's part of the WHOLE mesh `desc` (every rank passes the same desc and rank_of_leaf, HOST arrays read during
 * the call only; any ownership whose KINETIC leaves form one N-order range per rank is accepted, EINVAL otherwise).  The
 * handle steps the rank's own ("inner") KINETIC leaves; its slabs are the inner leaves in N-order followed by the ghost
 * cells: KINETIC leaves of other ranks that are upwind sources of inner leaves.  f_dev[0], f_dev[1]: DEVICE buffers of
 * (n_inner + n_ghost) * Nv elements (sizes: ufs_dvm_part_layout of the host-only variant); the caller fills the inner
 * slabs of f_dev[0] (ufs_dvm_layout gives leaf and slot order), the ghost slabs arrive by the exchange below.
 * Per step:   for every peer p:  ufs_dvm_halo_pack(h, p, send_p)  ->  transfer send_p to rank p's recv buffer for this
 * rank (ncclSend / ncclRecv on the handle's stream, or any copy)  ->  ufs_dvm_halo_unpack(h, p, recv_p);   then
 * ufs_dvm_halo_done(h);  ufs_dvm_step(h, dt, 1).   A step without fresh ghosts, or nsteps > 1, is EINVAL.  Needs the
 * octant layout (even, symmetric velocity grid).  ufs_dvm_moments / ufs_dvm_layout describe the inner leaves only;
 * ufs_dvm_run_host, ufs_dvm_remesh and ufs_dvm_remap_plan refuse a partitioned handle. */
int ufs_dvm_create_part(const ufs_dvm_desc *desc, const int32_t *rank_of_leaf, int32_t my_rank, int32_t n_ranks,
                        void *f_dev[2], void *cuda_stream, ufs_dvm_t *out);
int ufs_dvm_create_part_host(const ufs_dvm_desc *desc, const int32_t *rank_of_leaf, int32_t my_rank,
                             int32_t n_ranks, ufs_dvm_t *out);

/* Slab layout of a partitioned handle (HOST outputs, any may be NULL): *n_inner, *n_ghost, *first_global_slab (inner slab
 * s is slab first_global_slab + s of the unpartitioned mesh), leaf_of_slab[n_inner + n_ghost] (leaf-list indices),
 * owner_of_ghost[n_ghost].  For an unpartitioned handle n_ghost = 0. */
int ufs_dvm_part_layout(ufs_dvm_t h, int64_t *n_inner, int64_t *n_ghost, int64_t *first_global_slab,
                        int64_t *leaf_of_slab, int32_t *owner_of_ghost);

/* Halo lists towards rank `peer` (HOST outputs; NULL arrays for the counts): send_slab[n_send] inner slabs and
 * send_mask[n_send] which of their 8 octant chunks (bit o: sign group o = sx + 2 sy + 4 sz, bit set if xi > 0) the peer
 * needs; recv_slab[n_recv] ghost slabs and recv_mask[n_recv] the chunks that arrive from the peer.  Both lists ascend in
 * the cell's slab number in the unpartitioned mesh, so the k-th entry sent is the k-th entry the peer receives.  Only the
 * upwind chunks cross: for a face on axis a the four sign groups whose xi_a points from the ghost into the inner cell
 * (PAPER.md:106-108). */
int ufs_dvm_halo(ufs_dvm_t h, int32_t peer, int64_t *n_send, int32_t *send_slab, uint8_t *send_mask,
                 int64_t *n_recv, int32_t *recv_slab, uint8_t *recv_mask);

/* Sizes in bytes of the packed buffers exchanged with `peer` (HOST outputs): listed chunks x chunk size, then 36 doubles per
 * listed cell (its carried velocity sums; none with the one-CTA-per-cell kernels, which carry no sums). */
int ufs_dvm_halo_bytes(ufs_dvm_t h, int32_t peer, int64_t *send_bytes, int64_t *recv_bytes);

/* Enqueue: gather the chunks of the send list of `peer` from the current f into buf_dev (DEVICE, 16-byte aligned,
 * send_bytes), entries in list order, a slab's chunks by ascending octant, and behind them the listed cells' carried sums
 * (formed first if f has not been summed yet) / scatter buf_dev (recv_bytes) into the ghost slabs of the current f and the
 * ghost rows of its sums.  The ghost rows thus hold the OWNER's sums, and a partitioned run is bit-identical to the
 * one-domain run. */
int ufs_dvm_halo_pack(ufs_dvm_t h, int32_t peer, void *buf_dev);
int ufs_dvm_halo_unpack(ufs_dvm_t h, int32_t peer, const void *buf_dev);

/* Every peer's chunks have been unpacked (enqueued on the handle's stream), or pushed by the peers' step kernels (below):
 * allow the next ufs_dvm_step.  Where the ghost cells' sums did not arrive with their f (fused exchange set up without
 * peer_sums) they are formed here from the ghost slabs, one pass of the sums kernel over them. */
int ufs_dvm_halo_done(ufs_dvm_t h);

/* Fused ghost exchange: step and exchange in ONE kernel over peer memory (PAPER.md:185-187 does the exchange as separate
 * MPI messages between GPUs; with NVLink / NVSwitch peer access the step kernel can write into the neighbour directly).
 * After this call every ufs_dvm_step of this handle stores each row of a cell that some peer lists as a ghost cell twice:
 * into the own next f, and -- for the octants that peer needs -- into that peer's ghost slab of ITS next f, while the rest
 * of the pass goes on; ufs_dvm_halo_pack / unpack and the transfer between them are then not needed.
 * Arrays of n_ranks entries (HOST, read during the call), entries of ranks that need nothing from this rank are ignored:
 * peer_f0[p], peer_f1[p] = rank p's f_dev[0], f_dev[1] as THIS device reaches them (the same process: the pointers
 * themselves after cudaDeviceEnablePeerAccess; another process: the mappings of cudaIpcOpenMemHandle or of a symmetric
 * allocation), 16-byte aligned; dest_slab[p][i] = the ghost slab of rank p that holds this rank's i-th send slab, i.e. rank
 * p's recv_slab list for this rank (ufs_dvm_halo on rank p), n_send entries.
 * Protocol.  All ranks hold the same ufs_dvm_current (true from creation on; every rank steps once per round).  The first
 * step still needs one ordinary exchange (pack / transfer / unpack / ufs_dvm_halo_done): nothing has been pushed yet.  From
 * then on, per step:  ufs_dvm_step(h, dt, 1) on every rank  ->  a barrier ACROSS the ranks' streams (every rank's step kernel
 * has finished: its ghost slabs are complete, and nobody still reads the buffers the next step will push into)  ->
 * ufs_dvm_halo_done(h) (ghost sums)  ->  next step.  Double buffering makes that one barrier per step enough.
 * peer_sums0 / peer_sums1 (both or neither; arrays of n_ranks entries like peer_f0): rank p's two arrays of carried velocity
 * sums (ufs_dvm_sums_dev on rank p).  With them the step kernel also writes the 36 sums of every pushed cell into the
 * peer's ghost row, ufs_dvm_halo_done has no pass over the ghost slabs left to launch, and -- the ghost rows now holding the
 * owner's own carried sums, not a re-summation -- the partitioned run is bit-identical to the one-domain run.  Every rank
 * must then be set up the same way.  NULL: ufs_dvm_halo_done sums the ghost slabs as after an ordinary exchange.
 * EINVAL: not a partitioned handle, not the tile kernel, a needed entry is NULL or misaligned, or some cell is needed by
 * more than four peers (then the pack / unpack exchange serves).  May be called again (new peer addresses). */
int ufs_dvm_halo_push_setup(ufs_dvm_t h, void *const *peer_f0, void *const *peer_f1, const int32_t *const *dest_slab,
                            void *const *peer_sums0, void *const *peer_sums1);

/* DEVICE addresses of the handle's two arrays of carried velocity sums ([n_inner + n_ghost][36] doubles, library-owned,
 * valid until ufs_dvm_destroy): what a peer passes as peer_sums0 / peer_sums1 above (the same process: the pointers
 * themselves with peer access enabled; another process: their cudaIpcOpenMemHandle mappings). */
int ufs_dvm_sums_dev(ufs_dvm_t h, void **sums0, void **sums1);

/* Make the handle keep its carried sums in two CALLER-owned DEVICE arrays, each (n_inner + n_ghost) * 36 doubles, 16-byte
 * aligned, instead of its own allocations (whose contents are copied over; the call synchronises the stream).  For ranks in
 * different processes: arrays from a symmetric allocation are mapped into every peer by the allocator's rendezvous, which
 * the library's own cudaMalloc'ed arrays are not; the peers' mappings are then the peer_sums0 / peer_sums1 of
 * ufs_dvm_halo_push_setup.  The arrays must outlive the handle; ufs_dvm_destroy does not free them. */
int ufs_dvm_sums_use(ufs_dvm_t h, void *sums0, void *sums1);

/* The push entries that ufs_dvm_halo_push_setup built (it also accepts a host-only handle: the records are built, nothing
 * is uploaded; the addresses are then just numbers), in the order the kernel reads them (HOST outputs, any may be NULL):
 * *n_entries, *n_push_tiles (the tiles with entries: the first ones of ufs_dvm_tiles); per entry: slab = the inner slab whose
 * rows are pushed, mask = the octants pushed, dst0 / dst1 = address of the peer's ghost slab in its f buffer 0 / 1,
 * sums0 / sums1 = address of that ghost cell's row in the peer's sums array 0 / 1 (0 if the sums are not pushed). */
int ufs_dvm_push_entries(ufs_dvm_t h, int64_t *n_entries, int64_t *n_push_tiles, int32_t *slab, uint8_t *mask, uint64_t *dst0,
                         uint64_t *dst1, uint64_t *sums0, uint64_t *sums1);

/* The tile records the flattener built for k_tiles (HOST outputs, any may be NULL; all empty for other kernels):
 * *n_tiles, *pmax (stride of the piece lists); hdr[n_tiles][8] int32 = {first slab, cells, pieces per octant (8 bytes),
 * level per cell (8 bytes), first push entry, eight 4-bit push counts (0, 0 without ufs_dvm_halo_push_setup)}; pieces[n_tiles][8][pmax] = source chunk codes: bits 0..29 = index * 8 + octant, the
 * index being a slab, or an inflow ghost table if bit 31 is set, or a fluid ghost if bit 30 is set (the frozen Maxwellian
 * of a FLUID leaf: nothing is copied, the kernel's producer warps write the leaf's separable factors into
 * the slot); cellidx[n_tiles][8][8][16] bytes = per octant and cell: [0] own piece, [1] flags (bit a: axis a has four
 * finer sources, bit 3: some source is a fluid ghost), [2..3] little-endian mask, bit 4a + k: source k on axis a is a fluid
 * ghost, [4 + 4a + k] piece of source k on axis a (0xFF unused); fluid_leaf[*n_fluid_ghosts] = leaf of each fluid ghost.
 * First-order form of the per-cell, per-sign-group stencil records of PAPER.md:113-115, deduplicated per tile. */
int ufs_dvm_tiles(ufs_dvm_t h, int64_t *n_tiles, int32_t *pmax, int32_t *hdr, uint32_t *pieces, uint8_t *cellidx,
                  int64_t *n_fluid_ghosts, int64_t *fluid_leaf);

/* Number of kernels this handle has launched so far (step + moments kernels). */
int64_t ufs_dvm_launch_count(ufs_dvm_t h);

/* Measurement aid.  ufs_dvm_profile(h, 1) makes the following steps (at most 64) bracket their main kernel -- the
 * streaming pass that reads and writes f -- with CUDA events on the handle's stream; ufs_dvm_profile(h, 0) stops.
 * ufs_dvm_kernel_ms synchronises the stream and returns (HOST outputs) the mean duration in ms of those launches
 * and their number.  The small per-cell Newton kernel that precedes the pass is not inside the bracket. */
int ufs_dvm_profile(ufs_dvm_t h, int enable);
int ufs_dvm_kernel_ms(ufs_dvm_t h, double *mean_ms, int32_t *n_launches);

/* Launch geometry of the step kernel: threads per CTA, dynamic shared memory per CTA, vector width in
 * elements, and 1 if the octant fast path is used (0 = generic per-slot path).  HOST outputs. */
int ufs_dvm_kernel_info(ufs_dvm_t h, int32_t *threads, int32_t *smem_bytes, int32_t *vec, int32_t *fast);

/* Name of the streaming kernel this handle launches: "k_tiles" (persistent, tiles of up to eight slabs share their
 * upwind chunks on chip), "k_rows" / "k_stream" (persistent, one cell at a time), "k_step_fast" (one CTA per cell,
 * octant layout) or "k_step_generic" (any velocity grid).  Never NULL. */
const char *ufs_dvm_kernel_name(ufs_dvm_t h);

/* Message of the last error on this handle (valid until the next call on it); never NULL. */
const char *ufs_dvm_last_error(ufs_dvm_t h);

#ifdef __cplusplus
}
#endif
#endif /* UFS_DVM_H */
