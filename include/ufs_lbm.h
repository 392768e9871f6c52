/*
 * ufs_lbm.h -- C ABI of the lattice-Boltzmann variant of the B200-native kinetic step (same library, libufs_dvm.so).
 *
 * "The LBM Module in UFS is designed as a subset of the DVM kinetic solvers" (arxiv 1503.00707): the
 * velocity nodes are those of a 3x3x3 Cartesian velocity grid with nodes -1, 0, 1 (lattice units, c_s^2 = 1/3): D3Q27,
 * or D3Q19 (|c|^2 <= 2).  One step, for every leaf j of the octree that is not SOLID and every lattice velocity c_i:
 *
 *   f*   = f - dt sum_F (A_F/V_j) (c_i . n_F) f_up     the finite-volume transport of the DVM step (Eq. 2, PAPER.md:103;
 *                                                      "finite volume LBM"; neighbour sums "from 6 to 6x4",
 *                                                      PAPER.md:251), first-order upwind, 2:1 faces as four sub-faces
 *   rho  = sum_i f*_i,   rho u = sum_i c_i f*_i
 *   f_eq = w_i rho (1 + c_i.u/cs^2 + (c_i.u)^2/(2 cs^4) - u^2/(2 cs^2))
 *   f'   = f* + (dt/tau) (f_eq - f*)                   BGK term -(f - f_eq)/tau, forward Euler
 *
 * Ghost states: periodic wrap; SPECULAR walls and SOLID leaves mirror the wall-normal lattice component;
 * OUTFLOW is zero-gradient; INFLOW is the equilibrium of the side's (rho, u).
 * Mapping: one thread per cell and f stored velocity-major, f[i][cell] (the paper's one-warp-per-cell grouping,
 * PAPER.md:251, was made for Fermi / Kepler; csrc/lbm.cu says what it costs on sm_100a).
 *
 * Conventions as in ufs_dvm.h: status codes (UFS_DVM_*), no exceptions, "host" / "device" per pointer, device work is
 * enqueued on the stream given at creation, asynchronous errors surface at ufs_lbm_sync.  The two f buffers and the
 * moments buffer belong to the caller.
 */
#ifndef UFS_LBM_H
#define UFS_LBM_H

#include <stdint.h>

#include "ufs_dvm.h" /* status codes, UFS_BC_*, UFS_CELL_*, UFS_STORE_* */

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ufs_lbm_s *ufs_lbm_t; /* opaque handle, owned by the library */

/* Problem statement.  All arrays are HOST memory, caller-owned, read during create only. */
typedef struct {
    int64_t n_leaves;
    const uint8_t *level;  /* [n]    octree level of each leaf (edge h = domain_len / 2^level)                 */
    const uint32_t *ijk;   /* [n][3] integer coordinates of the leaf at its own level                          */
    const uint8_t *kind;   /* [n]    UFS_CELL_KINETIC (a fluid cell of the LBM) or UFS_CELL_SOLID; no FLUID     */
    double domain_len;     /* cube edge, in lattice length units (dt in lattice time units: c = 1 crosses h in h) */
    int32_t bc[6];         /* UFS_BC_* for the sides -x,+x,-y,+y,-z,+z                                          */
    double inflow[6][4];   /* (rho, ux, uy, uz) of the equilibrium entering through INFLOW sides               */
    int32_t lattice;       /* 19 or 27                                                                         */
    double tau;            /* relaxation time; +inf switches the collision off                                 */
    int32_t storage;       /* UFS_STORE_F64 or UFS_STORE_F32: element type of the f buffers                    */
} ufs_lbm_desc;

/* Flatten the mesh (N-order, per-cell upwind gather records: the same flattener as ufs_dvm_create), upload it, and bind
 * the two caller-owned DEVICE buffers f_dev[0], f_dev[1], each Q * n_cells elements of the storage type, 16-byte aligned,
 * and the CUDA stream.  Before the first step the caller fills f_dev[0], velocity-major: element [i * n_cells + r] is
 * population i (lattice velocity c[i]) of leaf cell_of_row[r] (ufs_lbm_layout).  EMESH / EINVAL as ufs_dvm_create; FLUID leaves and lattices other than 19 / 27: EINVAL. */
int ufs_lbm_create(const ufs_lbm_desc *desc, void *f_dev[2], void *cuda_stream, ufs_lbm_t *out);

/* Same flattening and validation without CUDA: answers ufs_lbm_layout and ufs_lbm_destroy. */
int ufs_lbm_create_host(const ufs_lbm_desc *desc, ufs_lbm_t *out);

/* Enqueue nsteps steps of size dt (transport -> moments -> equilibrium -> relaxation), one kernel launch per step;
 * f ping-pongs between the two buffers.  dt * (|cx|+|cy|+|cz|) / h_min <= 1 keeps every coefficient non-negative. */
int ufs_lbm_step(ufs_lbm_t h, double dt, int nsteps);

/* Enqueue the moments of the current f: mom_dev is DEVICE memory, [4][n_cells] doubles in row order: rho, rho ux,
 * rho uy, rho uz. */
int ufs_lbm_moments(ufs_lbm_t h, double *mom_dev);

/* Wait for the stream and report sticky asynchronous errors. */
int ufs_lbm_sync(ufs_lbm_t h);

/* Frees everything the library built.  The f buffers are not touched. */
int ufs_lbm_destroy(ufs_lbm_t h);

/* 0 or 1: which of f_dev[] holds the current f. */
int ufs_lbm_current(ufs_lbm_t h);

/* Layout (HOST outputs, any may be NULL): *n_cells (non-SOLID leaves), cell_of_row[n_cells] = index into the caller's leaf
 * list (cells are in N-order), *q, c[q][3] the lattice velocities in population order (ascending (kz*3+ky)*3+kx
 * with c = k - 1), w[q] their weights. */
int ufs_lbm_layout(ufs_lbm_t h, int64_t *n_cells, int64_t *cell_of_row, int32_t *q, int8_t *c, double *w);

/* Number of kernels this handle has launched so far. */
int64_t ufs_lbm_launch_count(ufs_lbm_t h);

/* Message of the last error on this handle; never NULL. */
const char *ufs_lbm_last_error(ufs_lbm_t h);

#ifdef __cplusplus
}
#endif
#endif /* UFS_LBM_H */
