/*
 * dvm_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU statement of one explicit DVM
 * time step of the UFS kinetic module (arxiv 1503.00707), written from the paper.  It exists to
 * check the CUDA path; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code, header, table or constant with
 * paper_1503_00707_b200/csrc and never imports it.
 *
 * What is computed, one cell j and one velocity i at a time:
 *   S1  velocity nodes at the centres of a uniform Cartesian velocity grid
 *   S2  f*_ij = f_ij - dt * sum_F (A_F/V_j) (xi_i . n_F) f^up_{F,i}                 PAPER.md:103 (Eq. 2),
 *       first-order upwind finite-volume form over all faces / sub-faces F of leaf j (reading G2, G3, G4)
 *   S3  f^up = own value if xi.n > 0, value across the face if xi.n < 0, nothing if = 0
 *       value across: neighbour leaf's f_i, or a ghost state (boundary cells):
 *       specular wall / solid leaf: own f at the velocity mirrored in the wall normal;
 *       outflow: own f; inflow: Maxwellian of the inflow state; fluid leaf: Maxwellian of its
 *       given moments
 *   S4  rho_j = w sum_i m(xi_i) f*_ij,  m = (1, xi_x, xi_y, xi_z, |xi|^2)
 *   S5  discrete Maxwellian M_ij = exp(alpha_j . m(xi_i)) with w sum_i m M = rho_j, by Newton;
 *       each iteration solves a 5x5 system by Gauss elimination                    PAPER.md:145-163, 179 (reading G7, G8)
 *   S6  nu_j = c_nu n T^(1-omega) / Kn;  f^{n+1} = f* + dt nu (M - f*)             PAPER.md:231, 89 (reading G9)
 *   S7  reported moments = w sum_i m f, energy E = rho_4 / 2
 *
 * Neighbour search: own hash map (level,i,j,k) -> leaf; for each leaf and direction look up the
 * same-level key, else the parent-level key, else the 4 child keys on the shared side, with periodic
 * wrap where bc says so (tree rules: PAPER.md:45).
 *
 * Pins (tests/test_oracle_pins.py): uniform Maxwellian steady state, mass/momentum/energy
 * telescoping, the closed form of 1-D free-molecular streaming, brute-force face enumeration,
 * refinement / axis-permutation symmetry, linearity, positivity, relaxation invariants, homogeneous
 * relaxation closed form, entropy, specular box.  Parity unpinned by the paper (conventions only):
 * nu constants (G9), CFL convention (G11), Sod x-ends (G16); see DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORA_BC_PERIODIC = 0, ORA_BC_SPECULAR = 1, ORA_BC_INFLOW = 2, ORA_BC_OUTFLOW = 3 };
enum { ORA_KINETIC = 0, ORA_FLUID = 1, ORA_SOLID = 2 };
enum { ORA_OK = 0, ORA_EINVAL = -1, ORA_EMESH = -2, ORA_ENOMEM = -4, ORA_ENEWTON = -5 };

typedef struct {
    int64_t n_leaves;
    const uint8_t *level;        /* [n] */
    const uint32_t *ijk;         /* [n][3] coordinates at the leaf's own level */
    const uint8_t *kind;         /* [n] */
    double domain_len;
    int32_t bc[6];               /* -x,+x,-y,+y,-z,+z */
    double inflow[6][5];         /* (n,ux,uy,uz,T) */
    const double *fluid_moments; /* [n][5] (n,ux,uy,uz,T), FLUID leaves only */
    int32_t nv[3];
    double vmin[3], vmax[3];
    double kn, visc_exp, nu_prefactor;
    int32_t window;              /* 1: the leaf list is a window of a larger mesh; a missing neighbour
                                    is replaced by a zero-gradient ghost and coverage is not checked */
} oracle_desc;

/* one entry of a leaf's neighbour table: what lies across one face or sub-face */
enum { NB_LEAF = 0, NB_BOUNDARY = 1, NB_MISSING = 2 };
typedef struct { int32_t type; int32_t side; int64_t id; double area; } nb_entry;

typedef struct {
    oracle_desc d;
    uint8_t *level, *kind; uint32_t *ijk; double *fluid; /* private copies */
    int64_t n_kin; int64_t *kin_leaf;  /* kinetic row -> leaf */
    int64_t *row_of_leaf;              /* leaf -> kinetic row or -1 */
    int64_t Nv; double *xi[3]; double w;
    /* hash map */
    uint64_t *hkey; int64_t *hval; uint64_t hmask;
    /* neighbour table: [leaf][6 dirs][4] */
    nb_entry *nb; int8_t *nb_count;    /* [leaf][6] number of entries (1 or 4) */
    double *inflow_f;                  /* [6][Nv] inflow Maxwellians */
    int newton_fail; int newton_max_iters;
    char err[256];
} oracle_t;

static uint64_t make_key(int level, uint32_t i, uint32_t j, uint32_t k) {
    return ((uint64_t)level << 57) | ((uint64_t)i << 38) | ((uint64_t)j << 19) | (uint64_t)k;
}
static uint64_t mix(uint64_t x) { x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33; return x; }

static int64_t find_leaf(const oracle_t *o, int level, int64_t i, int64_t j, int64_t k) {
    if (level < 0) return -1;
    int64_t n = (int64_t)1 << level;
    if (i < 0 || j < 0 || k < 0 || i >= n || j >= n || k >= n) return -1;
    uint64_t key = make_key(level, (uint32_t)i, (uint32_t)j, (uint32_t)k);
    uint64_t p = mix(key) & o->hmask;
    while (o->hval[p] >= 0) {
        if (o->hkey[p] == key) return o->hval[p];
        p = (p + 1) & o->hmask;
    }
    return -1;
}

/* pointwise Maxwellian n/(2 pi T)^{3/2} exp(-|xi-u|^2 / 2T): inflow state and fluid leaves (G13) */
static double maxwell_point(const double *prim, double x, double y, double z) {
    double n = prim[0], T = prim[4];
    double cx = x - prim[1], cy = y - prim[2], cz = z - prim[3];
    return n / pow(2.0 * M_PI * T, 1.5) * exp(-(cx * cx + cy * cy + cz * cz) / (2.0 * T));
}

void oracle_dvm_destroy(oracle_t *o) {
    if (!o) return;
    free(o->level); free(o->kind); free(o->ijk); free(o->fluid); free(o->kin_leaf); free(o->row_of_leaf);
    for (int a = 0; a < 3; a++) free(o->xi[a]);
    free(o->hkey); free(o->hval); free(o->nb); free(o->nb_count); free(o->inflow_f);
    free(o);
}

const char *oracle_dvm_error(const oracle_t *o) { return o ? o->err : "null handle"; }

static int build_neighbours(oracle_t *o) {
    const int64_t n = o->d.n_leaves;
    o->nb = (nb_entry *)calloc((size_t)n * 24, sizeof(nb_entry));
    o->nb_count = (int8_t *)calloc((size_t)n * 6, 1);
    if (!o->nb || !o->nb_count) return ORA_ENOMEM;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (int64_t j = 0; j < n; j++) {
        const int l = o->level[j];
        const int64_t nl = (int64_t)1 << l;
        const double h = o->d.domain_len / (double)nl;
        for (int dir = 0; dir < 6; dir++) {
            const int a = dir >> 1, s = (dir & 1) ? +1 : -1;
            nb_entry *e = o->nb + (j * 6 + dir) * 4;
            int64_t c[3] = {o->ijk[3 * j], o->ijk[3 * j + 1], o->ijk[3 * j + 2]};
            c[a] += s;
            if (c[a] < 0 || c[a] >= nl) {
                if (o->d.bc[dir] == ORA_BC_PERIODIC) {
                    c[a] = (c[a] + nl) % nl;
                } else {
                    e[0].type = NB_BOUNDARY; e[0].side = dir; e[0].id = -1; e[0].area = h * h;
                    o->nb_count[j * 6 + dir] = 1;
                    continue;
                }
            }
            int64_t q = find_leaf(o, l, c[0], c[1], c[2]);
            if (q >= 0) { /* same level: one face of area h^2 */
                e[0].type = NB_LEAF; e[0].id = q; e[0].area = h * h; e[0].side = dir;
                o->nb_count[j * 6 + dir] = 1;
                continue;
            }
            q = find_leaf(o, l - 1, c[0] >> 1, c[1] >> 1, c[2] >> 1);
            if (q >= 0) { /* coarser neighbour: the fine cell sees one face of area h_fine^2 (G3) */
                e[0].type = NB_LEAF; e[0].id = q; e[0].area = h * h; e[0].side = dir;
                o->nb_count[j * 6 + dir] = 1;
                continue;
            }
            /* finer neighbours: the 4 children of the same-level position that touch the shared face */
            int cnt = 0, miss = 0;
            const int b1 = (a + 1) % 3, b2 = (a + 2) % 3;
            for (int u = 0; u < 2; u++)
                for (int v = 0; v < 2; v++) {
                    int64_t cc[3];
                    cc[a] = 2 * c[a] + (s > 0 ? 0 : 1);
                    cc[b1] = 2 * c[b1] + u;
                    cc[b2] = 2 * c[b2] + v;
                    int64_t r = find_leaf(o, l + 1, cc[0], cc[1], cc[2]);
                    e[cnt].side = dir; e[cnt].area = 0.25 * h * h; /* sub-face (h/2)^2 */
                    if (r >= 0) { e[cnt].type = NB_LEAF; e[cnt].id = r; }
                    else { e[cnt].type = NB_MISSING; e[cnt].id = -1; miss++; }
                    cnt++;
                }
            if (miss == 4) { /* nothing there at all */
                e[0].type = NB_MISSING; e[0].id = -1; e[0].area = h * h; e[0].side = dir;
                o->nb_count[j * 6 + dir] = 1;
                if (!o->d.window) bad |= 1;
            } else {
                o->nb_count[j * 6 + dir] = 4;
                if (miss && !o->d.window) bad |= 1;
            }
        }
    }
    if (bad) { snprintf(o->err, sizeof o->err, "mesh: a face has no neighbour within one level (gap or 2:1 violation)"); return ORA_EMESH; }
    return ORA_OK;
}

int oracle_dvm_create(const oracle_desc *d, oracle_t **out) {
    if (!d || !out || d->n_leaves <= 0) return ORA_EINVAL;
    oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
    if (!o) return ORA_ENOMEM;
    *out = o;
    o->d = *d;
    const int64_t n = d->n_leaves;
    for (int a = 0; a < 3; a++)
        if (d->nv[a] <= 0 || !(d->vmax[a] > d->vmin[a])) { snprintf(o->err, sizeof o->err, "bad velocity grid"); return ORA_EINVAL; }
    o->level = (uint8_t *)malloc(n); o->kind = (uint8_t *)malloc(n); o->ijk = (uint32_t *)malloc(n * 12);
    memcpy(o->level, d->level, n); memcpy(o->kind, d->kind, n); memcpy(o->ijk, d->ijk, n * 12);
    if (d->fluid_moments) { o->fluid = (double *)malloc(n * 40); memcpy(o->fluid, d->fluid_moments, n * 40); }
    o->d.level = o->level; o->d.kind = o->kind; o->d.ijk = o->ijk; o->d.fluid_moments = o->fluid;
    /* S1: velocity nodes and the quadrature weight (midpoint rule, G10) */
    o->Nv = (int64_t)d->nv[0] * d->nv[1] * d->nv[2];
    o->w = 1.0;
    for (int a = 0; a < 3; a++) {
        double dv = (d->vmax[a] - d->vmin[a]) / d->nv[a];
        o->xi[a] = (double *)malloc(sizeof(double) * d->nv[a]);
        for (int k = 0; k < d->nv[a]; k++) o->xi[a][k] = d->vmin[a] + (k + 0.5) * dv;
        o->w *= dv;
    }
    /* kinetic rows in leaf-list order */
    o->row_of_leaf = (int64_t *)malloc(n * 8);
    o->kin_leaf = (int64_t *)malloc(n * 8);
    for (int64_t j = 0; j < n; j++) {
        if (o->kind[j] == ORA_KINETIC) { o->row_of_leaf[j] = o->n_kin; o->kin_leaf[o->n_kin++] = j; }
        else o->row_of_leaf[j] = -1;
        if (o->kind[j] == ORA_FLUID && !o->fluid) { snprintf(o->err, sizeof o->err, "FLUID leaf but fluid_moments is NULL"); return ORA_EINVAL; }
        if (o->level[j] > 18) { snprintf(o->err, sizeof o->err, "level > 18"); return ORA_EINVAL; }
    }
    /* hash map */
    uint64_t cap = 16; while (cap < (uint64_t)n * 2) cap <<= 1;
    o->hmask = cap - 1;
    o->hkey = (uint64_t *)malloc(cap * 8); o->hval = (int64_t *)malloc(cap * 8);
    if (!o->hkey || !o->hval) return ORA_ENOMEM;
    for (uint64_t p = 0; p < cap; p++) o->hval[p] = -1;
    double vol = 0.0;
    for (int64_t j = 0; j < n; j++) {
        int l = o->level[j]; uint32_t nl = 1u << l;
        if (o->ijk[3 * j] >= nl || o->ijk[3 * j + 1] >= nl || o->ijk[3 * j + 2] >= nl) { snprintf(o->err, sizeof o->err, "leaf %lld outside the cube", (long long)j); return ORA_EMESH; }
        uint64_t key = make_key(l, o->ijk[3 * j], o->ijk[3 * j + 1], o->ijk[3 * j + 2]);
        uint64_t p = mix(key) & o->hmask;
        while (o->hval[p] >= 0) {
            if (o->hkey[p] == key) { snprintf(o->err, sizeof o->err, "duplicate leaf %lld", (long long)j); return ORA_EMESH; }
            p = (p + 1) & o->hmask;
        }
        o->hkey[p] = key; o->hval[p] = j;
        vol += ldexp(1.0, -3 * l);
    }
    if (!d->window) {
        /* leaves must tile the cube: total volume 1 and no leaf below another leaf */
        if (vol != 1.0) { snprintf(o->err, sizeof o->err, "leaves do not tile the cube (volume %.17g)", vol); return ORA_EMESH; }
        for (int64_t j = 0; j < n; j++) {
            int64_t c[3] = {o->ijk[3 * j], o->ijk[3 * j + 1], o->ijk[3 * j + 2]};
            for (int l = o->level[j] - 1; l >= 0; l--) {
                c[0] >>= 1; c[1] >>= 1; c[2] >>= 1;
                if (find_leaf(o, l, c[0], c[1], c[2]) >= 0) { snprintf(o->err, sizeof o->err, "leaf %lld overlaps a coarser leaf", (long long)j); return ORA_EMESH; }
            }
        }
    }
    int rc = build_neighbours(o);
    if (rc) return rc;
    /* specular reflection mirrors the node index; it needs a symmetric grid on that axis (G12) */
    for (int a = 0; a < 3; a++) {
        int need = (d->bc[2 * a] == ORA_BC_SPECULAR || d->bc[2 * a + 1] == ORA_BC_SPECULAR);
        for (int64_t j = 0; j < n && !need; j++) if (o->kind[j] == ORA_SOLID) need = 1;
        if (need && fabs(d->vmin[a] + d->vmax[a]) > 1e-14 * fabs(d->vmax[a])) { snprintf(o->err, sizeof o->err, "specular wall needs vmin=-vmax on axis %d", a); return ORA_EINVAL; }
    }
    /* inflow ghost states (a1b): fixed Maxwellian of the inflow state at every node */
    o->inflow_f = (double *)calloc((size_t)6 * o->Nv, sizeof(double));
    for (int s = 0; s < 6; s++)
        if (d->bc[s] == ORA_BC_INFLOW)
            for (int kz = 0; kz < d->nv[2]; kz++) for (int ky = 0; ky < d->nv[1]; ky++) for (int kx = 0; kx < d->nv[0]; kx++)
                o->inflow_f[s * o->Nv + ((int64_t)kz * d->nv[1] + ky) * d->nv[0] + kx] = maxwell_point(d->inflow[s], o->xi[0][kx], o->xi[1][ky], o->xi[2][kz]);
    return ORA_OK;
}

int64_t oracle_dvm_n_kinetic(const oracle_t *o) { return o->n_kin; }
/* Replaces the ghost state of INFLOW side `side` by a caller-given table values[Nv] (canonical velocity order).  The
 * lattice-Boltzmann variant (oracle/lbm_oracle.py) puts its polynomial equilibrium there (the weights serve
 * "the equilibrium distribution function for initial and boundary conditions"); the arithmetic of S2/S3 is unchanged. */
int oracle_dvm_set_inflow_table(oracle_t *o, int side, const double *values) {
    if (!o || side < 0 || side >= 6 || !values) return -1;
    memcpy(o->inflow_f + (size_t)side * o->Nv, values, (size_t)o->Nv * sizeof(double));
    return 0;
}

void oracle_dvm_kinetic_leaves(const oracle_t *o, int64_t *leaf_of_row) { memcpy(leaf_of_row, o->kin_leaf, o->n_kin * 8); }

/* ---- S2 + S3 for one kinetic leaf: fstar[Nv] from f (all kinetic rows) ---- */
static void cell_transport(const oracle_t *o, const double *f, int64_t row, double dt, double *fstar) {
    const int64_t j = o->kin_leaf[row];
    const int nx = o->d.nv[0], ny = o->d.nv[1], nz = o->d.nv[2];
    const double h = o->d.domain_len / (double)((int64_t)1 << o->level[j]);
    const double V = h * h * h;
    const double *fj = f + row * o->Nv;
    for (int kz = 0; kz < nz; kz++) for (int ky = 0; ky < ny; ky++) for (int kx = 0; kx < nx; kx++) {
        const int64_t i = ((int64_t)kz * ny + ky) * nx + kx;
        const double xi[3] = {o->xi[0][kx], o->xi[1][ky], o->xi[2][kz]};
        const int kk[3] = {kx, ky, kz};
        double acc = 0.0;
        for (int dir = 0; dir < 6; dir++) {
            const int a = dir >> 1;
            const double xin = (dir & 1) ? xi[a] : -xi[a]; /* xi . n_F, n_F outward */
            if (xin == 0.0) continue;
            const nb_entry *e = o->nb + (j * 6 + dir) * 4;
            for (int t = 0; t < o->nb_count[j * 6 + dir]; t++) {
                double fup;
                if (xin > 0.0) {
                    fup = fj[i];
                } else {
                    int mirror = 0, bc = -1;
                    if (e[t].type == NB_LEAF) {
                        int kd = o->kind[e[t].id];
                        if (kd == ORA_KINETIC) fup = f[o->row_of_leaf[e[t].id] * o->Nv + i];
                        else if (kd == ORA_FLUID) fup = maxwell_point(o->fluid + 5 * e[t].id, xi[0], xi[1], xi[2]);
                        else { mirror = 1; fup = 0.0; }
                    } else if (e[t].type == NB_BOUNDARY) {
                        bc = o->d.bc[e[t].side];
                        if (bc == ORA_BC_SPECULAR) { mirror = 1; fup = 0.0; }
                        else if (bc == ORA_BC_INFLOW) fup = o->inflow_f[e[t].side * o->Nv + i];
                        else fup = fj[i]; /* outflow: zero gradient */
                    } else {
                        fup = fj[i]; /* window edge: zero gradient */
                    }
                    if (mirror) {
                        int km[3] = {kk[0], kk[1], kk[2]};
                        km[a] = o->d.nv[a] - 1 - kk[a];
                        fup = fj[((int64_t)km[2] * ny + km[1]) * nx + km[0]];
                    }
                }
                acc += (e[t].area / V) * xin * fup;
            }
        }
        fstar[i] = fj[i] - dt * acc;
    }
}

/* ---- S4: rho = w sum m f ---- */
static void cell_moments(const oracle_t *o, const double *fc, double rho[5]) {
    const int nx = o->d.nv[0], ny = o->d.nv[1], nz = o->d.nv[2];
    double s[5] = {0, 0, 0, 0, 0};
    for (int kz = 0; kz < nz; kz++) for (int ky = 0; ky < ny; ky++) for (int kx = 0; kx < nx; kx++) {
        const double x = o->xi[0][kx], y = o->xi[1][ky], z = o->xi[2][kz];
        const double v = fc[((int64_t)kz * ny + ky) * nx + kx];
        s[0] += v; s[1] += x * v; s[2] += y * v; s[3] += z * v; s[4] += (x * x + y * y + z * z) * v;
    }
    for (int a = 0; a < 5; a++) rho[a] = o->w * s[a];
}

/* Gauss elimination with partial pivoting, 5x5 ("Gauss method") */
static int solve5(double A[5][5], double b[5], double x[5]) {
    for (int c = 0; c < 5; c++) {
        int p = c;
        for (int r = c + 1; r < 5; r++) if (fabs(A[r][c]) > fabs(A[p][c])) p = r;
        if (A[p][c] == 0.0) return -1;
        if (p != c) { for (int k = 0; k < 5; k++) { double t = A[c][k]; A[c][k] = A[p][k]; A[p][k] = t; } double t = b[c]; b[c] = b[p]; b[p] = t; }
        for (int r = c + 1; r < 5; r++) {
            double m = A[r][c] / A[c][c];
            for (int k = c; k < 5; k++) A[r][k] -= m * A[c][k];
            b[r] -= m * b[c];
        }
    }
    for (int r = 4; r >= 0; r--) {
        double s = b[r];
        for (int k = r + 1; k < 5; k++) s -= A[r][k] * x[k];
        x[r] = s / A[r][r];
    }
    return 0;
}

/* ---- S5: alpha with w sum m exp(alpha.m) = rho.  Returns iterations used, or -1 on failure ---- */
static int cell_newton(const oracle_t *o, const double rho[5], double alpha[5]) {
    const int nx = o->d.nv[0], ny = o->d.nv[1], nz = o->d.nv[2];
    const double n = rho[0];
    const double u[3] = {rho[1] / n, rho[2] / n, rho[3] / n};
    const double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    const double T = (rho[4] - n * uu) / (3.0 * n);
    if (!(n > 0.0) || !(T > 0.0)) return -1;
    alpha[0] = log(n / pow(2.0 * M_PI * T, 1.5)) - uu / (2.0 * T);
    alpha[1] = u[0] / T; alpha[2] = u[1] / T; alpha[3] = u[2] / T;
    alpha[4] = -1.0 / (2.0 * T);
    const double sT = n * sqrt(T);
    const double scale[5] = {n, sT + fabs(rho[1]), sT + fabs(rho[2]), sT + fabs(rho[3]), rho[4]};
    for (int it = 0; it <= 50; it++) {
        double F[5] = {0, 0, 0, 0, 0}, J[5][5];
        memset(J, 0, sizeof J);
        for (int kz = 0; kz < nz; kz++) for (int ky = 0; ky < ny; ky++) for (int kx = 0; kx < nx; kx++) {
            const double x = o->xi[0][kx], y = o->xi[1][ky], z = o->xi[2][kz];
            const double m[5] = {1.0, x, y, z, x * x + y * y + z * z};
            const double M = exp(alpha[0] + alpha[1] * x + alpha[2] * y + alpha[3] * z + alpha[4] * m[4]);
            for (int a = 0; a < 5; a++) {
                F[a] += m[a] * M;
                for (int b = a; b < 5; b++) J[a][b] += m[a] * m[b] * M;
            }
        }
        double res = 0.0;
        for (int a = 0; a < 5; a++) {
            F[a] = o->w * F[a] - rho[a];
            double r = fabs(F[a]) / scale[a];
            if (!(r <= res)) res = r; /* also catches NaN */
            for (int b = a; b < 5; b++) { J[a][b] *= o->w; J[b][a] = J[a][b]; }
        }
        if (res <= 1e-13) return it;
        if (it == 50 || !(res == res)) return -1;
        double dx[5];
        if (solve5(J, F, dx)) return -1;
        for (int a = 0; a < 5; a++) alpha[a] -= dx[a];
    }
    return -1;
}

/* ---- S4-S6 for one cell: fout[Nv] from fstar[Nv] ---- */
static int cell_relax(const oracle_t *o, const double *fstar, double dt, double *fout) {
    const int nx = o->d.nv[0], ny = o->d.nv[1], nz = o->d.nv[2];
    if (isinf(o->d.kn)) { memcpy(fout, fstar, o->Nv * sizeof(double)); return 0; } /* Kn = inf: nu = 0 */
    double rho[5], alpha[5];
    cell_moments(o, fstar, rho);
    int it = cell_newton(o, rho, alpha);
    if (it < 0) { memcpy(fout, fstar, o->Nv * sizeof(double)); return -1; }
    const double n = rho[0];
    const double uu = (rho[1] * rho[1] + rho[2] * rho[2] + rho[3] * rho[3]) / (n * n);
    const double T = (rho[4] - n * uu) / (3.0 * n);
    /* G9: nu = c_nu n T^(1-omega) / Kn; omega = 1/2 uses sqrt, not pow */
    const double Tp = (o->d.visc_exp == 0.5) ? sqrt(T) : pow(T, 1.0 - o->d.visc_exp);
    const double nu = o->d.nu_prefactor * n * Tp / o->d.kn;
    for (int kz = 0; kz < nz; kz++) for (int ky = 0; ky < ny; ky++) for (int kx = 0; kx < nx; kx++) {
        const int64_t i = ((int64_t)kz * ny + ky) * nx + kx;
        const double x = o->xi[0][kx], y = o->xi[1][ky], z = o->xi[2][kz];
        const double M = exp(alpha[0] + alpha[1] * x + alpha[2] * y + alpha[3] * z + alpha[4] * (x * x + y * y + z * z));
        fout[i] = fstar[i] + dt * nu * (M - fstar[i]);
    }
    return it;
}

static void note_newton(oracle_t *o, int it) {
    if (it < 0) {
#pragma omp atomic write
        o->newton_fail = 1;
    } else if (it > o->newton_max_iters) {
#pragma omp critical
        if (it > o->newton_max_iters) o->newton_max_iters = it;
    }
}

/* f_in, f_out: [n_kinetic][Nv], rows in leaf-list order of the kinetic leaves, canonical velocity order */
int oracle_dvm_transport(oracle_t *o, const double *f_in, double *f_out, double dt) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t r = 0; r < o->n_kin; r++) cell_transport(o, f_in, r, dt, f_out + r * o->Nv);
    return ORA_OK;
}

int oracle_dvm_relax(oracle_t *o, const double *fstar, double *f_out, double dt) {
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t r = 0; r < o->n_kin; r++) note_newton(o, cell_relax(o, fstar + r * o->Nv, dt, f_out + r * o->Nv));
    return o->newton_fail ? ORA_ENEWTON : ORA_OK;
}

int oracle_dvm_step(oracle_t *o, const double *f_in, double *f_out, double dt) {
    int oom = 0;
#pragma omp parallel
    {
        double *fstar = (double *)malloc(o->Nv * sizeof(double));
        if (!fstar) {
#pragma omp atomic write
            oom = 1;
        }
#pragma omp barrier
        if (!oom) {
#pragma omp for schedule(dynamic, 4)
            for (int64_t r = 0; r < o->n_kin; r++) {
                cell_transport(o, f_in, r, dt, fstar);
                note_newton(o, cell_relax(o, fstar, dt, f_out + r * o->Nv));
            }
        }
        free(fstar);
    }
    if (oom) return ORA_ENOMEM;
    return o->newton_fail ? ORA_ENEWTON : ORA_OK;
}

/* S7: mom[5][n_kinetic] = (n, n ux, n uy, n uz, E = rho_4/2) */
int oracle_dvm_moments(const oracle_t *o, const double *f, double *mom) {
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < o->n_kin; r++) {
        double rho[5];
        cell_moments(o, f + r * o->Nv, rho);
        for (int a = 0; a < 4; a++) mom[a * o->n_kin + r] = rho[a];
        mom[4 * o->n_kin + r] = 0.5 * rho[4];
    }
    return ORA_OK;
}

/* the Newton solve alone (pins P8, G7): returns iterations or -1 */
int oracle_dvm_newton(const oracle_t *o, const double *rho, double *alpha) { return cell_newton(o, rho, alpha); }
int oracle_dvm_newton_max_iters(const oracle_t *o) { return o->newton_max_iters; }

/* Interior faces between two non-solid leaves, each once, from the low-side cell's +direction entries
 * (owner = low-side cell, neigh = high-side cell, area = min(h)^2, ratio = level(neigh)-level(owner)).
 * Arrays may be NULL to get the count only. */
int64_t oracle_dvm_faces(const oracle_t *o, int64_t *owner, int64_t *neigh, double *area, int8_t *axis, int8_t *ratio) {
    int64_t cnt = 0;
    for (int64_t j = 0; j < o->d.n_leaves; j++) {
        if (o->kind[j] == ORA_SOLID) continue;
        for (int dir = 0; dir < 6; dir++) {
            const nb_entry *e = o->nb + (j * 6 + dir) * 4;
            for (int t = 0; t < o->nb_count[j * 6 + dir]; t++) {
                if (e[t].type != NB_LEAF || o->kind[e[t].id] == ORA_SOLID) continue;
                const int64_t q = e[t].id;
                /* list the face from the + side of the low cell; a coarse/fine pair is listed from
                 * whichever side is "+": the entry area is already min(h)^2 in both cases */
                if (!(dir & 1)) continue;
                if (owner) { owner[cnt] = j; neigh[cnt] = q; area[cnt] = e[t].area; axis[cnt] = (int8_t)(dir >> 1); ratio[cnt] = (int8_t)((int)o->level[q] - (int)o->level[j]); }
                cnt++;
            }
        }
    }
    return cnt;
}

/* boundary faces of non-solid leaves: counts per kind [periodic(unused), specular-domain, inflow, outflow, solid] */
void oracle_dvm_boundary_counts(const oracle_t *o, int64_t counts[5]) {
    for (int k = 0; k < 5; k++) counts[k] = 0;
    for (int64_t j = 0; j < o->d.n_leaves; j++) {
        if (o->kind[j] == ORA_SOLID) continue;
        for (int dir = 0; dir < 6; dir++) {
            const nb_entry *e = o->nb + (j * 6 + dir) * 4;
            for (int t = 0; t < o->nb_count[j * 6 + dir]; t++) {
                if (e[t].type == NB_BOUNDARY) counts[o->d.bc[e[t].side]]++;
                else if (e[t].type == NB_LEAF && o->kind[e[t].id] == ORA_SOLID) counts[4]++;
            }
        }
    }
}

/* ---- mesh change: f of a new leaf set from f of the old one ("steps 2 and 4 are
 * redone each time the spatial mesh is changed").  The paper does not say how f is carried over; reading G20
 * (DESIGN.md), the one consistent with the first-order piecewise-constant scheme (G2): the new value is the VOLUME
 * AVERAGE over the new leaf of the old piecewise-constant field --
 *   an unchanged leaf keeps its f; a leaf created by refinement takes the value of the old leaf that covers it
 *   (injection); a leaf created by coarsening takes sum_k (V_k / V_new) f_k over the old leaves k inside it;
 *   where the old covering leaf was FLUID the field is the Maxwellian of its frozen moments (G13).
 * One new leaf and one velocity at a time, plain recursion over the octree. */
static int remap_add(const oracle_t *old, const double *f_old, int level, int64_t cx, int64_t cy, int64_t cz, double wgt, double *acc) {
    const int64_t q = find_leaf(old, level, cx, cy, cz);
    if (q >= 0) {
        if (old->kind[q] == ORA_SOLID) return ORA_EINVAL;
        const int nx = old->d.nv[0], ny = old->d.nv[1], nz = old->d.nv[2];
        for (int kz = 0; kz < nz; kz++) for (int ky = 0; ky < ny; ky++) for (int kx = 0; kx < nx; kx++) {
            const int64_t i = ((int64_t)kz * ny + ky) * nx + kx;
            const double v = old->kind[q] == ORA_KINETIC ? f_old[old->row_of_leaf[q] * old->Nv + i]
                                                         : maxwell_point(old->fluid + 5 * q, old->xi[0][kx], old->xi[1][ky], old->xi[2][kz]);
            acc[i] += wgt * v;
        }
        return ORA_OK;
    }
    if (level >= 18) return ORA_EMESH; /* nothing of the old mesh lies here */
    for (int d = 0; d < 8; d++) {
        int rc = remap_add(old, f_old, level + 1, 2 * cx + (d & 1), 2 * cy + ((d >> 1) & 1), 2 * cz + ((d >> 2) & 1), wgt / 8.0, acc);
        if (rc) return rc;
    }
    return ORA_OK;
}

/* f_old: [old n_kinetic][Nv], f_new: [new n_kinetic][Nv]; both meshes must carry the same velocity grid */
int oracle_dvm_remap(const oracle_t *old, const oracle_t *neu, const double *f_old, double *f_new) {
    for (int a = 0; a < 3; a++)
        if (old->d.nv[a] != neu->d.nv[a] || old->d.vmin[a] != neu->d.vmin[a] || old->d.vmax[a] != neu->d.vmax[a]) return ORA_EINVAL;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t r = 0; r < neu->n_kin; r++) {
        const int64_t j = neu->kin_leaf[r];
        const int l = neu->level[j];
        const int64_t c[3] = {neu->ijk[3 * j], neu->ijk[3 * j + 1], neu->ijk[3 * j + 2]};
        double *out = f_new + r * neu->Nv;
        for (int64_t i = 0; i < neu->Nv; i++) out[i] = 0.0;
        /* an old leaf at the same level or above covers the new leaf: its (constant) value is the average */
        int done = 0;
        for (int ll = l; ll >= 0 && !done; ll--) {
            const int sh = l - ll;
            if (find_leaf(old, ll, c[0] >> sh, c[1] >> sh, c[2] >> sh) >= 0) {
                int rc = remap_add(old, f_old, ll, c[0] >> sh, c[1] >> sh, c[2] >> sh, 1.0, out);
                if (rc) {
#pragma omp atomic write
                    bad = rc;
                }
                done = 1;
            }
        }
        /* otherwise the old leaves inside the new one, each with its volume fraction */
        if (!done) {
            int rc = remap_add(old, f_old, l, c[0], c[1], c[2], 1.0, out);
            if (rc) {
#pragma omp atomic write
                bad = rc;
            }
        }
    }
    return bad;
}

/* face neighbours of one leaf (mesh query used to cut windows): returns count (<= 24) */
int oracle_dvm_leaf_neighbours(const oracle_t *o, int64_t leaf, int64_t *ids) {
    int cnt = 0;
    for (int dir = 0; dir < 6; dir++) {
        const nb_entry *e = o->nb + (leaf * 6 + dir) * 4;
        for (int t = 0; t < o->nb_count[leaf * 6 + dir]; t++)
            if (e[t].type == NB_LEAF) ids[cnt++] = e[t].id;
    }
    return cnt;
}

int oracle_dvm_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* timing aid (bench.py: the oracle with 1 thread and with all cores); no effect on any result */
void oracle_dvm_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
