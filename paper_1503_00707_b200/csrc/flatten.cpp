// flatten.cpp -- host-side octree flattener (see flatten.hpp).  Neighbour search by binary search in
// the Morton-sorted leaf array: a leaf at level l covers the key interval [key, key + 8^(lmax-l)), the
// leaves tile [0, 8^lmax), so "which leaf covers this point" is one upper_bound.
#include "flatten.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

namespace ufs {
namespace {

inline uint64_t spread3(uint64_t v) {  // 21 bits -> every third bit
    v &= 0x1fffffULL;
    v = (v | (v << 32)) & 0x1f00000000ffffULL;
    v = (v | (v << 16)) & 0x1f0000ff0000ffULL;
    v = (v | (v << 8)) & 0x100f00f00f00f00fULL;
    v = (v | (v << 4)) & 0x10c30c30c30c30c3ULL;
    v = (v | (v << 2)) & 0x1249249249249249ULL;
    return v;
}
// depth-first order with child index x + 2y + 4z
inline uint64_t morton(uint64_t x, uint64_t y, uint64_t z) { return spread3(x) | (spread3(y) << 1) | (spread3(z) << 2); }

struct Tree {
    const ufs_dvm_desc& d;
    int lmax;
    std::vector<uint64_t> start;  // Morton-sorted start keys
    std::vector<int64_t> order;   // rank -> leaf
    // leaf covering the finest-level point (x,y,z)
    int64_t cover(int64_t x, int64_t y, int64_t z) const {
        uint64_t key = morton((uint64_t)x, (uint64_t)y, (uint64_t)z);
        auto it = std::upper_bound(start.begin(), start.end(), key);
        return order[(it - start.begin()) - 1];
    }
};

enum : int8_t { NB_NONE = 0, NB_LEAF = 1, NB_DOMAIN = 2 };
struct Nb {
    int8_t type[4];
    int8_t cnt;
    int64_t id[4];  // leaf, or domain side
};

int build_velocity(const ufs_dvm_desc& d, VelLayout& v, std::string& err) {
    v.Nv = 1;
    v.w = 1.0;
    v.fast = true;
    for (int a = 0; a < 3; a++) {
        if (d.nv[a] < 1 || d.nv[a] > NV_MAX) { err = "nv must be in 1.." + std::to_string(NV_MAX) + " on every axis"; return UFS_DVM_EINVAL; }
        if (!(d.vmax[a] > d.vmin[a])) { err = "vmax must exceed vmin"; return UFS_DVM_EINVAL; }
        v.nv[a] = d.nv[a];
        v.Nv *= d.nv[a];
        const double dv = (d.vmax[a] - d.vmin[a]) / d.nv[a];
        v.w *= dv;
        v.ncls[a][0] = v.ncls[a][1] = v.ncls[a][2] = 0;
        for (int k = 0; k < d.nv[a]; k++) v.xi[a][k] = d.vmin[a] + (k + 0.5) * dv;
        v.symmetric[a] = std::fabs(d.vmin[a] + d.vmax[a]) <= 1e-14 * std::fabs(d.vmax[a]);
        if (v.symmetric[a]) {  // make the nodes exactly mirror-symmetric so |xi| depends on the rank only
            for (int k = 0; k < d.nv[a] / 2; k++) v.xi[a][k] = -v.xi[a][d.nv[a] - 1 - k];
            if (d.nv[a] % 2) v.xi[a][d.nv[a] / 2] = 0.0;
        }
        for (int k = 0; k < d.nv[a]; k++) v.ncls[a][v.xi[a][k] < 0 ? 0 : (v.xi[a][k] > 0 ? 1 : 2)]++;
        v.nh[a] = d.nv[a] / 2;
        if (!(v.symmetric[a] && d.nv[a] % 2 == 0)) v.fast = false;
        if (v.ncls[a][2] > 1) { err = "internal: two zero nodes"; return UFS_DVM_EINVAL; }
    }
    // class and rank (by increasing |xi|) of every node
    int cls[3][NV_MAX], rk[3][NV_MAX];
    for (int a = 0; a < 3; a++)
        for (int k = 0; k < v.nv[a]; k++) {
            const double x = v.xi[a][k];
            if (x < 0) { cls[a][k] = 0; rk[a][k] = v.ncls[a][0] - 1 - k; }       // negative nodes come first
            else if (x > 0) { cls[a][k] = 1; rk[a][k] = k - (v.nv[a] - v.ncls[a][1]); }
            else { cls[a][k] = 2; rk[a][k] = 0; }
        }
    // groups in order (cz, cy, cx), cx fastest; with no zero class this is octant sx + 2 sy + 4 sz
    int64_t gstart[3][3][3];
    int64_t off = 0;
    for (int cz = 0; cz < 3; cz++) for (int cy = 0; cy < 3; cy++) for (int cx = 0; cx < 3; cx++) {
        gstart[cz][cy][cx] = off;
        off += (int64_t)v.ncls[0][cx] * v.ncls[1][cy] * v.ncls[2][cz];
    }
    v.vel_of_slot.assign(v.Nv, -1);
    v.slot_of_vel.assign(v.Nv, -1);
    v.slot_k.assign(v.Nv * 4, 0);
    for (int kz = 0; kz < v.nv[2]; kz++) for (int ky = 0; ky < v.nv[1]; ky++) for (int kx = 0; kx < v.nv[0]; kx++) {
        const int cx = cls[0][kx], cy = cls[1][ky], cz = cls[2][kz];
        const int64_t slot = gstart[cz][cy][cx] + ((int64_t)rk[2][kz] * v.ncls[1][cy] + rk[1][ky]) * v.ncls[0][cx] + rk[0][kx];
        const int64_t can = ((int64_t)kz * v.nv[1] + ky) * v.nv[0] + kx;
        v.vel_of_slot[slot] = (int32_t)can;
        v.slot_of_vel[can] = (int32_t)slot;
        v.slot_k[slot * 4 + 0] = (uint8_t)kx; v.slot_k[slot * 4 + 1] = (uint8_t)ky; v.slot_k[slot * 4 + 2] = (uint8_t)kz;
    }
    for (int a = 0; a < 3; a++) {
        v.mirror_slot[a].assign(v.Nv, -1);
        if (!v.symmetric[a]) continue;
        for (int64_t s = 0; s < v.Nv; s++) {
            int k[3] = {v.slot_k[s * 4], v.slot_k[s * 4 + 1], v.slot_k[s * 4 + 2]};
            k[a] = v.nv[a] - 1 - k[a];
            v.mirror_slot[a][s] = v.slot_of_vel[((int64_t)k[2] * v.nv[1] + k[1]) * v.nv[0] + k[0]];
        }
    }
    return UFS_DVM_OK;
}

// pointwise Maxwellian n/(2 pi T)^{3/2} exp(-|xi-u|^2/2T) as separable factors (reading G13)
void maxwell_factors(const double* prim, const VelLayout& v, FluidGhost& g) {
    const double PI = 3.14159265358979323846;
    const double n = prim[0], T = prim[4];
    g.amp = n / std::pow(2.0 * PI * T, 1.5);
    for (int a = 0; a < 3; a++)
        for (int k = 0; k < v.nv[a]; k++) {
            const double c = v.xi[a][k] - prim[1 + a];
            g.g[a][k] = std::exp(-c * c / (2.0 * T));
        }
}

}  // namespace

int flatten(const ufs_dvm_desc& d, FlatMesh& m, std::string& err) {
    if (d.n_leaves <= 0 || !d.level || !d.ijk || !d.kind) { err = "empty or NULL leaf list"; return UFS_DVM_EINVAL; }
    if (!(d.domain_len > 0)) { err = "domain_len must be positive"; return UFS_DVM_EINVAL; }
    if (d.storage != UFS_STORE_F64 && d.storage != UFS_STORE_F32) { err = "unknown storage type"; return UFS_DVM_EINVAL; }
    if (!(d.kn > 0)) { err = "kn must be positive (+inf = collisions off)"; return UFS_DVM_EINVAL; }
    for (int a = 0; a < 3; a++) {
        for (int s = 0; s < 2; s++)
            if (d.bc[2 * a + s] < UFS_BC_PERIODIC || d.bc[2 * a + s] > UFS_BC_OUTFLOW) { err = "unknown boundary code"; return UFS_DVM_EINVAL; }
        if ((d.bc[2 * a] == UFS_BC_PERIODIC) != (d.bc[2 * a + 1] == UFS_BC_PERIODIC)) { err = "periodic must be set on both sides of an axis"; return UFS_DVM_EINVAL; }
    }
    int rc = build_velocity(d, m.vel, err);
    if (rc) return rc;
    const VelLayout& vel = m.vel;
    const int64_t n = d.n_leaves;
    m.n_leaves = n;

    // ---- Morton order and the tiling check --------------------------------------------------------
    int lmax = 0;
    bool any_solid = false, any_fluid = false;
    for (int64_t j = 0; j < n; j++) {
        if (d.level[j] > 18) { err = "level > 18"; return UFS_DVM_EINVAL; }
        if (d.kind[j] > UFS_CELL_SOLID) { err = "unknown cell kind"; return UFS_DVM_EINVAL; }
        lmax = std::max<int>(lmax, d.level[j]);
        any_solid |= d.kind[j] == UFS_CELL_SOLID;
        any_fluid |= d.kind[j] == UFS_CELL_FLUID;
    }
    if (any_fluid && !d.fluid_moments) { err = "FLUID leaves need fluid_moments"; return UFS_DVM_EINVAL; }
    m.lmax = lmax;
    std::vector<uint64_t> key(n);
    for (int64_t j = 0; j < n; j++) {
        const int l = d.level[j];
        const uint32_t nl = 1u << l;
        const uint32_t* c = d.ijk + 3 * j;
        if (c[0] >= nl || c[1] >= nl || c[2] >= nl) { err = "leaf " + std::to_string(j) + " lies outside the cube"; return UFS_DVM_EMESH; }
        const int sh = lmax - l;
        key[j] = morton((uint64_t)c[0] << sh, (uint64_t)c[1] << sh, (uint64_t)c[2] << sh);
    }
    m.order.resize(n);
    std::iota(m.order.begin(), m.order.end(), (int64_t)0);
    std::sort(m.order.begin(), m.order.end(), [&](int64_t a, int64_t b) { return key[a] != key[b] ? key[a] < key[b] : d.level[a] < d.level[b]; });
    Tree t{d, lmax, {}, m.order};
    t.start.resize(n);
    uint64_t expect = 0;
    for (int64_t r = 0; r < n; r++) {
        const int64_t j = m.order[r];
        t.start[r] = key[j];
        if (key[j] != expect) {
            err = std::string(key[j] < expect ? "leaves overlap" : "leaves leave a gap") + " at leaf " + std::to_string(j);
            return UFS_DVM_EMESH;
        }
        expect = key[j] + (1ULL << (3 * (lmax - d.level[j])));
    }
    if (expect != (1ULL << (3 * lmax))) { err = "leaves do not fill the cube"; return UFS_DVM_EMESH; }
    m.rank.resize(n);
    for (int64_t r = 0; r < n; r++) m.rank[m.order[r]] = r;

    // ---- neighbour search (6 faces) and the 26-neighbour 2:1 check --------------------
    std::vector<Nb> nb((size_t)n * 6);
    int bad = 0;
    const int64_t NF = (int64_t)1 << lmax;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (int64_t j = 0; j < n; j++) {
        const int l = d.level[j];
        const int sh = lmax - l;
        const int64_t nl = (int64_t)1 << l;
        const int64_t c[3] = {d.ijk[3 * j], d.ijk[3 * j + 1], d.ijk[3 * j + 2]};
        // 26 neighbours: the covering leaf of the adjacent same-size block may not be coarser than l-1
        for (int dz = -1; dz <= 1; dz++) for (int dy = -1; dy <= 1; dy++) for (int dx = -1; dx <= 1; dx++) {
            if (!dx && !dy && !dz) continue;
            int64_t q[3] = {c[0] + dx, c[1] + dy, c[2] + dz};
            bool outside = false;
            for (int a = 0; a < 3; a++) {
                if (q[a] < 0 || q[a] >= nl) {
                    if (d.bc[2 * a] == UFS_BC_PERIODIC) q[a] = (q[a] + nl) % nl;
                    else outside = true;
                }
            }
            if (outside) continue;
            const int64_t cov = t.cover(q[0] << sh, q[1] << sh, q[2] << sh);
            if ((int)d.level[cov] < l - 1) bad |= 1;
        }
        for (int dir = 0; dir < 6; dir++) {
            Nb& e = nb[(size_t)j * 6 + dir];
            std::memset(&e, 0, sizeof e);
            const int a = dir >> 1, s = (dir & 1) ? 1 : -1;
            int64_t q[3] = {c[0], c[1], c[2]};
            q[a] += s;
            if (q[a] < 0 || q[a] >= nl) {
                if (d.bc[dir] == UFS_BC_PERIODIC) q[a] = (q[a] + nl) % nl;
                else { e.cnt = 1; e.type[0] = NB_DOMAIN; e.id[0] = dir; continue; }
            }
            const int64_t cov = t.cover(q[0] << sh, q[1] << sh, q[2] << sh);
            const int lc = d.level[cov];
            if (lc <= l) {  // same level or coarser: one face
                if (lc < l - 1) bad |= 1;
                e.cnt = 1; e.type[0] = NB_LEAF; e.id[0] = cov;
                continue;
            }
            // finer: the four level-(l+1) children of the adjacent block that touch the shared face
            if (sh < 1) { bad |= 1; continue; }
            const int b1 = (a + 1) % 3, b2 = (a + 2) % 3;
            int cnt = 0;
            for (int u = 0; u < 2; u++) for (int w = 0; w < 2; w++) {
                int64_t cc[3];
                cc[a] = 2 * q[a] + (s > 0 ? 0 : 1);
                cc[b1] = 2 * q[b1] + u;
                cc[b2] = 2 * q[b2] + w;
                const int64_t ch = t.cover(cc[0] << (sh - 1), cc[1] << (sh - 1), cc[2] << (sh - 1));
                if ((int)d.level[ch] != l + 1) bad |= 1;
                e.type[cnt] = NB_LEAF; e.id[cnt] = ch; cnt++;
            }
            e.cnt = 4;
        }
    }
    (void)NF;
    if (bad) { err = "octree is not 2:1 balanced (face, edge or corner neighbours differ by more than one level)"; return UFS_DVM_EMESH; }

    // ---- specular reflection needs a mirror-symmetric velocity grid on the wall-normal axis -----------
    for (int a = 0; a < 3; a++) {
        const bool need = any_solid || d.bc[2 * a] == UFS_BC_SPECULAR || d.bc[2 * a + 1] == UFS_BC_SPECULAR;
        if (need && !vel.symmetric[a]) { err = "specular walls / SOLID leaves need vmin = -vmax on axis " + std::to_string(a); return UFS_DVM_EINVAL; }
    }

    // ---- slabs: kinetic leaves in Morton order -----------------------------------------------------
    m.slab_of_leaf.assign(n, -1);
    m.cell_of_slab.clear();
    for (int64_t r = 0; r < n; r++) {
        const int64_t j = m.order[r];
        if (d.kind[j] == UFS_CELL_KINETIC) { m.slab_of_leaf[j] = (int64_t)m.cell_of_slab.size(); m.cell_of_slab.push_back(j); }
    }
    m.n_kin = (int64_t)m.cell_of_slab.size();
    if (m.n_kin >= (1 << SRC_SHIFT)) { err = "too many kinetic leaves for the 28-bit source index"; return UFS_DVM_EINVAL; }

    // ---- face lists, in Morton order of the owner ----------------------------------------------------
    for (int64_t r = 0; r < n; r++) {
        const int64_t j = m.order[r];
        if (d.kind[j] == UFS_CELL_SOLID) continue;
        const double h = d.domain_len / (double)((int64_t)1 << d.level[j]);
        for (int a = 0; a < 3; a++) {
            for (int side = 0; side < 2; side++) {
                const Nb& e = nb[(size_t)j * 6 + 2 * a + side];
                for (int k = 0; k < e.cnt; k++) {
                    const double area = (e.cnt == 4) ? 0.25 * h * h : h * h;  // min(h_o,h_n)^2: our own face is never the larger one unless cnt==4
                    if (e.type[k] == NB_DOMAIN) {
                        const int bc = d.bc[e.id[k]];
                        m.b_cell.push_back(j); m.b_axis.push_back((int8_t)a); m.b_side.push_back((int8_t)side); m.b_area.push_back(area);
                        m.b_kind.push_back((int8_t)(bc == UFS_BC_SPECULAR ? UFS_BF_SPECULAR : bc == UFS_BC_INFLOW ? UFS_BF_INFLOW : UFS_BF_OUTFLOW));
                        m.b_state.push_back(e.id[k]);
                        continue;
                    }
                    const int64_t q = e.id[k];
                    if (d.kind[q] == UFS_CELL_SOLID) {
                        m.b_cell.push_back(j); m.b_axis.push_back((int8_t)a); m.b_side.push_back((int8_t)side); m.b_area.push_back(area);
                        m.b_kind.push_back((int8_t)UFS_BF_SOLID); m.b_state.push_back(q);
                        continue;
                    }
                    if (d.kind[j] == UFS_CELL_KINETIC && d.kind[q] == UFS_CELL_FLUID) {
                        m.b_cell.push_back(j); m.b_axis.push_back((int8_t)a); m.b_side.push_back((int8_t)side); m.b_area.push_back(area);
                        m.b_kind.push_back((int8_t)UFS_BF_FLUID); m.b_state.push_back(q);
                    }
                    if (side == 1) {  // interior face, listed once from its low-side cell
                        m.f_owner.push_back(j); m.f_neigh.push_back(q); m.f_area.push_back(area);
                        m.f_axis.push_back((int8_t)a); m.f_ratio.push_back((int8_t)((int)d.level[q] - (int)d.level[j]));
                    }
                }
            }
        }
    }

    // ---- ghost states: inflow tables (slot order) and fluid-leaf Maxwellian factors -----------------
    m.n_tables = 0;
    for (int s = 0; s < 6; s++) {
        m.table_of_side[s] = -1;
        if (d.bc[s] != UFS_BC_INFLOW) continue;
        if (!(d.inflow[s][0] > 0) || !(d.inflow[s][4] > 0)) { err = "inflow state needs n > 0 and T > 0"; return UFS_DVM_EINVAL; }
        m.table_of_side[s] = m.n_tables++;
        FluidGhost g;
        maxwell_factors(d.inflow[s], vel, g);
        const size_t base = m.tables.size();
        m.tables.resize(base + vel.Nv);
        for (int64_t sl = 0; sl < vel.Nv; sl++)
            m.tables[base + sl] = g.amp * g.g[2][vel.slot_k[sl * 4 + 2]] * g.g[1][vel.slot_k[sl * 4 + 1]] * g.g[0][vel.slot_k[sl * 4 + 0]];
    }
    std::vector<int64_t> ghost_of_leaf;
    if (any_fluid) ghost_of_leaf.assign(n, -1);
    auto fluid_ghost = [&](int64_t q) -> int64_t {
        if (ghost_of_leaf[q] < 0) {
            const double* pm = d.fluid_moments + 5 * q;
            ghost_of_leaf[q] = (int64_t)m.fluid.size();
            m.fluid_leaf.push_back(q);
            m.fluid.emplace_back();
            maxwell_factors(pm, vel, m.fluid.back());
        }
        return ghost_of_leaf[q];
    };

    // ---- per-cell upwind gather records, derived from the two face lists ---------------------------
    m.recs.assign(m.n_kin, CellRec{});
    for (auto& r : m.recs) {
        for (int dd = 0; dd < 6; dd++) for (int k = 0; k < 4; k++) r.src[dd][k] = -1;
    }
    std::vector<int8_t> cnt((size_t)m.n_kin * 6, 0);
    auto push = [&](int64_t slab, int dir, int32_t code) -> bool {
        int8_t& c = cnt[(size_t)slab * 6 + dir];
        if (c >= 4) return false;
        m.recs[slab].src[dir][c++] = code;
        return true;
    };
    auto code_of = [&](int64_t q) -> int32_t {  // data of leaf q as seen from a kinetic neighbour
        if (d.kind[q] == UFS_CELL_KINETIC) return src_code(SRC_SLAB, m.slab_of_leaf[q]);
        return src_code(SRC_FLUID, fluid_ghost(q));
    };
    bool ok = true;
    for (size_t f = 0; f < m.f_owner.size(); f++) {
        const int64_t p = m.f_owner[f], q = m.f_neigh[f];
        const int a = m.f_axis[f];
        if (d.kind[p] == UFS_CELL_KINETIC) {
            if (d.kind[q] == UFS_CELL_FLUID && !(d.fluid_moments[5 * q] > 0 && d.fluid_moments[5 * q + 4] > 0)) { err = "fluid_moments need n > 0 and T > 0"; return UFS_DVM_EINVAL; }
            ok &= push(m.slab_of_leaf[p], 2 * a + 1, code_of(q));
        }
        if (d.kind[q] == UFS_CELL_KINETIC) {
            if (d.kind[p] == UFS_CELL_FLUID && !(d.fluid_moments[5 * p] > 0 && d.fluid_moments[5 * p + 4] > 0)) { err = "fluid_moments need n > 0 and T > 0"; return UFS_DVM_EINVAL; }
            ok &= push(m.slab_of_leaf[q], 2 * a, code_of(p));
        }
    }
    for (size_t b = 0; b < m.b_cell.size(); b++) {
        const int64_t j = m.b_cell[b];
        if (d.kind[j] != UFS_CELL_KINETIC || m.b_kind[b] == UFS_BF_FLUID) continue;
        const int64_t slab = m.slab_of_leaf[j];
        const int dir = 2 * m.b_axis[b] + m.b_side[b];
        int32_t code;
        switch (m.b_kind[b]) {
            case UFS_BF_SPECULAR: case UFS_BF_SOLID: code = src_code(SRC_MIRROR, slab); break;
            case UFS_BF_INFLOW: code = src_code(SRC_TABLE, m.table_of_side[m.b_state[b]]); break;
            default: code = src_code(SRC_SLAB, slab); break;  // outflow: ghost = own cell (zero gradient)
        }
        ok &= push(slab, dir, code);
    }
    m.n_simple = 0;
    for (int64_t s = 0; s < m.n_kin; s++) {
        CellRec& r = m.recs[s];
        r.level = d.level[m.cell_of_slab[s]];
        bool simple = true, nofluid = true, ringfluid = true;
        for (int dd = 0; dd < 6; dd++) {
            const int c = cnt[(size_t)s * 6 + dd];
            if (c != 1 && c != 4) ok = false;
            if (c != 1) simple = false;
            for (int k = 0; k < c; k++)
                if ((r.src[dd][k] >> SRC_SHIFT) == SRC_FLUID) {
                    simple = nofluid = false;
                    if (c != 1) ringfluid = false;  // a fluid leaf among four finer neighbours: plain gather path
                }
        }
        r.flags = (simple ? CELL_SIMPLE : 0) | (nofluid ? CELL_NOFLUID : 0) | (!nofluid && ringfluid ? CELL_RINGFLUID : 0);
        // per velocity octant: which upwind directions (xi_a > 0: the low side) bring four sources / a fluid source
        r.masks = r.fmasks = 0;
        for (int o = 0; o < 8; o++)
            for (int a = 0; a < 3; a++) {
                const int dd = 2 * a + (1 - ((o >> a) & 1));
                if (cnt[(size_t)s * 6 + dd] == 4) r.masks |= 1 << (3 * o + a);
                else if ((r.src[dd][0] >> SRC_SHIFT) == SRC_FLUID) r.fmasks |= 1 << (3 * o + a);
            }
        m.n_simple += simple;
    }
    if (!ok) { err = "internal: a kinetic cell has a direction with neither 1 nor 4 sources"; return UFS_DVM_EMESH; }

    // ---- the leaf list and its sorted keys stay with the mesh (mesh changes: build_remap) ----
    m.leaf_level.assign(d.level, d.level + n);
    m.leaf_kind.assign(d.kind, d.kind + n);
    if (d.fluid_moments) m.leaf_fluid.assign(d.fluid_moments, d.fluid_moments + 5 * n);
    m.start_keys = t.start;

    // ---- sibling octets among the slabs (tiles): eight consecutive slabs that are the children 0..7 of one parent ----
    m.octet_start.assign(m.n_kin, 0);
    for (int64_t s = 0; s + 7 < m.n_kin; s++) {
        const int64_t j = m.cell_of_slab[s];
        const uint32_t* c = d.ijk + 3 * j;
        if (d.level[j] == 0 || ((c[0] | c[1] | c[2]) & 1u)) continue;
        bool all = true;
        for (int i = 1; i < 8 && all; i++) {
            const int64_t q = m.cell_of_slab[s + i];
            const uint32_t* cq = d.ijk + 3 * q;
            all = d.level[q] == d.level[j] && cq[0] == c[0] + (i & 1) && cq[1] == c[1] + ((i >> 1) & 1) && cq[2] == c[2] + ((i >> 2) & 1);
        }
        m.octet_start[s] = all ? 1 : 0;
    }
    m.n_slabs = m.n_kin;
    return UFS_DVM_OK;
}

// ---- multi-GPU: N-order partition and one rank's part of the mesh ----------------------------
int partition_leaves(const ufs_dvm_desc& d, int n_ranks, double w_kinetic, double w_fluid, int32_t* rank_of_leaf, std::string& err) {
    if (d.n_leaves <= 0 || !d.level || !d.ijk || !d.kind || !rank_of_leaf) { err = "empty or NULL leaf list"; return UFS_DVM_EINVAL; }
    if (n_ranks < 1) { err = "n_ranks must be at least 1"; return UFS_DVM_EINVAL; }
    if (!(w_kinetic > 0) || !(w_fluid >= 0)) { err = "weights: w_kinetic > 0, w_fluid >= 0"; return UFS_DVM_EINVAL; }
    const int64_t n = d.n_leaves;
    int lmax = 0;
    for (int64_t j = 0; j < n; j++) {
        if (d.level[j] > 18) { err = "level > 18"; return UFS_DVM_EINVAL; }
        lmax = std::max<int>(lmax, d.level[j]);
    }
    std::vector<uint64_t> key(n);
    for (int64_t j = 0; j < n; j++) {
        const int sh = lmax - d.level[j];
        const uint32_t* c = d.ijk + 3 * j;
        key[j] = morton((uint64_t)c[0] << sh, (uint64_t)c[1] << sh, (uint64_t)c[2] << sh);
    }
    std::vector<int64_t> order(n);
    std::iota(order.begin(), order.end(), (int64_t)0);
    std::sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return key[a] != key[b] ? key[a] < key[b] : d.level[a] < d.level[b]; });
    auto weight = [&](int64_t j) { return d.kind[j] == UFS_CELL_KINETIC ? w_kinetic : d.kind[j] == UFS_CELL_FLUID ? w_fluid : 0.0; };
    long double total = 0;
    for (int64_t j = 0; j < n; j++) total += weight(j);
    if (!(total > 0)) { err = "the mesh has no leaf of positive weight"; return UFS_DVM_EINVAL; }
    long double before = 0;
    int last = 0;
    for (int64_t r = 0; r < n; r++) {
        const int64_t j = order[r];
        int rk = (int)(before * n_ranks / total);
        rk = std::min(std::max(rk, last), n_ranks - 1);   // monotone along the curve whatever the rounding does
        rank_of_leaf[j] = rk;
        last = rk;
        before += weight(j);
    }
    return UFS_DVM_OK;
}

int restrict_to_rank(FlatMesh& m, const int32_t* rank_of_leaf, int my_rank, int n_ranks, std::string& err) {
    if (!rank_of_leaf || n_ranks < 1 || my_rank < 0 || my_rank >= n_ranks) { err = "bad rank arguments"; return UFS_DVM_EINVAL; }
    const int64_t NG = m.n_kin;   // slabs of the whole mesh
    // the rank's kinetic leaves must be one range of consecutive slabs (a range of the N-order curve)
    int64_t g0 = -1, g1 = -1;
    for (int64_t s = 0; s < NG; s++) {
        const int32_t rk = rank_of_leaf[m.cell_of_slab[s]];
        if (rk < 0 || rk >= n_ranks) { err = "rank_of_leaf out of range"; return UFS_DVM_EINVAL; }
        if (rk != my_rank) continue;
        if (g0 < 0) g0 = s;
        else if (g1 != s) { err = "the kinetic leaves of a rank must be consecutive in N-order (Morton) among the kinetic leaves"; return UFS_DVM_EINVAL; }
        g1 = s + 1;
    }
    if (g0 < 0) g0 = g1 = 0;
    const int64_t n_in = g1 - g0;
    auto octants_of_dir = [](int dd) -> uint8_t {   // octants whose upwind side on axis dd/2 is side dd%2 (low side: xi > 0)
        uint8_t mk = 0;
        for (int o = 0; o < 8; o++)
            if (((o >> (dd >> 1)) & 1) == 1 - (dd & 1)) mk |= (uint8_t)(1u << o);
        return mk;
    };
    // what each rank needs of the slabs it does not own: need[slab] = octant mask, per needing rank (sparse maps)
    std::vector<std::vector<std::pair<int64_t, uint8_t>>> wanted_from_me(n_ranks);   // (my global slab, mask) wanted by rank p
    std::vector<std::pair<int64_t, uint8_t>> my_ghosts;                             // (global slab, mask) I want
    {
        std::vector<uint8_t> mine(NG, 0);                       // masks of the ghosts I want
        std::vector<std::vector<uint8_t>> theirs;               // per peer: masks over MY slabs [g0, g1)
        theirs.assign(n_ranks, std::vector<uint8_t>());
        for (int64_t s = 0; s < NG; s++) {
            const int32_t rk = rank_of_leaf[m.cell_of_slab[s]];
            const CellRec& r = m.recs[s];
            for (int dd = 0; dd < 6; dd++)
                for (int k = 0; k < 4; k++) {
                    const int32_t code = r.src[dd][k];
                    if (code < 0 || (code >> SRC_SHIFT) != SRC_SLAB) continue;
                    const int64_t q = code & SRC_INDEX_MASK;
                    const int32_t rq = rank_of_leaf[m.cell_of_slab[q]];
                    if (rq == rk) continue;
                    if (rk == my_rank) mine[q] |= octants_of_dir(dd);
                    else if (rq == my_rank) {
                        if (theirs[rk].empty()) theirs[rk].assign(n_in, 0);
                        theirs[rk][q - g0] |= octants_of_dir(dd);
                    }
                }
        }
        for (int64_t q = 0; q < NG; q++)
            if (mine[q]) my_ghosts.emplace_back(q, mine[q]);
        for (int pr = 0; pr < n_ranks; pr++)
            for (int64_t i = 0; i < (int64_t)theirs[pr].size(); i++)
                if (theirs[pr][i]) wanted_from_me[pr].emplace_back(g0 + i, theirs[pr][i]);
    }
    const int64_t n_gh = (int64_t)my_ghosts.size();
    if (n_in + n_gh >= (1 << SRC_SHIFT)) { err = "too many slabs for the 28-bit source index"; return UFS_DVM_EINVAL; }
    // local numbering: inner slabs first, ghosts after, both in ascending global order
    std::vector<int64_t> local_of_global(NG, -1);
    for (int64_t s = g0; s < g1; s++) local_of_global[s] = s - g0;
    for (int64_t i = 0; i < n_gh; i++) local_of_global[my_ghosts[i].first] = n_in + i;
    std::vector<CellRec> recs(m.recs.begin() + g0, m.recs.begin() + g1);
    for (auto& r : recs)
        for (int dd = 0; dd < 6; dd++)
            for (int k = 0; k < 4; k++) {
                const int32_t code = r.src[dd][k];
                if (code < 0) continue;
                const int kind = code >> SRC_SHIFT;
                if (kind != SRC_SLAB && kind != SRC_MIRROR) continue;
                r.src[dd][k] = src_code((SrcKind)kind, local_of_global[code & SRC_INDEX_MASK]);
            }
    std::vector<int64_t> cell_of_slab(n_in + n_gh);
    for (int64_t s = 0; s < n_in; s++) cell_of_slab[s] = m.cell_of_slab[g0 + s];
    m.ghost_owner.assign(n_gh, 0);
    m.send_slab.assign(n_ranks, {}); m.recv_slab.assign(n_ranks, {});
    m.send_mask.assign(n_ranks, {}); m.recv_mask.assign(n_ranks, {});
    for (int64_t i = 0; i < n_gh; i++) {
        const int64_t leaf = m.cell_of_slab[my_ghosts[i].first];
        cell_of_slab[n_in + i] = leaf;
        const int32_t ow = rank_of_leaf[leaf];
        m.ghost_owner[i] = ow;
        m.recv_slab[ow].push_back((int32_t)(n_in + i));
        m.recv_mask[ow].push_back(my_ghosts[i].second);
    }
    for (int pr = 0; pr < n_ranks; pr++)
        for (const auto& e : wanted_from_me[pr]) {
            m.send_slab[pr].push_back((int32_t)(e.first - g0));
            m.send_mask[pr].push_back(e.second);
        }
    std::vector<uint8_t> octet(n_in, 0);
    for (int64_t s = 0; s + 7 < n_in; s++) octet[s] = m.octet_start[g0 + s];
    m.octet_start.swap(octet);
    m.recs.swap(recs);
    m.cell_of_slab.swap(cell_of_slab);
    std::fill(m.slab_of_leaf.begin(), m.slab_of_leaf.end(), (int64_t)-1);
    for (int64_t s = 0; s < n_in + n_gh; s++) m.slab_of_leaf[m.cell_of_slab[s]] = s;
    m.n_kin = n_in;
    m.n_slabs = n_in + n_gh;
    m.partial = true;
    m.my_rank = my_rank; m.n_ranks = n_ranks;
    m.first_global_slab = g0;
    m.n_simple = 0;
    for (const auto& r : m.recs) m.n_simple += (r.flags & CELL_SIMPLE) ? 1 : 0;
    return UFS_DVM_OK;
}

namespace {

// Piece list and cell index tables of the tile [s0, s0 + nc) for every octant.  Returns false if an octant needs more
// than pmax pieces.
struct TileBuild {
    uint32_t pieces[8][256];
    int np[8];
    uint8_t cidx[8][TILE_CELLS][CELLIDX_BYTES];
    bool any_fluid;
};
bool make_tile(const FlatMesh& m, int64_t s0, int nc, int pmax, TileBuild& t) {
    t.any_fluid = false;
    for (int o = 0; o < 8; o++) {
        int np = 0;
        auto piece = [&](uint32_t code) -> int {
            for (int i = 0; i < np; i++) if (t.pieces[o][i] == code) return i;
            if (np < 255) t.pieces[o][np] = code;
            return np++;
        };
        std::memset(t.cidx[o], IDX_NONE, sizeof t.cidx[o]);
        // own chunks first: piece c is the own chunk of cell c
        for (int c = 0; c < nc; c++) t.cidx[o][c][0] = (uint8_t)piece((uint32_t)((s0 + c) * 8 + o));
        for (int c = 0; c < nc; c++) {
            const CellRec& r = m.recs[s0 + c];
            uint8_t flags = 0;
            uint32_t fmask = 0;   // bit 4a + k: source k on axis a is a fluid leaf
            for (int a = 0; a < 3; a++) {
                const int dir = 2 * a + (1 - ((o >> a) & 1));  // xi_a > 0: data comes from the low side
                const int cnt = r.src[dir][1] >= 0 ? 4 : 1;
                if (cnt == 4) flags |= (uint8_t)(1 << a);
                for (int k = 0; k < cnt; k++) {
                    const int32_t code = r.src[dir][k];
                    const int kind = code >> SRC_SHIFT;
                    const int64_t idx = code & SRC_INDEX_MASK;
                    uint32_t pc;
                    if (kind == SRC_SLAB) pc = (uint32_t)(idx * 8 + o);
                    else if (kind == SRC_MIRROR) pc = (uint32_t)(idx * 8 + (o ^ (1 << a)));  // specular: mirrored octant of the own slab
                    else if (kind == SRC_FLUID) {   // the producer warps write its factor rows into the slot (nothing is copied)
                        pc = PIECE_FLUID | (uint32_t)(idx * 8 + o);
                        flags |= CIDX_FLUID; fmask |= 1u << (4 * a + k); t.any_fluid = true;
                    } else pc = PIECE_TABLE | (uint32_t)(idx * 8 + o);
                    const int pi = piece(pc);
                    if (pi >= IDX_NONE) return false;
                    t.cidx[o][c][4 + 4 * a + k] = (uint8_t)pi;
                }
            }
            t.cidx[o][c][1] = flags;
            t.cidx[o][c][2] = (uint8_t)(fmask & 0xff);
            t.cidx[o][c][3] = (uint8_t)(fmask >> 8);
        }
        if (np > pmax) return false;
        t.np[o] = np;
    }
    return true;
}

}  // namespace

int build_remap(const FlatMesh& o, const FlatMesh& nw, RemapPlan& plan, std::string& err) {
    for (int a = 0; a < 3; a++)
        if (o.vel.nv[a] != nw.vel.nv[a] || o.vel.xi[a][0] != nw.vel.xi[a][0] || o.vel.xi[a][o.vel.nv[a] - 1] != nw.vel.xi[a][o.vel.nv[a] - 1]) {
            err = "mesh change: the two meshes must carry the same velocity grid";
            return UFS_DVM_EINVAL;
        }
    const int LM = std::max(o.lmax, nw.lmax);               // common key depth
    const int sh_o = 3 * (LM - o.lmax), sh_n = 3 * (LM - nw.lmax);
    plan = RemapPlan{};
    plan.off.assign(nw.n_kin + 1, 0);
    std::vector<int64_t> ghost_of_leaf;
    for (int64_t s = 0; s < nw.n_kin; s++) {
        const int64_t j = nw.cell_of_slab[s];
        const uint64_t k0 = nw.start_keys[nw.rank[j]] << sh_n;
        const uint64_t size = 1ULL << (3 * (LM - nw.leaf_level[j]));
        // first old leaf whose key interval contains k0
        auto it = std::upper_bound(o.start_keys.begin(), o.start_keys.end(), k0 >> sh_o);
        int64_t r = (it - o.start_keys.begin()) - 1;
        int nsrc = 0;
        while (r < o.n_leaves && (o.start_keys[r] << sh_o) < k0 + size) {
            const int64_t q = o.order[r];
            const uint64_t qsize = 1ULL << (3 * (LM - o.leaf_level[q]));
            int32_t code;
            if (o.leaf_kind[q] == UFS_CELL_KINETIC) {
                code = (int32_t)o.slab_of_leaf[q];
            } else if (o.leaf_kind[q] == UFS_CELL_FLUID) {
                if (ghost_of_leaf.empty()) ghost_of_leaf.assign(o.n_leaves, -1);
                if (ghost_of_leaf[q] < 0) {
                    ghost_of_leaf[q] = (int64_t)plan.ghosts.size();
                    plan.ghosts.emplace_back();
                    plan.ghost_leaf.push_back(q);
                    maxwell_factors(o.leaf_fluid.data() + 5 * q, o.vel, plan.ghosts.back());
                }
                code = (int32_t)(-1 - ghost_of_leaf[q]);
                plan.n_from_fluid++;
            } else {
                err = "mesh change: a new KINETIC leaf lies over a SOLID leaf of the old mesh";
                return UFS_DVM_EINVAL;
            }
            plan.src.push_back(code);
            plan.wgt.push_back(qsize >= size ? 1.0 : (double)qsize / (double)size);
            nsrc++;
            if (qsize >= size) break;   // one old leaf covers the new one
            r++;
        }
        if (nsrc == 0) { err = "mesh change: internal: no source for a new leaf"; return UFS_DVM_EMESH; }
        const int64_t q0 = o.order[(it - o.start_keys.begin()) - 1];
        if (nsrc > 1) plan.n_restrict++;
        else if (o.leaf_level[q0] == nw.leaf_level[j]) plan.n_copy++;
        else plan.n_prolong++;
        plan.off[s + 1] = (int64_t)plan.src.size();
    }
    return UFS_DVM_OK;
}

void build_tiles(FlatMesh& m, int pmax) {
    m.tile_pmax = pmax;
    m.tiles.clear(); m.tile_pieces.clear(); m.tile_cellidx.clear();
    m.tiles_have_fluid = !m.fluid.empty();
    // pass 1 (serial, cheap): tile boundaries; pass 2: fill the arrays
    std::vector<int64_t> start; std::vector<int> count;
    TileBuild* tb = new TileBuild;
    for (int64_t s = 0; s < m.n_kin;) {
        int nc = 0;
        if (m.octet_start[s] && make_tile(m, s, 8, pmax, *tb)) nc = 8;
        if (!nc) {
            // a run of consecutive slabs that stops before the next complete octet and while the piece lists fit
            nc = 1;
            while (nc < TILE_CELLS && s + nc < m.n_kin && !m.octet_start[s + nc] && make_tile(m, s, nc + 1, pmax, *tb)) nc++;
        }
        start.push_back(s); count.push_back(nc);
        s += nc;
    }
    delete tb;
    const int64_t nt = (int64_t)start.size();
    m.tiles.assign(nt, TileHdr{});
    m.tile_pieces.assign((size_t)nt * 8 * pmax, 0u);
    m.tile_cellidx.assign((size_t)nt * 8 * TILE_CELLS * CELLIDX_BYTES, IDX_NONE);
#pragma omp parallel
    {
        TileBuild* t = new TileBuild;
#pragma omp for schedule(static)
        for (int64_t i = 0; i < nt; i++) {
            make_tile(m, start[i], count[i], pmax, *t);
            TileHdr& h = m.tiles[i];
            h.s0 = (int32_t)start[i]; h.nc = count[i];
            for (int c = 0; c < TILE_CELLS; c++) h.level[c] = c < count[i] ? (uint8_t)m.recs[start[i] + c].level : 0;
            for (int o = 0; o < 8; o++) {
                h.np[o] = (uint8_t)t->np[o];
                std::memcpy(&m.tile_pieces[((size_t)i * 8 + o) * pmax], t->pieces[o], (size_t)t->np[o] * 4);
                std::memcpy(&m.tile_cellidx[((size_t)i * 8 + o) * TILE_CELLS * CELLIDX_BYTES], t->cidx[o], TILE_CELLS * CELLIDX_BYTES);
            }
        }
        delete t;
    }
}

int build_push(FlatMesh& m, const void* const* peer_f0, const void* const* peer_f1, const int32_t* const* dest_slab, int64_t slab_bytes,
               const void* const* peer_sums0, const void* const* peer_sums1, int64_t sums_row_bytes, std::string& err) {
    if (!m.partial) { err = "fused ghost exchange: not a partitioned mesh"; return UFS_DVM_EINVAL; }
    if (m.tiles.empty() && m.n_kin > 0) { err = "fused ghost exchange: needs the tile kernel (k_tiles)"; return UFS_DVM_EINVAL; }
    // per inner slab: the peers that need it
    std::vector<std::vector<PushEntry>> of_slab(m.n_kin);
    for (int pr = 0; pr < m.n_ranks; pr++) {
        const size_t ns = m.send_slab[pr].size();
        if (ns == 0) continue;
        if (!peer_f0[pr] || !peer_f1[pr] || !dest_slab[pr]) {
            err = "fused ghost exchange: rank " + std::to_string(pr) + " needs cells of this rank, but its buffers or slab list are NULL";
            return UFS_DVM_EINVAL;
        }
        for (size_t i = 0; i < ns; i++) {
            const int32_t s = m.send_slab[pr][i], d = dest_slab[pr][i];
            if (s < 0 || s >= m.n_kin || d < 0) { err = "fused ghost exchange: slab out of range"; return UFS_DVM_EINVAL; }
            PushEntry e{};
            e.dst[0] = (uint64_t)(uintptr_t)peer_f0[pr] + (uint64_t)d * (uint64_t)slab_bytes;
            e.dst[1] = (uint64_t)(uintptr_t)peer_f1[pr] + (uint64_t)d * (uint64_t)slab_bytes;
            if (peer_sums0 && peer_sums1) {
                if (!peer_sums0[pr] || !peer_sums1[pr]) {
                    err = "fused ghost exchange: the sums arrays of rank " + std::to_string(pr) + " are NULL";
                    return UFS_DVM_EINVAL;
                }
                e.sums_dst[0] = (uint64_t)(uintptr_t)peer_sums0[pr] + (uint64_t)d * (uint64_t)sums_row_bytes;
                e.sums_dst[1] = (uint64_t)(uintptr_t)peer_sums1[pr] + (uint64_t)d * (uint64_t)sums_row_bytes;
            }
            e.info = m.send_mask[pr][i];
            if ((e.dst[0] | e.dst[1]) & 15) { err = "fused ghost exchange: peer buffers must be 16-byte aligned"; return UFS_DVM_EINVAL; }
            of_slab[s].push_back(e);
        }
    }
    // tiles with a cell some peer needs come first: k_tiles' PUSH instantiation runs over them, before the plain one runs
    // over the rest (the pushed rows are on their way while the interior is computed)
    const size_t nt = m.tiles.size();
    std::vector<size_t> perm;
    perm.reserve(nt);
    auto needed = [&](const TileHdr& t) {
        for (int c = 0; c < t.nc; c++)
            if (!of_slab[t.s0 + c].empty()) return true;
        return false;
    };
    for (size_t i = 0; i < nt; i++) if (needed(m.tiles[i])) perm.push_back(i);
    m.n_push_tiles = (int64_t)perm.size();
    for (size_t i = 0; i < nt; i++) if (!needed(m.tiles[i])) perm.push_back(i);
    {
        const size_t ps = (size_t)8 * m.tile_pmax, cs = (size_t)8 * TILE_CELLS * CELLIDX_BYTES;
        std::vector<TileHdr> th(nt);
        std::vector<uint32_t> tp(m.tile_pieces.size());
        std::vector<uint8_t> tc(m.tile_cellidx.size());
        for (size_t i = 0; i < nt; i++) {
            th[i] = m.tiles[perm[i]];
            std::memcpy(tp.data() + i * ps, m.tile_pieces.data() + perm[i] * ps, ps * 4);
            std::memcpy(tc.data() + i * cs, m.tile_cellidx.data() + perm[i] * cs, cs);
        }
        m.tiles.swap(th); m.tile_pieces.swap(tp); m.tile_cellidx.swap(tc);
    }
    m.tile_push.clear();
    for (TileHdr& t : m.tiles) {
        t.pad[0] = (int32_t)m.tile_push.size();
        uint32_t counts = 0;
        for (int c = 0; c < t.nc; c++) {
            const std::vector<PushEntry>& v = of_slab[t.s0 + c];
            if ((int)v.size() > PUSH_PER_CELL_MAX) {
                err = "fused ghost exchange: a cell is needed by more than " + std::to_string(PUSH_PER_CELL_MAX) + " peers; use ufs_dvm_halo_pack / unpack";
                return UFS_DVM_EINVAL;
            }
            counts |= (uint32_t)v.size() << (4 * c);
            m.tile_push.insert(m.tile_push.end(), v.begin(), v.end());
        }
        t.pad[1] = (int32_t)counts;
    }
    return UFS_DVM_OK;
}

}  // namespace ufs
