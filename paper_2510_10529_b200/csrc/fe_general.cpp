// fe_general.cpp -- builds the tables of a general hexahedral mesh with hanging nodes from the caller's leaf list.
//
// Node identity uses exact integer keys (the oracle matches nodes geometrically instead): along an axis a local node a of
// the level-l cell i is (l, i, a), with the last node a = p of a cell renamed (l, i+1, 0), so that the two cells of one
// level that share a face produce the same key.  A node of a level-l cell hangs when it lies in the closure of a leaf of
// level l-1; whether it does is integer arithmetic on (i, a).  Numbering (reading R23): cells in the caller's order, local
// nodes a = ax + n (ay + n az); unconstrained nodes 0..N-1 in order of first appearance, hanging nodes N.. likewise.
#include "fe_general.h"

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <map>
#include <unordered_map>

namespace fecheb {
namespace {

struct KeyHash {
    size_t operator()(const std::array<int32_t, 7>& k) const
    {
        uint64_t h = 1469598103934665603ull;
        for (int32_t v : k) { h ^= (uint32_t)v; h *= 1099511628211ull; }
        return (size_t)h;
    }
};
struct LeafHash {
    size_t operator()(const std::array<int32_t, 4>& k) const
    {
        uint64_t h = 1469598103934665603ull;
        for (int32_t v : k) { h ^= (uint32_t)v; h *= 1099511628211ull; }
        return (size_t)h;
    }
};

// position, Jacobian J[i][j] = dx_i / dxi_j of the trilinear map at reference point (x, y, z)
void trilinear(const double* V, double x, double y, double z, double pos[3], double J[3][3])
{
    const double tx[2] = {0.5 * (1 - x), 0.5 * (1 + x)}, ty[2] = {0.5 * (1 - y), 0.5 * (1 + y)}, tz[2] = {0.5 * (1 - z), 0.5 * (1 + z)};
    const double d[2] = {-0.5, 0.5};
    for (int i = 0; i < 3; ++i) { pos[i] = 0; J[i][0] = J[i][1] = J[i][2] = 0; }
    for (int v = 0; v < 8; ++v) {
        const int vx = v & 1, vy = (v >> 1) & 1, vz = v >> 2;
        const double w = tx[vx] * ty[vy] * tz[vz], wx = d[vx] * ty[vy] * tz[vz], wy = tx[vx] * d[vy] * tz[vz], wz = tx[vx] * ty[vy] * d[vz];
        for (int i = 0; i < 3; ++i) {
            const double c = V[3 * v + i];
            pos[i] += c * w; J[i][0] += c * wx; J[i][1] += c * wy; J[i][2] += c * wz;
        }
    }
}

double det3(const double J[3][3])
{
    return J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0]) +
           J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
}

}  // namespace

int build_general_mesh(int cx, int cy, int cz, const int32_t* cells, int64_t ncells, const double* verts, int p,
                       const Tables1D& tab, GeneralHost* out, char* err, size_t errlen)
{
    auto fail = [&](const char* msg, long long a = 0, long long b = 0) {
        snprintf(err, errlen, msg, a, b);
        return -1;
    };
    const int n = p + 1, nc = n * n * n;
    const int croot[3] = {cx, cy, cz};
    GeneralHost& g = *out;
    g.p = p; g.n = n; g.nc = nc; g.ncells = ncells;
    std::unordered_map<std::array<int32_t, 4>, int32_t, LeafHash> leaf;
    leaf.reserve((size_t)ncells * 2);
    int maxlevel = 0;
    for (int64_t e = 0; e < ncells; ++e) {
        const int32_t* c = cells + 4 * e;
        if (c[0] < 0 || c[0] > 12) return fail("fe_mesh_create_general: cell %lld has level %lld outside 0..12", e, c[0]);
        for (int d = 0; d < 3; ++d)
            if (c[1 + d] < 0 || c[1 + d] >= (croot[d] << c[0])) return fail("fe_mesh_create_general: cell %lld lies outside the root grid", e);
        if (!leaf.emplace(std::array<int32_t, 4>{c[0], c[1], c[2], c[3]}, (int32_t)e).second)
            return fail("fe_mesh_create_general: cell %lld listed twice", e);
        maxlevel = std::max(maxlevel, (int)c[0]);
    }
    // leaves must not overlap (no ancestor of a leaf is a leaf) and levels of touching leaves differ by at most one
    auto leaf_at_or_above = [&](int l, int ix, int iy, int iz, int* found_level) -> int {
        for (; l >= 0; --l, ix >>= 1, iy >>= 1, iz >>= 1) {
            auto it = leaf.find({l, ix, iy, iz});
            if (it != leaf.end()) { *found_level = l; return it->second; }
        }
        return -1;
    };
    for (int64_t e = 0; e < ncells; ++e) {
        const int32_t* c = cells + 4 * e;
        int fl;
        if (c[0] > 0 && leaf_at_or_above(c[0] - 1, c[1] >> 1, c[2] >> 1, c[3] >> 1, &fl) >= 0)
            return fail("fe_mesh_create_general: cell %lld overlaps a coarser leaf", e);
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    const int jx = c[1] + dx, jy = c[2] + dy, jz = c[3] + dz;
                    if (jx < 0 || jy < 0 || jz < 0 || jx >= (cx << c[0]) || jy >= (cy << c[0]) || jz >= (cz << c[0])) continue;
                    if (leaf_at_or_above(c[0], jx, jy, jz, &fl) >= 0 && fl < c[0] - 1)
                        return fail("fe_mesh_create_general: 2:1 balance violated at cell %lld (neighbour of level %lld)", e, fl);
                }
    }

    // ---- pass 1: slots in order of first appearance; hanging test and parent (coarse leaf) per slot ------------------------
    struct Slot { int32_t parent; double xi[3]; };
    std::unordered_map<std::array<int32_t, 7>, int32_t, KeyHash> slot_of;
    slot_of.reserve((size_t)ncells * nc);
    std::vector<Slot> slots;
    std::vector<int32_t> l2slot((size_t)ncells * nc);
    std::vector<uint8_t> slot_bnd;
    for (int64_t e = 0; e < ncells; ++e) {
        const int32_t* c = cells + 4 * e;
        const int l = c[0];
        for (int a = 0; a < nc; ++a) {
            const int la[3] = {a % n, (a / n) % n, a / (n * n)};
            int idx[3], loc[3];
            for (int d = 0; d < 3; ++d) {
                idx[d] = c[1 + d] + (la[d] == p ? 1 : 0);
                loc[d] = la[d] == p ? 0 : la[d];
            }
            const std::array<int32_t, 7> key{l, idx[0], loc[0], idx[1], loc[1], idx[2], loc[2]};
            auto it = slot_of.find(key);
            if (it == slot_of.end()) {
                Slot s;
                s.parent = -1;
                if (l > 0) {
                    // candidate level-(l-1) cells per axis: the node at fine position idx (+ a fraction if loc > 0) lies in
                    // [2j, 2j+2] (fine units)
                    int cand[3][2], ncand[3];
                    for (int d = 0; d < 3; ++d) {
                        ncand[d] = 0;
                        if (loc[d] > 0) cand[d][ncand[d]++] = idx[d] >> 1;
                        else {
                            const int lim = croot[d] << (l - 1);
                            if ((idx[d] & 1) == 0) {  // on a coarse lattice plane: the coarse cells on both sides
                                if (idx[d] / 2 - 1 >= 0) cand[d][ncand[d]++] = idx[d] / 2 - 1;
                                if (idx[d] / 2 < lim) cand[d][ncand[d]++] = idx[d] / 2;
                            } else cand[d][ncand[d]++] = idx[d] >> 1;
                        }
                    }
                    int best = -1, bj[3] = {0, 0, 0};
                    for (int kz = 0; kz < ncand[2]; ++kz)
                        for (int ky = 0; ky < ncand[1]; ++ky)
                            for (int kx = 0; kx < ncand[0]; ++kx) {
                                auto lt = leaf.find({l - 1, cand[0][kx], cand[1][ky], cand[2][kz]});
                                if (lt != leaf.end() && (best < 0 || lt->second < best)) {
                                    best = lt->second;
                                    bj[0] = cand[0][kx]; bj[1] = cand[1][ky]; bj[2] = cand[2][kz];
                                }
                            }
                    if (best >= 0) {
                        s.parent = best;
                        for (int d = 0; d < 3; ++d) {
                            const double t = loc[d] > 0 ? 0.5 * (tab.gll_x[loc[d]] + 1.0) : 0.0;
                            const int off = idx[d] - 2 * bj[d];  // 0, 1 or 2
                            s.xi[d] = off == 2 ? 1.0 : (off == 0 && loc[d] == 0 ? -1.0 : (double)(off - 1) + t);
                        }
                    }
                }
                bool bnd = false;
                for (int d = 0; d < 3; ++d) bnd = bnd || (loc[d] == 0 && (idx[d] == 0 || idx[d] == (croot[d] << l)));
                it = slot_of.emplace(key, (int32_t)slots.size()).first;
                slots.push_back(s);
                slot_bnd.push_back(bnd ? 1 : 0);
            }
            l2slot[(size_t)e * nc + a] = it->second;
        }
    }
    const int64_t nslots = (int64_t)slots.size();
    if (nslots > 2147483647ll) return fail("fe_mesh_create_general: more than 2^31-1 nodes");
    std::vector<int32_t> id(nslots);
    int64_t nm = 0, nh = 0;
    for (int64_t s = 0; s < nslots; ++s)
        if (slots[s].parent < 0) id[s] = (int32_t)nm++;
    for (int64_t s = 0; s < nslots; ++s)
        if (slots[s].parent >= 0) id[s] = (int32_t)(nm + nh++);
    g.N = nm; g.N_all = nslots;
    g.l2g.resize((size_t)ncells * nc);
    for (size_t i = 0; i < g.l2g.size(); ++i) g.l2g[i] = id[l2slot[i]];
    g.mask.assign((size_t)nm, 1);
    for (int64_t s = 0; s < nslots; ++s)
        if (slots[s].parent < 0 && slot_bnd[s]) g.mask[id[s]] = 0;

    // ---- constraint rows: the coarse cell's Lagrange basis at the node, chains substituted ----------------------------------
    std::vector<std::map<int32_t, double>> rows((size_t)nh);
    for (int64_t s = 0; s < nslots; ++s) {
        if (slots[s].parent < 0) continue;
        double w[3][kMaxN];
        for (int d = 0; d < 3; ++d) lagrange_gll(tab, slots[s].xi[d], w[d]);
        auto& row = rows[(size_t)(id[s] - nm)];
        const int32_t* pl = &g.l2g[(size_t)slots[s].parent * nc];
        for (int b = 0; b < nc; ++b) {
            const double v = w[0][b % n] * w[1][(b / n) % n] * w[2][b / (n * n)];
            if (std::fabs(v) > 1e-14) row[pl[b]] += v;
        }
    }
    for (bool changed = true; changed;) {
        changed = false;
        for (auto& row : rows)
            for (auto it = row.begin(); it != row.end();) {
                if (it->first < nm) { ++it; continue; }
                const double w = it->second;
                const auto sub = rows[(size_t)(it->first - nm)];  // copy: the row itself may be edited below
                it = row.erase(it);
                for (const auto& kv : sub) row[kv.first] += w * kv.second;
                changed = true;
                it = row.begin();
            }
    }
    g.crow.assign((size_t)nh + 1, 0);
    for (int64_t r = 0; r < nh; ++r) g.crow[r + 1] = g.crow[r] + (int64_t)rows[r].size();
    g.ccol.resize((size_t)g.crow[nh]);
    g.cval.resize((size_t)g.crow[nh]);
    for (int64_t r = 0; r < nh; ++r) {
        int64_t k = g.crow[r];
        for (const auto& kv : rows[r]) { g.ccol[k] = kv.first; g.cval[k] = kv.second; ++k; }
    }

    // ---- geometry: nodal masses and coordinates at the GLL nodes, metric and coordinates at the Gauss points ------------------
    g.node_xyz.assign((size_t)nslots * 3, 0.0);
    g.m_all.assign((size_t)nslots, 0.0);
    g.quad_xyz.resize((size_t)ncells * nc * 3);
    g.metric.resize((size_t)ncells * 7 * nc);
    for (int64_t e = 0; e < ncells; ++e) {
        const double* V = verts + (size_t)e * 24;
        for (int a = 0; a < nc; ++a) {
            const int ax = a % n, ay = (a / n) % n, az = a / (n * n);
            double pos[3], J[3][3];
            trilinear(V, tab.gll_x[ax], tab.gll_x[ay], tab.gll_x[az], pos, J);
            const int32_t gi = g.l2g[(size_t)e * nc + a];
            for (int d = 0; d < 3; ++d) g.node_xyz[(size_t)gi * 3 + d] = pos[d];
            g.m_all[gi] += tab.gll_w[ax] * tab.gll_w[ay] * tab.gll_w[az] * std::fabs(det3(J));
        }
        double* M = &g.metric[(size_t)e * 7 * nc];
        for (int q = 0; q < nc; ++q) {
            const int qx = q % n, qy = (q / n) % n, qz = q / (n * n);
            double pos[3], J[3][3];
            trilinear(V, tab.gl_x[qx], tab.gl_x[qy], tab.gl_x[qz], pos, J);
            const double det = det3(J);
            if (!(std::fabs(det) > 0.0) || !std::isfinite(det)) return fail("fe_mesh_create_general: cell %lld is degenerate at quadrature point %lld", e, q);
            for (int d = 0; d < 3; ++d) g.quad_xyz[((size_t)e * nc + q) * 3 + d] = pos[d];
            // Ji = J^-1 (cofactors);  metric = Ji Ji^T  (reference-space Gram matrix of the physical gradients)
            double Ji[3][3];
            Ji[0][0] = (J[1][1] * J[2][2] - J[1][2] * J[2][1]) / det; Ji[0][1] = (J[0][2] * J[2][1] - J[0][1] * J[2][2]) / det;
            Ji[0][2] = (J[0][1] * J[1][2] - J[0][2] * J[1][1]) / det; Ji[1][0] = (J[1][2] * J[2][0] - J[1][0] * J[2][2]) / det;
            Ji[1][1] = (J[0][0] * J[2][2] - J[0][2] * J[2][0]) / det; Ji[1][2] = (J[0][2] * J[1][0] - J[0][0] * J[1][2]) / det;
            Ji[2][0] = (J[1][0] * J[2][1] - J[1][1] * J[2][0]) / det; Ji[2][1] = (J[0][1] * J[2][0] - J[0][0] * J[2][1]) / det;
            Ji[2][2] = (J[0][0] * J[1][1] - J[0][1] * J[1][0]) / det;
            const double wd = tab.gl_w[qx] * tab.gl_w[qy] * tab.gl_w[qz] * std::fabs(det);
            int c = 0;
            for (int i = 0; i < 3; ++i)
                for (int j = i; j < 3; ++j) {
                    const double gij = Ji[i][0] * Ji[j][0] + Ji[i][1] * Ji[j][1] + Ji[i][2] * Ji[j][2];
                    M[(size_t)c * nc + q] = 0.5 * wd * gij;
                    ++c;
                }
            M[(size_t)6 * nc + q] = wd;
        }
    }
    g.mass.assign((size_t)nm, 0.0);
    for (int64_t i = 0; i < nm; ++i) g.mass[i] = g.m_all[i];
    for (int64_t r = 0; r < nh; ++r)
        for (int64_t k = g.crow[r]; k < g.crow[r + 1]; ++k) g.mass[g.ccol[k]] += g.cval[k] * g.m_all[nm + r];
    for (int64_t i = 0; i < nm; ++i)
        if (g.mask[i] && !(g.mass[i] > 0.0)) return fail("fe_mesh_create_general: lumped mass of node %lld is not positive", i);
    return 0;
}

}  // namespace fecheb
