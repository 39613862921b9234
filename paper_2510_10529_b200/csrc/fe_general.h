// fe_general.h -- host-side description of a general hexahedral mesh with hanging nodes (PAPER.md
// l.151, l.273, Fig. 6) as the library builds it from the caller's leaf list: explicit local-to-global map, constraint rows
// of the hanging nodes, nodal masses, Dirichlet mask and the per-quadrature-point metric of the trilinear cells.
#pragma once
#include <cstddef>
#include <cstdint>
#include <vector>

#include "fe_tables.h"

namespace fecheb {

struct GeneralHost {
    int p = 0, n = 0, nc = 0;
    int64_t ncells = 0, N = 0, N_all = 0;       // N unconstrained nodes (rows of the blocks), N_all - N hanging nodes
    std::vector<int32_t> l2g;                   // ncells * nc, ids in [0, N_all): < N unconstrained, >= N hanging
    std::vector<int64_t> crow;                  // N_all - N + 1: constraint rows, hanging node h = N + r
    std::vector<int32_t> ccol;                  //   unconstrained node ids
    std::vector<double> cval;                   //   weights: u_h = sum_k cval u_ccol
    std::vector<double> node_xyz;               // N_all * 3
    std::vector<double> quad_xyz;               // ncells * nc * 3
    std::vector<double> m_all;                  // N_all: GLL-quadrature nodal masses  w_a |det J(xi_a)|  summed over cells
    std::vector<double> mass;                   // N: lumped constrained mass  C^T m_all  (reading R25)
    std::vector<uint8_t> mask;                  // N: 1 = free, 0 = on the surface of the root box
    // per cell and quadrature point q = qx + n (qy + n qz):  [e][c][q], c = 0..5: 1/2 w_q |det J| (J^-1 J^-T) entries
    // (xx, xy, xz, yy, yz, zz) in reference coordinates; c = 6: w_q |det J|
    std::vector<double> metric;
};

// cells: ncells rows (level, ix, iy, iz); verts: ncells * 8 * 3 corner coordinates, corner v = vx + 2 (vy + 2 vz).
// Returns 0, or -1 with a message (invalid leaf list, 2:1 balance violated, inverted cell).
int build_general_mesh(int cx, int cy, int cz, const int32_t* cells, int64_t ncells, const double* verts, int p,
                       const Tables1D& tab, GeneralHost* out, char* err, size_t errlen);

}  // namespace fecheb
