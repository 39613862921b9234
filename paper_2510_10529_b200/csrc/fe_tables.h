// 1-D reference tables of the spectral element (host side).  PAPER.md Eq. 12 (l.124), l.185; readings R1, R4.
#pragma once

namespace fecheb {

constexpr int kMaxN = 9;  // p <= 8

struct Tables1D {
    int p, n;
    double gll_x[kMaxN], gll_w[kMaxN];  // Gauss-Lobatto-Legendre nodes / weights (nodes of the basis, lumped mass)
    double gl_x[kMaxN], gl_w[kMaxN];    // Gauss-Legendre points / weights, n_q = p+1 (quadrature of K and M_V)
    double N[kMaxN * kMaxN];            // N[q*n+a] = l_a(gl_x[q]): interpolation GLL nodes -> Gauss points
    double G[kMaxN * kMaxN];            // G[q*n+r] = sum_s w_s D~[s][q] D~[s][r]: 1-D stiffness on the Gauss points
    double D[kMaxN * kMaxN];            // D[s*n+q] = l^_q'(gl_x[s]): collocation derivative on the Gauss points
};

// Golub-Welsch nodes (Jacobi rotations on the Jacobi matrices of the Legendre and Jacobi(1,1) weights),
// barycentric Lagrange evaluation, collocation derivative on the Gauss points.
void build_tables(int p, Tables1D* t);

// l_a(x), a = 0..p, of the GLL Lagrange basis at an arbitrary point (barycentric form; exact cardinality at the nodes)
void lagrange_gll(const Tables1D& t, double x, double* out);

}  // namespace fecheb
