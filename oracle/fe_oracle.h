/*
 * fe_oracle.h -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * Plain, slow, serial FP64 restatement of what the hot path of invDFT (arXiv 2510.10529) computes:
 * the spectral-finite-element Kohn-Sham operator  H~ = M^{-1/2} (1/2 K + M_V) M^{-1/2}  (PAPER.md
 * Eq. 17, Eq. 19-20, l.165-185) applied to a block of vectors, the per-column shifted apply
 * (H~ - eps_i) X_i (Eq. 20, l.183) and the Chebyshev filter of ChFSI (l.208-210).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.  It shares no code, table or constant with paper_2510_10529_b200/ (the CUDA
 * product) and neither side includes the other.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed-form GLL/Gauss rules and polynomial
 * exactness; brute-force l2g; sum(M) = volume; K.1 = 0; K(x^2+y^2+z^2) = -6 M; the textbook 8x8
 * trilinear Laplacian; symmetry; sum of cells == assembled CSR; 3-D harmonic oscillator levels
 * 1.5 / 2.5 / 3.5 converging with p; filter == T_m through a LAPACK eigendecomposition.
 * General (trilinearly mapped) cells and hanging nodes (orc_general_*, oracle/fe_general.py) are pinned in
 * tests/test_general_pins.py: an unrefined undeformed mesh reproduces everything above; a sheared cell equals the analytically
 * transformed reference matrix; continuity and patch tests (K_c linear = 0, K_c r^2 = -6 M_c) through hanging faces and edges;
 * density, potential-only operator and preconditioner through closed forms; apply_rows against the assembled operator.
 * "parity unpinned": the soft-Coulomb eigenvalues of configs 2-4 have no external truth; those
 * configs are pinned only through the invariants above.
 */
#ifndef FE_ORACLE_H
#define FE_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_mesh orc_mesh;
typedef struct orc_csr orc_csr;

/* 1-D rules (survey 8(c) step 1; PAPER.md l.185 names GLL; Gauss-Legendre n_q = p+1 is reading R1) */
int orc_gll(int p, double* x, double* w);            /* p+1 nodes/weights on [-1,1] */
int orc_gauss(int nq, double* x, double* w);         /* nq nodes/weights on [-1,1] */
/* Eq. 12: l_a(x) = prod_{j!=a} (x-x_j)/(x_a-x_j), and d/dx by the product rule */
double orc_lagrange(int n, const double* nodes, int a, double x);
double orc_lagrange_deriv(int n, const double* nodes, int a, double x);

/* tensor-product hex mesh, order p, GLL nodes, Dirichlet on the box surface (readings R2-R5) */
orc_mesh* orc_mesh_create(const double* xe, int cx, const double* ye, int cy, const double* ze, int cz, int p);
void orc_mesh_destroy(orc_mesh* m);
int64_t orc_num_nodes(const orc_mesh* m);
int64_t orc_num_free(const orc_mesh* m);
int64_t orc_num_cells(const orc_mesh* m);
int orc_nodes_per_cell(const orc_mesh* m);
int orc_quad_per_cell(const orc_mesh* m);
void orc_get_l2g(const orc_mesh* m, int32_t* l2g);          /* cells*n_c */
void orc_get_node_coords(const orc_mesh* m, double* xyz);   /* N*3 */
void orc_get_quad_coords(const orc_mesh* m, double* xyz);   /* cells*n_q^3*3 */
void orc_get_mass(const orc_mesh* m, double* Mdiag);        /* N, lumped GLL mass (l.185) */
void orc_get_mask(const orc_mesh* m, uint8_t* mask);        /* N, 1 = free, 0 = boundary */

/* Eq. 17 by explicit 3-D Gauss quadrature, one cell:  He = kin*K_e + pot*M_{V,e}  (n_c x n_c, row-major).
 * K_e[a,b] = int grad Phi_a . grad Phi_b,  M_{V,e}[a,b] = int V Phi_a Phi_b.  H_e = 0.5 K_e + M_V,e. */
void orc_cell_matrix(const orc_mesh* m, int64_t e, const double* Vq_cell, double kin, double pot, double* He);
/* all cells: He_all[e*n_c*n_c + a*n_c + b] = 0.5 K_e + M_V,e  (setup; OpenMP over cells) */
void orc_build_cell_matrices(const orc_mesh* m, const double* Vq, double* He_all);

/* H = sum_e P_e^T H_e P_e as CSR (int64 row pointers).  scaled != 0: H~ = S H S with boundary rows and
 * columns zeroed (Eq. 19, R5, R6); scaled == 0: the raw assembled H. */
orc_csr* orc_assemble(const orc_mesh* m, const double* He_all, int scaled);
void orc_csr_destroy(orc_csr* A);
int64_t orc_csr_nnz(const orc_csr* A);
void orc_csr_copy(const orc_csr* A, int64_t* row_ptr, int32_t* col, double* val);

/* Y = H~ X - X diag(eps) on free rows, 0 on boundary rows (Eq. 20).  X, Y: N x B, X[a*B+j]. eps may be NULL.
 * nthreads <= 1: serial; otherwise OpenMP over rows (same arithmetic per row). */
void orc_csr_apply(const orc_mesh* m, const orc_csr* A, const double* X, int B, const double* eps, double* Y, int nthreads);
/* same result from the cell-wise definition  Y = mu S sum_e P_e^T H_e P_e S mu X - eps X  (l.237, l.253) */
void orc_cellwise_apply(const orc_mesh* m, const double* He_all, const double* X, int B, const double* eps, double* Y);
/* selected rows of the same product straight from Eq. 17 (no stored matrices): Yrows[r*B+j] */
void orc_apply_rows(const orc_mesh* m, const double* Vq, const double* X, int B, const double* eps,
                    const int64_t* rows, int64_t nrows, double* Yrows);

/* Chebyshev filter (l.208-210; scaled three-term recurrence of reading R7), in place:
 * X <- T_m((H~-c)/e) X / T_m((a0-c)/e),  e=(b-a)/2, c=(b+a)/2.  Uses the CSR if A != NULL else He_all. */
int orc_filter(const orc_mesh* m, const orc_csr* A, const double* He_all, double* X, int B, int deg,
               double a, double b, double a0, int nthreads);

/* General (trilinearly mapped) hexahedral cell, corners verts[8*3] with corner v = vx + 2(vy + 2vz) (NEXT-3; l.151, l.273):
 * He = kin*K_e + pot*M_{V,e} by explicit quadrature with the Jacobian of the map at every Gauss point. */
void orc_general_cell_matrix(int p, const double* verts, const double* Vq_cell, double kin, double pot, double* He);
/* positions and |det J| of the trilinear map at npts reference points xi (npts*3) */
void orc_general_map(const double* verts, const double* xi, int npts, double* pos, double* det);

#ifdef __cplusplus
}
#endif
#endif
