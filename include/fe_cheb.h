/*
 * fe_cheb.h -- C ABI of the B200-native hot path of invDFT (arXiv 2510.10529).
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers; R-numbers are the readings listed
 * in DESIGN.md):
 *
 *   H~ = M^{-1/2} (1/2 K + M_V) M^{-1/2}                                   (Eq. 17 l.171, Eq. 19 l.181-185)
 *
 * the spectral-finite-element Kohn-Sham operator on a tensor-product hexahedral mesh (Lagrange order p on
 * Gauss-Lobatto-Legendre nodes, Eq. 12 l.124; lumped GLL mass, l.185; zero Dirichlet data on the box surface, R5;
 * K and M_V integrated with p+1 Gauss-Legendre points per direction, R1), applied to a block of B vectors stored
 * "all vectors of one basis function contiguous" (l.233-235, Fig. 4(a) l.253):  X[a*B + j] = node a, vector j.
 *
 *   fe_apply_H : Y = H~ X, or column-wise (H~ - eps_j I) X_j                  (Eq. 20 l.183; adjoint solve l.221-225)
 *   cheb_filter: X <- T_m((H~ - c)/e) X / T_m((a0 - c)/e)                     (ChFSI filter, l.208-210; R7)
 *
 * Every step runs in hand-written sm_100a kernels; there is no CPU fallback.  All functions return 0 on success
 * and a negative code on failure (FE_ERR_*); fe_last_error() gives a thread-local message owned by the library.
 * No exception crosses this boundary.  The library never frees caller memory and keeps no caller pointer after
 * a call returns.  "HOST" / "DEVICE" below say where a pointer must live.  FP64 throughout.
 */
#ifndef FE_CHEB_H
#define FE_CHEB_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define FE_OK 0
#define FE_ERR_INVALID (-1) /* bad argument */
#define FE_ERR_NOMEM (-2)   /* host or device allocation failed */
#define FE_ERR_CUDA (-3)    /* CUDA runtime error (message in fe_last_error) */
#define FE_ERR_STATE (-4)   /* e.g. apply before fe_set_potential */

typedef struct fe_mesh fe_mesh; /* opaque; owns all device tables; one stream at a time per handle */

/* Mesh of the box [xe[0],xe[cx]] x [ye[0],ye[cy]] x [ze[0],ze[cz]] (HOST arrays of cx+1, cy+1, cz+1 strictly
 * increasing edges), Lagrange order p in 1..8 on GLL nodes.  Numbering (R3), x fastest everywhere:
 *   cell e = ex + cx*(ey + cy*ez);  local node a = ax + n*(ay + n*az), n = p+1;
 *   global node g = (ex*p+ax) + Nx*((ey*p+ay) + Ny*(ez*p+az)), Nd = cd*p+1;  quadrature point q = qx + n*(qy + n*qz).
 * Builds the 1-D tables, the lumped mass (l.185), M^{-1/2} and the Dirichlet mask on cuda_device.  Synchronous. */
int fe_mesh_create(const double* xe, int cx, const double* ye, int cy, const double* ze, int cz, int p,
                   int cuda_device, fe_mesh** out);
int fe_mesh_destroy(fe_mesh* m);

int64_t fe_num_nodes(const fe_mesh* m); /* N = Nx*Ny*Nz */
int64_t fe_num_free(const fe_mesh* m);  /* (Nx-2)(Ny-2)(Nz-2) unconstrained nodes (R14: the "DoF" of the metric) */
int64_t fe_num_cells(const fe_mesh* m);
int fe_nodes_per_cell(const fe_mesh* m); /* n^3 */
int fe_quad_per_cell(const fe_mesh* m);  /* n_q^3, n_q = p+1 */

/* Parity accessors: fill caller-allocated HOST arrays.  Synchronous. */
int fe_get_l2g(const fe_mesh* m, int32_t* l2g);            /* cells*n^3, R3 */
int fe_get_node_coords(const fe_mesh* m, double* xyz);     /* N*3, R4 */
int fe_get_quad_coords(const fe_mesh* m, double* xyz);     /* cells*n_q^3*3: where the caller evaluates V */
int fe_get_mass(const fe_mesh* m, double* Mdiag);          /* N, diagonal of the GLL-lumped M (l.185) */
int fe_get_dirichlet_mask(const fe_mesh* m, uint8_t* mask); /* N, 1 = free, 0 = boundary */

/* General hexahedral mesh with hanging nodes (the adaptively refined meshes of l.151, l.273, Fig. 6): the leaves of an
 * octree refinement of a cx x cy x cz root grid.  cells: HOST, ncells rows (level, ix, iy, iz) -- leaf (ix, iy, iz) of the
 * level-`level` lattice of 2^level (cx, cy, cz) cells; levels of leaves whose closures touch may differ by at most one.
 * verts: HOST, ncells*8*3 corner coordinates, corner v = vx + 2*(vy + 2*vz); a cell is the trilinear image of [-1,1]^3, so
 * the metric is a full symmetric 3x3 matrix per quadrature point -- unless EVERY cell is an axis-aligned box (the leaves of an
 * octree refinement of an undeformed box, the paper's meshes): the library detects that from the corners and, for p <= 7, runs the
 * 10-sweep box-cell kernel instead of the generic 12-sweep one (same results to rounding; fe_set_variant(m, 9) forces the generic
 * kernel).  Corners shared by cells must coincide and a corner hanging
 * on a coarser neighbour must lie on that neighbour's edge / face (not checked).  Numbering (reading R23): cells in the
 * given order, local nodes a = ax + n*(ay + n*az); unconstrained nodes get ids 0..N-1 in order of first appearance, hanging
 * nodes (nodes of a cell lying on a coarser leaf) ids N..N_all-1 likewise.  Blocks X, Y have N = fe_num_nodes rows: hanging
 * nodes are no degrees of freedom, their values are u_h = sum_k c_hk u_k (fe_get_constraints).  Lumped mass of the
 * constrained problem: diag(C^T m) with m the GLL-quadrature nodal masses (R25).  Dirichlet on the surface of the root box.
 * On such a handle fe_set_potential, fe_apply_H, cheb_filter, cheb_filter_host, fe_rayleigh_ritz, fe_ritz_residuals,
 * fe_chfsi, fe_lanczos_bounds, fe_minres_shifted, fe_gram, fe_add_subspace, fe_density and fe_apply_potential work as on a
 * box mesh (the MINRES preconditioner is M_c,ii / d_i with d_i = kd_i + sum_h C_hi^2 kd_h, kd the diagonal of the assembled
 * 1/2 K over all nodes, reading R27; psi at the quadrature points uses the hanging values u_h = sum_k c_hk u_k).  FE_ERR_INVALID for an inconsistent leaf list.  cuda_device = -1 builds the
 * tables only (sizes, l2g, constraints, coordinates, mass, mask can be queried; no potential can be set).  Synchronous. */
int fe_mesh_create_general(int cx, int cy, int cz, const int32_t* cells, int64_t ncells, const double* verts, int p,
                           int cuda_device, fe_mesh** out);
int64_t fe_num_all_nodes(const fe_mesh* m);          /* N_all: rows of fe_get_node_coords, range of fe_get_l2g */
int64_t fe_num_constraint_entries(const fe_mesh* m); /* non-zeros of the hanging rows */
/* Hanging-node constraints as CSR over the rows h = N..N_all-1: row_ptr (HOST, N_all-N+1 int64), col (unconstrained node
 * ids), val (weights).  A box mesh has none (row_ptr[0] = 0). */
int fe_get_constraints(const fe_mesh* m, int64_t* row_ptr, int32_t* col, double* val);

/* V = v_H + v_N + v_xc (l.68) at the quadrature points: Vq_dev is a DEVICE array of cells*n_q^3 doubles, cell-major,
 * q = qx + n_q*(qy + n_q*qz) inside a cell.  The library stores J*w_q*V_q in its own buffer (one kernel on
 * cuda_stream); `copy` is accepted for ABI stability and ignored: Vq_dev is never retained.  Asynchronous. */
int fe_set_potential(fe_mesh* m, const double* Vq_dev, int copy, void* cuda_stream);

/* Y = H~ X (eps_dev == NULL) or Y[:,j] = (H~ - eps_dev[j] I) X[:,j] (Eq. 20; the shift multiplies the identity of the
 * standard form, R18).  X, Y: DEVICE, N*B doubles, X[a*B+j]; must not overlap.  eps_dev: DEVICE, B doubles.
 * Boundary rows of X are ignored (treated as 0); boundary rows of Y are written 0 (R5).  B >= 1.
 * Asynchronous on cuda_stream. */
int fe_apply_H(fe_mesh* m, const double* X, double* Y, int B, const double* eps_dev, void* cuda_stream);

/* fe_apply_H for a CHAIN of applies into alternating blocks (the operator inside a Krylov iteration, l.221-225; BASELINE
 * config 5): the result is the same Y, but the zero-fill that fe_apply_H needs in front of every call is taken over by the
 * previous call -- while this call computes Y it also clears Ynext (DEVICE, N*B doubles, may be NULL), the block the caller
 * will pass as Y next time, through the store path of the operator kernel.  y_is_clear != 0 promises that Y was cleared that
 * way (or is all zero) and has not been written since; with y_is_clear == 0 the call clears Y itself like fe_apply_H.
 * X, Y, Ynext must not overlap.  Asynchronous on cuda_stream. */
int fe_apply_H_chain(fe_mesh* m, const double* X, double* Y, double* Ynext, int B, const double* eps_dev, int y_is_clear,
                     void* cuda_stream);

/* Chebyshev filter of ChFSI (l.208-210), in place, by the scaled three-term recurrence (R7):
 *   e=(b-a)/2, c=(b+a)/2, s1=e/(a0-c);  Y1=(s1/e)(H~-c)X;  s_{k+1}=1/(2/s1-s_k);
 *   Y_{k+1} = (2 s_{k+1}/e)(H~-c)Y_k - s_k s_{k+1} Y_{k-1};   X <- Y_m  (= T_m((H~-c)/e) X / T_m((a0-c)/e)).
 * Requires a0 < a < b and m >= 1.  work: DEVICE, 2*N*B doubles, caller-owned, must not overlap X.
 * Each step is one fused operator launch (no separate axpy kernels).  Asynchronous on cuda_stream. */
int cheb_filter(fe_mesh* m, double* X, int B, int deg, double a, double b, double a0, double* work,
                void* cuda_stream);

/* The same filter end to end from a HOST block (N*B doubles, X[a*B+j], filtered in place; pinned memory makes the
 * copies asynchronous): host->device copy, cheb_filter, device->host copy.  Columns are independent, so for B a
 * multiple of 32 (B > 32) chunks of 32 columns are pipelined on two internal streams and the PCIe transfers of one
 * chunk overlap the filter of the other (box meshes at p >= 6: the first and the last chunk are 16 columns wide, which halves
 * the copy-in and copy-out that nothing can overlap).  The device staging (3*N*min(B,64) doubles) lives in the handle.
 * SYNCHRONOUS: returns when X_host holds the result.  This is the call bench.py's `e2e` times. */
int cheb_filter_host(fe_mesh* m, double* X_host, int B, int deg, double a, double b, double a0);

/* Rayleigh-Ritz step of ChFSI in span(Y) (Eq. 23-24 l.210-219; R8: H~_Y = Y^T H~ Y; R9: the Cholesky of Y^T Y is
 * done twice, CholQR2):  S = Y^T Y = L L^T, Q = Y L^{-T} (twice);  G = Q^T H~ Q;  G v = theta v;  Y <- Q V.
 * Y: DEVICE, N*B doubles, in: filtered block (Dirichlet rows ignored), out: Ritz vectors (orthonormal columns, Ritz
 * values ascending).  theta_host: HOST, B doubles.  work: DEVICE, N*B doubles, must not overlap Y.  1 <= B <= 128.
 * The tall-skinny products (Gram matrices, rotations) and H~ Q run on the device; the B x B Cholesky and the
 * symmetric eigenproblem run on the host.  SYNCHRONOUS: returns after cuda_stream has drained.
 * FE_ERR_STATE if Y^T Y is not numerically positive definite. */
int fe_rayleigh_ritz(fe_mesh* m, double* Y, int B, double* theta_host, double* work, void* cuda_stream);

/* Block preconditioned MINRES for the adjoint systems (l.221-225):  (H~ - eps_j I) x_j = g_j  for j = 0..B-1 (Eq. 20,
 * l.183), every column with its own Paige-Saunders recurrences, all columns advancing together so that a Krylov
 * step is ONE fused fe_apply_H launch with per-column shifts.  Starts from x = 0; Dirichlet rows of G are ignored and
 * those of X are 0.  When g_j is orthogonal to the null vectors of a singular (H~ - eps_j I), so is the Krylov space
 * and the result is the component p_perp of l.223; the component along the null vectors (Eq. 8) is added with
 * fe_add_subspace.  precondition != 0: inverse diagonal of the mass-scaled negative Laplacian
 * 1/diag(M^{-1/2} (1/2 K) M^{-1/2}) (l.225, positive definite); 0: identity.
 * A column stops when its (preconditioned) residual estimate phibar_j <= tol * beta1_j; the call stops when all have,
 * or after maxit steps (checked every 8 steps: this call synchronises the stream).
 * G: DEVICE N*B (read only); X: DEVICE N*B (out); eps_dev: DEVICE B doubles or NULL; work: DEVICE 6*N*B doubles;
 * relres_host: HOST B doubles (phibar_j / beta1_j at exit) or NULL; iters_host: HOST int or NULL.  1 <= B <= 128. */
int fe_minres_shifted(fe_mesh* m, const double* G, double* X, int B, const double* eps_dev, int maxit, double tol,
                      int precondition, double* relres_host, int* iters_host, double* work, void* cuda_stream);

/* C = A^T Bm (B x B, row-major, HOST) of two DEVICE N x B blocks: the tall-skinny Gram product of Eq. 23 (Y^T Y,
 * Y^T H~ Y) and of the projections Psi^T P of the adjoint solve.  All N rows take part.  Synchronous. */
int fe_gram(fe_mesh* m, const double* A, const double* Bm, int B, double* C_host, void* cuda_stream);

/* fe_gram for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same product with the same kernels, but the B x B device accumulator is a file-scope static __device__
 * array of the library (128 x 128 doubles = 128 KB, held by every GPU that loads the library until exit) instead of a
 * cudaMalloc'ed buffer of the mesh.  The call itself never calls cudaMalloc, cudaFree or an allocating library routine.
 * Arguments as fe_gram: A, Bm DEVICE N*B (read only), C_host HOST B*B doubles (out, row-major).  1 <= B <= 128: a larger
 * B is rejected with FE_ERR_INVALID (the accumulator cannot hold it).  Synchronous (the stream is synchronised before
 * return).  ALL calls on one GPU share the accumulator: each call clears the B*B entries it uses first, and calls that
 * overlap on the GPU (two streams, two host threads) race on it -- serialise them. */
int fe_gram_static(fe_mesh* m, const double* A, const double* Bm, int B, double* C_host, void* cuda_stream);

/* P <- P + Psi D  (N x B block times a HOST B x B row-major matrix D): the completion p = p_perp + Psi~_k d_k of
 * l.223.  Psi, P: DEVICE N*B, must not overlap.  Synchronous. */
int fe_add_subspace(fe_mesh* m, const double* Psi, const double* D_host, double* P, int B, void* cuda_stream);

/* Electron density at the quadrature points (Eq. 4 l.73-77):  rho[e][q] = sum_j f[j] psi_j(x_q)^2 with
 * psi_j = M^{-1/2} psi~_j (the API vectors are psi~ = M^{1/2} psi, Eq. 19; Dirichlet rows count as 0), in the layout of
 * fe_set_potential's Vq (cells*n_q^3, cell-major, q = qx + n_q*(qy + n_q*qz)).  X: DEVICE N*B; f_dev: DEVICE B
 * occupancies; rho_dev: DEVICE cells*n_q^3 doubles (overwritten).  Asynchronous on cuda_stream. */
int fe_density(fe_mesh* m, const double* X, int B, const double* f_dev, double* rho_dev, void* cuda_stream);

/* Spectral bounds for the filter window (reading R10; BASELINE.json config 1 "bounds from 20 Lanczos steps"): k Lanczos
 * steps on H~ (free rows) from the start vector v0 (DEVICE, N doubles, Dirichlet rows ignored, normalised inside),
 * no re-orthogonalisation.  out3_host (HOST, 3 doubles) = {theta_min, theta_max, beta_k} of the k x k tridiagonal
 * matrix; the caller takes b = theta_max + beta_k, a0 = theta_min.  work: DEVICE, 3*N doubles.  1 <= k <= 128.
 * Synchronous (two inner products per step come back to the host). */
int fe_lanczos_bounds(fe_mesh* m, const double* v0_dev, int k, double* out3_host, double* work, void* cuda_stream);

/* Potential-only operator  Y = M^{-1/2} M_U M^{-1/2} X,  (M_U)_ab = int N_a U N_b  with the field U given at the
 * quadrature points like V (DEVICE, cells*n_q^3), without touching the potential set by fe_set_potential.  It is the
 * integral of the adjoint right-hand side (Eq. 18, l.174-177) with U = 4 w (rho_data - rho):
 *   g~ = [M^{-1/2} M_U M^{-1/2} Psi~] diag(f) - Psi~ (D + D^T)
 * (the second term is fe_add_subspace; the lumped GLL mass makes M^{-1/2} M M^{-1/2} the identity).  X, Y: DEVICE N*B,
 * no overlap; Dirichlet rows ignored / written 0.  Runs the legacy kernel with the stiffness switched off.  Asynchronous. */
int fe_apply_potential(fe_mesh* m, const double* Uq_dev, const double* X, double* Y, int B, void* cuda_stream);

/* Kernel variant for experiments and tests: 0 = default (TMA generation when B is even and the blocks are 16-byte
 * aligned, else the legacy atomics kernel), 3 = legacy kernel always, 4 = legacy kernel with a colour-ordered
 * scatter (the 8 parity classes of the cell grid launched in order: cells of one class share no node, so every sum
 * has a fixed order and results are bit-reproducible; slower; on a general mesh: cells coloured greedily so that no two
 * cells of a colour share a node, launched colour by colour, hanging contributions collapsed over the transposed constraint
 * rows), 5..8 = launch shapes of the TMA kernel (fe_apply_tma.cuh; test and experiment hooks), 9 = on a general mesh whose
 * cells are all axis-aligned boxes: the generic 12-sweep cell kernel instead of the 10-sweep box-cell kernel (cross-check).
 * FE_ERR_INVALID if unknown. */
int fe_set_variant(fe_mesh* m, int variant);
/* Kernels launched by this handle since creation (bench.py's gpu_launches). */
int64_t fe_launch_count(const fe_mesh* m);

/* Ritz residual norms  res[j] = || H~ x_j - theta_j x_j ||_2  over the free rows, for a block X (DEVICE, N*B) and B values
 * theta_host (HOST): the quantity the eigensolver tolerance t_eig of l.296 is applied to.  One fused shifted apply
 * (Eq. 20 with eps = theta) plus one column reduction.  res_host: HOST, B doubles.  work: DEVICE, N*B doubles, must not
 * overlap X.  1 <= B <= 128.  Synchronous. */
int fe_ritz_residuals(fe_mesh* m, const double* X, const double* theta_host, int B, double* res_host, double* work,
                      void* cuda_stream);

/* Chebyshev-filtered subspace iteration driven by the residual (l.208-219, l.296): repeat { cheb_filter of degree deg on
 * the window (a0, a, b); fe_rayleigh_ritz; fe_ritz_residuals } until the residual norms of the n_gate lowest Ritz pairs
 * (the occupied states) are all <= t_eig, or max_cycles cycles have run.  The paper sets t_eig = e_L2^2 / c_eig from the
 * density error of the previous outer iteration (c_eig = 100 by default); the caller passes the number.  After every
 * cycle the window becomes a = largest, a0 = smallest Ritz value of the block; b (an upper bound of the spectrum, e.g.
 * from fe_lanczos_bounds) is kept.  X: DEVICE N*B, in: start block, out: Ritz vectors.  theta_host, res_host: HOST, B
 * doubles of the last cycle.  cycles_host: HOST int or NULL.  work: DEVICE 2*N*B doubles.  Synchronous.
 * FE_ERR_STATE if the Ritz values leave (a0, b). */
int fe_chfsi(fe_mesh* m, double* X, int B, int deg, double a, double b, double a0, double t_eig, int n_gate,
             int max_cycles, double* theta_host, double* res_host, int* cycles_host, double* work, void* cuda_stream);

/* Step-0 ceilings of the device (not on the product path): a diagnostic kernel of the given
 * kind is launched back to back for at least min_seconds (0 < min_seconds <= 30) and the best launch is reported in
 * *value_host (HOST):  kind 0 = register-resident DFMA chains, TFLOP/s (the FP64 pipe that bounds fe_apply_H / cheb_filter);
 * 1 = mma.sync.m8n8k4.f64 chains, TFLOP/s (the FP64 tensor path; tcgen05 has no FP64 kind);  2 = y = a x + z over 1 GiB
 * arrays, GB/s of the two reads and one write (the 24 B per node-vector of a filter step);  3 = cp.reduce.async.bulk
 * .add.f64 shared -> global, GB/s of payload (the scatter of the TMA kernel);  4 = red.global.add.f64, GB/s of payload (the
 * scatter of the legacy kernel).  Allocates and frees its own buffers (up to 3 GiB).  Synchronous. */
int fe_diag_peak(int cuda_device, int kind, double min_seconds, double* value_host);

const char* fe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
