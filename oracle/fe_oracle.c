/*
 * fe_oracle.c -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).  See fe_oracle.h.
 *
 * Everything here is the plain definition written out: 1-D rules by Newton on Legendre polynomials,
 * Lagrange polynomials by the literal product formula (Eq. 12, l.124), cell matrices by an
 * explicit loop over all 3-D quadrature points (Eq. 17, l.171; no sum factorisation), lumped GLL mass
 * (l.185), assembled CSR, H~ = M^{-1/2} H M^{-1/2} (Eq. 19), serial three-term Chebyshev recurrence
 * (l.208-210, reading R7).  No blocking, fusion or reordering.  FP64 throughout (long double only
 * inside the Newton iterations of the 1-D rules so that their doubles are correctly rounded).
 */
#include "fe_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct orc_mesh {
    int p, n, nq, cx, cy, cz, nc;
    int64_t Nx, Ny, Nz, N, ncells;
    double *xe, *ye, *ze;
    double *gll_x, *gll_w, *gl_x, *gl_w;
    double *phi;  /* phi[q*n+a]  = l_a(gl_x[q])   (Eq. 12 at the Gauss points) */
    double *dphi; /* dphi[q*n+a] = l_a'(gl_x[q]) */
    double *mass; /* N */
    uint8_t *mask; /* N */
};

struct orc_csr {
    int64_t nrows, nnz;
    int64_t *row_ptr;
    int32_t *col;
    double *val;
};

/* Legendre P_k(x) and P_k'(x) by the three-term recurrence (textbook) */
static void legendre(int k, long double x, long double* P, long double* dP)
{
    long double p0 = 1.0L, p1 = x;
    if (k == 0) { *P = 1.0L; *dP = 0.0L; return; }
    for (int j = 2; j <= k; ++j) {
        long double pj = ((2 * j - 1) * x * p1 - (j - 1) * p0) / j;
        p0 = p1; p1 = pj;
    }
    *P = p1;
    /* (1-x^2) P_k' = k (P_{k-1} - x P_k) */
    /* P_k'(+-1) = (+-1)^{k+1} k(k+1)/2 */
    *dP = (fabsl(x) == 1.0L) ? 0.5L * k * (k + 1) * ((x > 0 || k % 2 == 1) ? 1.0L : -1.0L)
                             : k * (p0 - x * p1) / (1.0L - x * x);
}

int orc_gll(int p, double* x, double* w)
{
    /* nodes: +-1 and the roots of P_p'; weights 2/(p(p+1) P_p(x)^2)  (survey 8(c) step 1) */
    if (p < 1) return -1;
    const long double PI = 3.141592653589793238462643383279502884L;
    for (int i = 0; i <= p; ++i) {
        long double xi;
        if (i == 0) xi = -1.0L;
        else if (i == p) xi = 1.0L;
        else {
            xi = -cosl(PI * i / p); /* Chebyshev-Gauss-Lobatto start */
            for (int it = 0; it < 200; ++it) {
                /* Newton on f = P_p'(x);  f' = P_p'' = (2x P_p' - p(p+1) P_p)/(1-x^2) */
                long double P, dP;
                legendre(p, xi, &P, &dP);
                long double d2P = (2.0L * xi * dP - (long double)p * (p + 1) * P) / (1.0L - xi * xi);
                long double dx = dP / d2P;
                xi -= dx;
                if (fabsl(dx) < 1e-19L) break;
            }
        }
        long double P, dP;
        legendre(p, xi, &P, &dP);
        x[i] = (double)xi;
        w[i] = (double)(2.0L / ((long double)p * (p + 1) * P * P));
    }
    /* enforce exact symmetry of the stored doubles */
    for (int i = 0; i < (p + 1) / 2; ++i) {
        x[p - i] = -x[i];
        w[p - i] = w[i];
    }
    if (p % 2 == 0) x[p / 2] = 0.0;
    return 0;
}

int orc_gauss(int nq, double* x, double* w)
{
    /* roots of P_nq; weights 2/((1-x^2) P_nq'(x)^2) */
    if (nq < 1) return -1;
    const long double PI = 3.141592653589793238462643383279502884L;
    for (int i = 0; i < nq; ++i) {
        long double xi = -cosl(PI * (i + 0.75L) / (nq + 0.5L));
        long double P, dP;
        for (int it = 0; it < 200; ++it) {
            legendre(nq, xi, &P, &dP);
            long double dx = P / dP;
            xi -= dx;
            if (fabsl(dx) < 1e-19L) break;
        }
        legendre(nq, xi, &P, &dP);
        x[i] = (double)xi;
        w[i] = (double)(2.0L / ((1.0L - xi * xi) * dP * dP));
    }
    for (int i = 0; i < nq / 2; ++i) {
        x[nq - 1 - i] = -x[i];
        w[nq - 1 - i] = w[i];
    }
    if (nq % 2 == 1) x[nq / 2] = 0.0;
    return 0;
}

double orc_lagrange(int n, const double* nodes, int a, double x)
{
    double v = 1.0;
    for (int j = 0; j < n; ++j)
        if (j != a) v *= (x - nodes[j]) / (nodes[a] - nodes[j]);
    return v;
}

double orc_lagrange_deriv(int n, const double* nodes, int a, double x)
{
    /* product rule on Eq. 12: sum_k 1/(x_a-x_k) prod_{j!=a,k} (x-x_j)/(x_a-x_j) */
    double s = 0.0;
    for (int k = 0; k < n; ++k) {
        if (k == a) continue;
        double t = 1.0 / (nodes[a] - nodes[k]);
        for (int j = 0; j < n; ++j)
            if (j != a && j != k) t *= (x - nodes[j]) / (nodes[a] - nodes[j]);
        s += t;
    }
    return s;
}

/* R3 numbering */
static inline int64_t node_id(const orc_mesh* m, int ex, int ey, int ez, int ax, int ay, int az)
{
    int64_t gx = (int64_t)ex * m->p + ax, gy = (int64_t)ey * m->p + ay, gz = (int64_t)ez * m->p + az;
    return gx + m->Nx * (gy + m->Ny * gz);
}
static inline void cell_xyz(const orc_mesh* m, int64_t e, int* ex, int* ey, int* ez)
{
    *ex = (int)(e % m->cx);
    *ey = (int)((e / m->cx) % m->cy);
    *ez = (int)(e / ((int64_t)m->cx * m->cy));
}
/* R4 coordinates */
static inline double map_coord(const double* edges, int ec, double xi, int is_last)
{
    if (is_last) return edges[ec + 1];
    return edges[ec] + 0.5 * (xi + 1.0) * (edges[ec + 1] - edges[ec]);
}

orc_mesh* orc_mesh_create(const double* xe, int cx, const double* ye, int cy, const double* ze, int cz, int p)
{
    if (p < 1 || cx < 1 || cy < 1 || cz < 1) return NULL;
    orc_mesh* m = (orc_mesh*)calloc(1, sizeof(orc_mesh));
    m->p = p; m->n = p + 1; m->nq = p + 1; m->cx = cx; m->cy = cy; m->cz = cz;
    m->nc = m->n * m->n * m->n;
    m->Nx = (int64_t)cx * p + 1; m->Ny = (int64_t)cy * p + 1; m->Nz = (int64_t)cz * p + 1;
    m->N = m->Nx * m->Ny * m->Nz;
    m->ncells = (int64_t)cx * cy * cz;
    m->xe = (double*)malloc((cx + 1) * sizeof(double)); memcpy(m->xe, xe, (cx + 1) * sizeof(double));
    m->ye = (double*)malloc((cy + 1) * sizeof(double)); memcpy(m->ye, ye, (cy + 1) * sizeof(double));
    m->ze = (double*)malloc((cz + 1) * sizeof(double)); memcpy(m->ze, ze, (cz + 1) * sizeof(double));
    int n = m->n, nq = m->nq;
    m->gll_x = (double*)malloc(n * sizeof(double)); m->gll_w = (double*)malloc(n * sizeof(double));
    m->gl_x = (double*)malloc(nq * sizeof(double)); m->gl_w = (double*)malloc(nq * sizeof(double));
    orc_gll(p, m->gll_x, m->gll_w);
    orc_gauss(nq, m->gl_x, m->gl_w);
    m->phi = (double*)malloc((size_t)nq * n * sizeof(double));
    m->dphi = (double*)malloc((size_t)nq * n * sizeof(double));
    for (int q = 0; q < nq; ++q)
        for (int a = 0; a < n; ++a) {
            m->phi[q * n + a] = orc_lagrange(n, m->gll_x, a, m->gl_x[q]);
            m->dphi[q * n + a] = orc_lagrange_deriv(n, m->gll_x, a, m->gl_x[q]);
        }
    /* lumped mass: M_gg += J w_ax w_ay w_az over the cells touching g (l.185; survey 8(c) step 4) */
    m->mass = (double*)calloc((size_t)m->N, sizeof(double));
    m->mask = (uint8_t*)malloc((size_t)m->N);
    for (int64_t e = 0; e < m->ncells; ++e) {
        int ex, ey, ez; cell_xyz(m, e, &ex, &ey, &ez);
        double hx = m->xe[ex + 1] - m->xe[ex], hy = m->ye[ey + 1] - m->ye[ey], hz = m->ze[ez + 1] - m->ze[ez];
        double J = hx * hy * hz / 8.0;
        for (int az = 0; az < n; ++az)
            for (int ay = 0; ay < n; ++ay)
                for (int ax = 0; ax < n; ++ax)
                    m->mass[node_id(m, ex, ey, ez, ax, ay, az)] += J * m->gll_w[ax] * m->gll_w[ay] * m->gll_w[az];
    }
    for (int64_t gz = 0; gz < m->Nz; ++gz)
        for (int64_t gy = 0; gy < m->Ny; ++gy)
            for (int64_t gx = 0; gx < m->Nx; ++gx) {
                int bnd = (gx == 0 || gx == m->Nx - 1 || gy == 0 || gy == m->Ny - 1 || gz == 0 || gz == m->Nz - 1);
                m->mask[gx + m->Nx * (gy + m->Ny * gz)] = bnd ? 0 : 1;
            }
    return m;
}

void orc_mesh_destroy(orc_mesh* m)
{
    if (!m) return;
    free(m->xe); free(m->ye); free(m->ze); free(m->gll_x); free(m->gll_w); free(m->gl_x); free(m->gl_w);
    free(m->phi); free(m->dphi); free(m->mass); free(m->mask); free(m);
}

int64_t orc_num_nodes(const orc_mesh* m) { return m->N; }
int64_t orc_num_free(const orc_mesh* m) { return (m->Nx - 2) * (m->Ny - 2) * (m->Nz - 2); }
int64_t orc_num_cells(const orc_mesh* m) { return m->ncells; }
int orc_nodes_per_cell(const orc_mesh* m) { return m->nc; }
int orc_quad_per_cell(const orc_mesh* m) { return m->nq * m->nq * m->nq; }

void orc_get_l2g(const orc_mesh* m, int32_t* l2g)
{
    int n = m->n;
    for (int64_t e = 0; e < m->ncells; ++e) {
        int ex, ey, ez; cell_xyz(m, e, &ex, &ey, &ez);
        for (int az = 0; az < n; ++az)
            for (int ay = 0; ay < n; ++ay)
                for (int ax = 0; ax < n; ++ax)
                    l2g[e * m->nc + ax + n * (ay + n * az)] = (int32_t)node_id(m, ex, ey, ez, ax, ay, az);
    }
}

void orc_get_node_coords(const orc_mesh* m, double* xyz)
{
    int n = m->n, p = m->p;
    for (int64_t e = 0; e < m->ncells; ++e) {
        int ex, ey, ez; cell_xyz(m, e, &ex, &ey, &ez);
        for (int az = 0; az < n; ++az)
            for (int ay = 0; ay < n; ++ay)
                for (int ax = 0; ax < n; ++ax) {
                    int64_t g = node_id(m, ex, ey, ez, ax, ay, az);
                    xyz[3 * g + 0] = map_coord(m->xe, ex, m->gll_x[ax], ax == p);
                    xyz[3 * g + 1] = map_coord(m->ye, ey, m->gll_x[ay], ay == p);
                    xyz[3 * g + 2] = map_coord(m->ze, ez, m->gll_x[az], az == p);
                }
    }
}

void orc_get_quad_coords(const orc_mesh* m, double* xyz)
{
    int nq = m->nq;
    int64_t nq3 = (int64_t)nq * nq * nq;
    for (int64_t e = 0; e < m->ncells; ++e) {
        int ex, ey, ez; cell_xyz(m, e, &ex, &ey, &ez);
        for (int qz = 0; qz < nq; ++qz)
            for (int qy = 0; qy < nq; ++qy)
                for (int qx = 0; qx < nq; ++qx) {
                    int64_t q = e * nq3 + qx + nq * (qy + nq * qz);
                    xyz[3 * q + 0] = map_coord(m->xe, ex, m->gl_x[qx], 0);
                    xyz[3 * q + 1] = map_coord(m->ye, ey, m->gl_x[qy], 0);
                    xyz[3 * q + 2] = map_coord(m->ze, ez, m->gl_x[qz], 0);
                }
    }
}

void orc_get_mass(const orc_mesh* m, double* Mdiag) { memcpy(Mdiag, m->mass, (size_t)m->N * sizeof(double)); }
void orc_get_mask(const orc_mesh* m, uint8_t* mask) { memcpy(mask, m->mask, (size_t)m->N); }

/* one entry of Eq. 17 restricted to cell e, by explicit 3-D quadrature */
static double cell_entry(const orc_mesh* m, double hx, double hy, double hz, const double* Vq_cell,
                         double kin, double pot, int a, int b)
{
    int n = m->n, nq = m->nq;
    int ax = a % n, ay = (a / n) % n, az = a / (n * n);
    int bx = b % n, by = (b / n) % n, bz = b / (n * n);
    double J = hx * hy * hz / 8.0;
    double sum = 0.0;
    for (int qz = 0; qz < nq; ++qz)
        for (int qy = 0; qy < nq; ++qy)
            for (int qx = 0; qx < nq; ++qx) {
                double wq = J * m->gl_w[qx] * m->gl_w[qy] * m->gl_w[qz];
                double pax = m->phi[qx * n + ax], pay = m->phi[qy * n + ay], paz = m->phi[qz * n + az];
                double pbx = m->phi[qx * n + bx], pby = m->phi[qy * n + by], pbz = m->phi[qz * n + bz];
                double dax = m->dphi[qx * n + ax], day = m->dphi[qy * n + ay], daz = m->dphi[qz * n + az];
                double dbx = m->dphi[qx * n + bx], dby = m->dphi[qy * n + by], dbz = m->dphi[qz * n + bz];
                /* physical gradients: d/dx = (2/hx) d/dxi */
                double gax = (2.0 / hx) * dax * pay * paz, gay = (2.0 / hy) * pax * day * paz, gaz = (2.0 / hz) * pax * pay * daz;
                double gbx = (2.0 / hx) * dbx * pby * pbz, gby = (2.0 / hy) * pbx * dby * pbz, gbz = (2.0 / hz) * pbx * pby * dbz;
                double Pa = pax * pay * paz, Pb = pbx * pby * pbz;
                double V = Vq_cell ? Vq_cell[qx + nq * (qy + nq * qz)] : 0.0;
                sum += wq * (kin * (gax * gbx + gay * gby + gaz * gbz) + pot * V * Pa * Pb);
            }
    return sum;
}

void orc_cell_matrix(const orc_mesh* m, int64_t e, const double* Vq_cell, double kin, double pot, double* He)
{
    int ex, ey, ez; cell_xyz(m, e, &ex, &ey, &ez);
    double hx = m->xe[ex + 1] - m->xe[ex], hy = m->ye[ey + 1] - m->ye[ey], hz = m->ze[ez + 1] - m->ze[ez];
    for (int a = 0; a < m->nc; ++a)
        for (int b = 0; b < m->nc; ++b)
            He[(size_t)a * m->nc + b] = cell_entry(m, hx, hy, hz, Vq_cell, kin, pot, a, b);
}

void orc_build_cell_matrices(const orc_mesh* m, const double* Vq, double* He_all)
{
    int64_t nq3 = orc_quad_per_cell(m);
    size_t nc2 = (size_t)m->nc * m->nc;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t e = 0; e < m->ncells; ++e)
        orc_cell_matrix(m, e, Vq + e * nq3, 0.5, 1.0, He_all + (size_t)e * nc2);
}

/* ---- assembled CSR: H = sum_e P_e^T H_e P_e ------------------------------------------------------------ */
typedef struct { int32_t col; double val; } entry_t;
static int cmp_entry(const void* x, const void* y)
{
    int32_t a = ((const entry_t*)x)->col, b = ((const entry_t*)y)->col;
    return (a > b) - (a < b);
}

orc_csr* orc_assemble(const orc_mesh* m, const double* He_all, int scaled)
{
    int n = m->n, nc = m->nc, p = m->p;
    orc_csr* A = (orc_csr*)calloc(1, sizeof(orc_csr));
    A->nrows = m->N;
    A->row_ptr = (int64_t*)calloc((size_t)m->N + 1, sizeof(int64_t));
    /* two passes over the rows: count, then fill.  For row g, visit every cell that contains g. */
    entry_t* buf = (entry_t*)malloc((size_t)8 * nc * sizeof(entry_t));
    for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1) {
            for (int64_t g = 0; g < m->N; ++g) A->row_ptr[g + 1] += A->row_ptr[g];
            A->nnz = A->row_ptr[m->N];
            A->col = (int32_t*)malloc((size_t)A->nnz * sizeof(int32_t));
            A->val = (double*)malloc((size_t)A->nnz * sizeof(double));
        }
        for (int64_t gz = 0; gz < m->Nz; ++gz)
            for (int64_t gy = 0; gy < m->Ny; ++gy)
                for (int64_t gx = 0; gx < m->Nx; ++gx) {
                    int64_t g = gx + m->Nx * (gy + m->Ny * gz);
                    int cnt = 0;
                    /* candidate cells per axis: the cell(s) whose node range contains the index */
                    for (int ez = 0; ez < m->cz; ++ez) {
                        if (gz < (int64_t)ez * p || gz > (int64_t)(ez + 1) * p) continue;
                        for (int ey = 0; ey < m->cy; ++ey) {
                            if (gy < (int64_t)ey * p || gy > (int64_t)(ey + 1) * p) continue;
                            for (int ex = 0; ex < m->cx; ++ex) {
                                if (gx < (int64_t)ex * p || gx > (int64_t)(ex + 1) * p) continue;
                                int64_t e = ex + (int64_t)m->cx * (ey + (int64_t)m->cy * ez);
                                int a = (int)(gx - (int64_t)ex * p) + n * ((int)(gy - (int64_t)ey * p) + n * (int)(gz - (int64_t)ez * p));
                                const double* row = He_all + ((size_t)e * nc + a) * nc;
                                for (int bz = 0; bz < n; ++bz)
                                    for (int by = 0; by < n; ++by)
                                        for (int bx = 0; bx < n; ++bx) {
                                            buf[cnt].col = (int32_t)node_id(m, ex, ey, ez, bx, by, bz);
                                            buf[cnt].val = row[bx + n * (by + n * bz)];
                                            ++cnt;
                                        }
                            }
                        }
                    }
                    qsort(buf, cnt, sizeof(entry_t), cmp_entry);
                    /* merge duplicates (nodes shared by several of the cells) */
                    int64_t k = (pass == 1) ? A->row_ptr[g] : 0;
                    int64_t nuniq = 0;
                    for (int i = 0; i < cnt;) {
                        int j = i; double s = 0.0;
                        while (j < cnt && buf[j].col == buf[i].col) { s += buf[j].val; ++j; }
                        if (pass == 1) {
                            int32_t c = buf[i].col;
                            if (scaled) {
                                /* H~_{gc} = M_gg^{-1/2} H_gc M_cc^{-1/2}; Dirichlet rows/columns zero (R5) */
                                s = (m->mask[g] && m->mask[c]) ? (1.0 / sqrt(m->mass[g])) * s * (1.0 / sqrt(m->mass[c])) : 0.0;
                            }
                            A->col[k] = c; A->val[k] = s; ++k;
                        }
                        ++nuniq; i = j;
                    }
                    if (pass == 0) A->row_ptr[g + 1] = nuniq;
                }
    }
    free(buf);
    return A;
}

void orc_csr_destroy(orc_csr* A)
{
    if (!A) return;
    free(A->row_ptr); free(A->col); free(A->val); free(A);
}
int64_t orc_csr_nnz(const orc_csr* A) { return A->nnz; }
void orc_csr_copy(const orc_csr* A, int64_t* row_ptr, int32_t* col, double* val)
{
    memcpy(row_ptr, A->row_ptr, (size_t)(A->nrows + 1) * sizeof(int64_t));
    memcpy(col, A->col, (size_t)A->nnz * sizeof(int32_t));
    memcpy(val, A->val, (size_t)A->nnz * sizeof(double));
}

void orc_csr_apply(const orc_mesh* m, const orc_csr* A, const double* X, int B, const double* eps, double* Y, int nthreads)
{
    (void)nthreads;
#pragma omp parallel for schedule(static) if (nthreads > 1) num_threads(nthreads > 1 ? nthreads : 1)
    for (int64_t g = 0; g < A->nrows; ++g) {
        double* y = Y + (size_t)g * B;
        for (int j = 0; j < B; ++j) y[j] = 0.0;
        if (!m->mask[g]) continue; /* boundary rows are written 0 (R5) */
        for (int64_t k = A->row_ptr[g]; k < A->row_ptr[g + 1]; ++k) {
            const double* x = X + (size_t)A->col[k] * B;
            double v = A->val[k];
            for (int j = 0; j < B; ++j) y[j] += v * x[j];
        }
        if (eps) {
            const double* x = X + (size_t)g * B;
            for (int j = 0; j < B; ++j) y[j] -= eps[j] * x[j]; /* shift multiplies the identity (Eq. 20) */
        }
    }
}

void orc_cellwise_apply(const orc_mesh* m, const double* He_all, const double* X, int B, const double* eps, double* Y)
{
    int nc = m->nc, n = m->n;
    int32_t* ids = (int32_t*)malloc((size_t)nc * sizeof(int32_t));
    double* xe = (double*)malloc((size_t)nc * B * sizeof(double));
    memset(Y, 0, (size_t)m->N * B * sizeof(double));
    for (int64_t e = 0; e < m->ncells; ++e) {
        int ex, ey, ez; cell_xyz(m, e, &ex, &ey, &ez);
        for (int az = 0; az < n; ++az)
            for (int ay = 0; ay < n; ++ay)
                for (int ax = 0; ax < n; ++ax)
                    ids[ax + n * (ay + n * az)] = (int32_t)node_id(m, ex, ey, ez, ax, ay, az);
        /* gather with S and mask: x_e = mu S X */
        for (int a = 0; a < nc; ++a) {
            int64_t g = ids[a];
            double s = m->mask[g] ? 1.0 / sqrt(m->mass[g]) : 0.0;
            for (int j = 0; j < B; ++j) xe[(size_t)a * B + j] = s * X[(size_t)g * B + j];
        }
        const double* He = He_all + (size_t)e * nc * nc;
        for (int a = 0; a < nc; ++a) {
            double* y = Y + (size_t)ids[a] * B;
            for (int b = 0; b < nc; ++b) {
                double v = He[(size_t)a * nc + b];
                const double* x = xe + (size_t)b * B;
                for (int j = 0; j < B; ++j) y[j] += v * x[j];
            }
        }
    }
    for (int64_t g = 0; g < m->N; ++g) {
        double s = m->mask[g] ? 1.0 / sqrt(m->mass[g]) : 0.0;
        for (int j = 0; j < B; ++j) {
            double v = s * Y[(size_t)g * B + j];
            if (eps && m->mask[g]) v -= eps[j] * X[(size_t)g * B + j];
            Y[(size_t)g * B + j] = v;
        }
    }
    free(ids); free(xe);
}

void orc_apply_rows(const orc_mesh* m, const double* Vq, const double* X, int B, const double* eps,
                    const int64_t* rows, int64_t nrows, double* Yrows)
{
    int n = m->n, p = m->p, nc = m->nc;
    int64_t nq3 = orc_quad_per_cell(m);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t g = rows[r];
        double* y = Yrows + (size_t)r * B;
        for (int j = 0; j < B; ++j) y[j] = 0.0;
        if (!m->mask[g]) continue;
        int64_t gx = g % m->Nx, gy = (g / m->Nx) % m->Ny, gz = g / (m->Nx * m->Ny);
        double sg = 1.0 / sqrt(m->mass[g]);
        for (int ez = 0; ez < m->cz; ++ez) {
            if (gz < (int64_t)ez * p || gz > (int64_t)(ez + 1) * p) continue;
            for (int ey = 0; ey < m->cy; ++ey) {
                if (gy < (int64_t)ey * p || gy > (int64_t)(ey + 1) * p) continue;
                for (int ex = 0; ex < m->cx; ++ex) {
                    if (gx < (int64_t)ex * p || gx > (int64_t)(ex + 1) * p) continue;
                    int64_t e = ex + (int64_t)m->cx * (ey + (int64_t)m->cy * ez);
                    double hx = m->xe[ex + 1] - m->xe[ex], hy = m->ye[ey + 1] - m->ye[ey], hz = m->ze[ez + 1] - m->ze[ez];
                    int a = (int)(gx - (int64_t)ex * p) + n * ((int)(gy - (int64_t)ey * p) + n * (int)(gz - (int64_t)ez * p));
                    for (int b = 0; b < nc; ++b) {
                        int bx = b % n, by = (b / n) % n, bz = b / (n * n);
                        int64_t c = node_id(m, ex, ey, ez, bx, by, bz);
                        if (!m->mask[c]) continue;
                        double h = cell_entry(m, hx, hy, hz, Vq + e * nq3, 0.5, 1.0, a, b);
                        double v = sg * h * (1.0 / sqrt(m->mass[c]));
                        const double* x = X + (size_t)c * B;
                        for (int j = 0; j < B; ++j) y[j] += v * x[j];
                    }
                }
            }
        }
        if (eps) {
            const double* x = X + (size_t)g * B;
            for (int j = 0; j < B; ++j) y[j] -= eps[j] * x[j];
        }
    }
}

int orc_filter(const orc_mesh* m, const orc_csr* A, const double* He_all, double* X, int B, int deg,
               double a, double b, double a0, int nthreads)
{
    /* survey 8(c) step 7 (PAPER.md l.208-210 + reading R7):
     * e=(b-a)/2, c=(b+a)/2, sigma_1 = e/(a0-c);  Y_1 = (sigma_1/e)(H~X - cX);
     * sigma_{k+1} = 1/(2/sigma_1 - sigma_k);  Y_{k+1} = (2 sigma_{k+1}/e)(H~Y_k - cY_k) - sigma_k sigma_{k+1} Y_{k-1}. */
    if (!(a0 < a && a < b) || deg < 1) return -1;
    size_t len = (size_t)m->N * B;
    double* Yk = (double*)malloc(len * sizeof(double));   /* Y_k   */
    double* Ykm = (double*)malloc(len * sizeof(double));  /* Y_{k-1} */
    double* HY = (double*)malloc(len * sizeof(double));
    double e = (b - a) / 2.0, c = (b + a) / 2.0;
    double sigma1 = e / (a0 - c), sigma = sigma1;
    /* Y_0 = X with boundary rows treated as 0 (R5) */
    for (int64_t g = 0; g < m->N; ++g)
        for (int j = 0; j < B; ++j) Ykm[(size_t)g * B + j] = m->mask[g] ? X[(size_t)g * B + j] : 0.0;
    if (A) orc_csr_apply(m, A, Ykm, B, NULL, HY, nthreads); else orc_cellwise_apply(m, He_all, Ykm, B, NULL, HY);
    for (size_t i = 0; i < len; ++i) Yk[i] = (sigma1 / e) * (HY[i] - c * Ykm[i]);
    for (int k = 1; k < deg; ++k) {
        double sigma_next = 1.0 / (2.0 / sigma1 - sigma);
        if (A) orc_csr_apply(m, A, Yk, B, NULL, HY, nthreads); else orc_cellwise_apply(m, He_all, Yk, B, NULL, HY);
        for (size_t i = 0; i < len; ++i) {
            double ynew = (2.0 * sigma_next / e) * (HY[i] - c * Yk[i]) - sigma * sigma_next * Ykm[i];
            Ykm[i] = Yk[i];
            Yk[i] = ynew;
        }
        sigma = sigma_next;
    }
    memcpy(X, Yk, len * sizeof(double));
    free(Yk); free(Ykm); free(HY);
    return 0;
}

/* ---- general hexahedral cell (Eq. 17 l.171 on a trilinearly mapped cell) -------------------
 * The cell is the image of [-1,1]^3 under x(xi) = sum_v X_v T_v(xi), T_v the 8 trilinear corner functions, corner
 * v = vx + 2(vy + 2vz).  Jacobian J_ij = dx_i/dxi_j at every quadrature point; physical gradient grad Phi = J^{-T} grad^ Phi;
 * H_e[a,b] = sum_q w_q |det J_q| [ kin grad Phi_a . grad Phi_b + pot V_q Phi_a Phi_b ], one entry and one point at a time. */
static void trilinear_jacobian(const double* verts, double x, double y, double z, double J[3][3], double pos[3])
{
    double tx[2] = {0.5 * (1.0 - x), 0.5 * (1.0 + x)}, ty[2] = {0.5 * (1.0 - y), 0.5 * (1.0 + y)}, tz[2] = {0.5 * (1.0 - z), 0.5 * (1.0 + z)};
    double dx[2] = {-0.5, 0.5};
    for (int i = 0; i < 3; ++i) { pos[i] = 0.0; for (int j = 0; j < 3; ++j) J[i][j] = 0.0; }
    for (int v = 0; v < 8; ++v) {
        int vx = v & 1, vy = (v >> 1) & 1, vz = v >> 2;
        for (int i = 0; i < 3; ++i) {
            double X = verts[3 * v + i];
            pos[i] += X * tx[vx] * ty[vy] * tz[vz];
            J[i][0] += X * dx[vx] * ty[vy] * tz[vz];
            J[i][1] += X * tx[vx] * dx[vy] * tz[vz];
            J[i][2] += X * tx[vx] * ty[vy] * dx[vz];
        }
    }
}

static double det3(double J[3][3])
{
    return J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0]) +
           J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
}

/* inverse by cofactors: Ji = J^{-1} */
static void inv3(double J[3][3], double det, double Ji[3][3])
{
    Ji[0][0] = (J[1][1] * J[2][2] - J[1][2] * J[2][1]) / det;
    Ji[0][1] = (J[0][2] * J[2][1] - J[0][1] * J[2][2]) / det;
    Ji[0][2] = (J[0][1] * J[1][2] - J[0][2] * J[1][1]) / det;
    Ji[1][0] = (J[1][2] * J[2][0] - J[1][0] * J[2][2]) / det;
    Ji[1][1] = (J[0][0] * J[2][2] - J[0][2] * J[2][0]) / det;
    Ji[1][2] = (J[0][2] * J[1][0] - J[0][0] * J[1][2]) / det;
    Ji[2][0] = (J[1][0] * J[2][1] - J[1][1] * J[2][0]) / det;
    Ji[2][1] = (J[0][1] * J[2][0] - J[0][0] * J[2][1]) / det;
    Ji[2][2] = (J[0][0] * J[1][1] - J[0][1] * J[1][0]) / det;
}

void orc_general_cell_matrix(int p, const double* verts, const double* Vq_cell, double kin, double pot, double* He)
{
    int n = p + 1, nq = p + 1, nc = n * n * n;
    double gx[16], gw[16], qx[16], qw[16];
    orc_gll(p, gx, gw);
    orc_gauss(nq, qx, qw);
    for (int i = 0; i < nc * nc; ++i) He[i] = 0.0;
    double* Pv = (double*)malloc((size_t)nc * sizeof(double));      /* Phi_a at the point */
    double* G = (double*)malloc((size_t)nc * 3 * sizeof(double));   /* physical gradient of Phi_a at the point */
    for (int kz = 0; kz < nq; ++kz)
        for (int ky = 0; ky < nq; ++ky)
            for (int kx = 0; kx < nq; ++kx) {
                double J[3][3], Ji[3][3], pos[3];
                trilinear_jacobian(verts, qx[kx], qx[ky], qx[kz], J, pos);
                double det = det3(J);
                inv3(J, det, Ji);
                double wq = qw[kx] * qw[ky] * qw[kz] * fabs(det);
                double V = Vq_cell ? Vq_cell[kx + nq * (ky + nq * kz)] : 0.0;
                for (int a = 0; a < nc; ++a) {
                    int ax = a % n, ay = (a / n) % n, az = a / (n * n);
                    double lx = orc_lagrange(n, gx, ax, qx[kx]), ly = orc_lagrange(n, gx, ay, qx[ky]), lz = orc_lagrange(n, gx, az, qx[kz]);
                    double dlx = orc_lagrange_deriv(n, gx, ax, qx[kx]), dly = orc_lagrange_deriv(n, gx, ay, qx[ky]), dlz = orc_lagrange_deriv(n, gx, az, qx[kz]);
                    double r[3] = {dlx * ly * lz, lx * dly * lz, lx * ly * dlz}; /* reference gradient */
                    Pv[a] = lx * ly * lz;
                    for (int i = 0; i < 3; ++i) /* (J^{-T} r)_i = sum_j Ji[j][i] r_j */
                        G[3 * a + i] = Ji[0][i] * r[0] + Ji[1][i] * r[1] + Ji[2][i] * r[2];
                }
                for (int a = 0; a < nc; ++a)
                    for (int b = 0; b < nc; ++b)
                        He[(size_t)a * nc + b] += wq * (kin * (G[3 * a] * G[3 * b] + G[3 * a + 1] * G[3 * b + 1] + G[3 * a + 2] * G[3 * b + 2]) +
                                                       pot * V * Pv[a] * Pv[b]);
            }
    free(Pv); free(G);
}

/* positions and |det J| of the trilinear map at npts reference points xi (npts x 3): pos (npts x 3), det (npts) */
void orc_general_map(const double* verts, const double* xi, int npts, double* pos, double* det)
{
    for (int k = 0; k < npts; ++k) {
        double J[3][3], q[3];
        trilinear_jacobian(verts, xi[3 * k], xi[3 * k + 1], xi[3 * k + 2], J, q);
        pos[3 * k] = q[0]; pos[3 * k + 1] = q[1]; pos[3 * k + 2] = q[2];
        det[k] = fabs(det3(J));
    }
}
