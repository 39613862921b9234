// fe_cheb.cu -- C-ABI entry points (include/fe_cheb.h) and host-side mesh setup.
//
// The operator H~ = M^{-1/2} (1/2 K + M_V) M^{-1/2} (Eq. 17, 19) is never stored: every apply runs the
// fused gather -> sum-factorised cell contraction -> scatter kernels of fe_kernels.cuh on the caller's stream.
#include "../../include/fe_cheb.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <mutex>
#include <vector>

#include "fe_apply_tma.cuh"
#include "fe_density.cuh"
#include "fe_diag.cuh"
#include "fe_general.cuh"
#include "fe_gbox.cuh"
#include "fe_general.h"
#include "fe_minres.cuh"
#include "fe_rr.cuh"
#include "fe_kernels.cuh"
#include "fe_tables.h"

using namespace fecheb;

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess)                                                                      \
            return fail(e_ == cudaErrorMemoryAllocation ? FE_ERR_NOMEM : FE_ERR_CUDA, "%s: %s", #expr, \
                        cudaGetErrorString(e_));                                                    \
    } while (0)

struct fe_mesh {
    int p = 0, n = 0, cx = 0, cy = 0, cz = 0, device = 0, nc = 0;
    int64_t Nx = 0, Ny = 0, Nz = 0, N = 0, ncells = 0;
    std::vector<double> xe, ye, ze;
    Tables1D tab;
    std::vector<double> mx, my, mz;  // per-axis lumped GLL mass: M_gg = mx[gx] my[gy] mz[gz]
    double* d_sm = nullptr;          // N: mu_g M_gg^{-1/2} (0 on the Dirichlet boundary)
    double *d_hx = nullptr, *d_hy = nullptr, *d_hz = nullptr;
    double* d_WV = nullptr;  // cells*n^3: J w_q V_q
    double* d_VZ = nullptr;  // cells*REC: per-cell records of the TMA kernel (VZ | s_g | kz s_g | ky/kx, kx/kz)
    double *d_sx = nullptr, *d_sy = nullptr, *d_sz = nullptr;  // per-axis mu M^{-1/2}
    EOTab eoN, eoNT, eoG;    // even-odd halves of N' = diag(sqrt w) N, N'^T, G' = diag(w^-1/2) G diag(w^-1/2)
    bool have_V = false;
    int variant = 0;
    double* d_minv = nullptr;   // N: MINRES preconditioner, 1 / diag(M^{-1/2} 1/2 K M^{-1/2}) on free rows (built on first use)
    double* d_mask = nullptr;   // N: 1 on free rows, 0 on Dirichlet rows (the unpreconditioned MINRES)
    double* d_scal = nullptr;   // 21 * 128 doubles: MINRES column scalars
    double *d_WU = nullptr, *d_VZU = nullptr;  // fe_apply_potential: J w U of the caller's field (+ unused record output)
    double* d_host = nullptr;   // device staging of cheb_filter_host (grown on demand)
    size_t host_cap = 0;
    cudaStream_t hstream[2] = {nullptr, nullptr};
    double* d_small = nullptr;  // 2 * 128 * 128: B x B scratch of the Rayleigh-Ritz step
    // general hexahedral mesh with hanging nodes (fe_mesh_create_general; fe_general.h / fe_general.cuh): N = unconstrained nodes
    int kind = 0;  // 0: tensor-product box mesh, 1: general
    GeneralHost* gh = nullptr;
    int32_t* d_gl2g = nullptr;
    double *d_gmetric = nullptr, *d_gwdet = nullptr, *d_gsc = nullptr;
    EOTab eoD, eoDT;  // even-odd halves of the collocation derivative and its transpose (centro-antisymmetric)
    struct GenBundlesDev {  // rows with identical column lists packed for k_gen_rows_times_block (fe_general.cuh)
        long long* bptr = nullptr;
        int32_t *bcol = nullptr, *brow = nullptr, *out = nullptr;
        double* bw = nullptr;
        long long nb = 0;
    } gexp,  // expansion X_h = C_h (s . X); the collapse Y += alpha s . C_h^T Y_h reads the same bundles the other way
      gtr;   // variant 4 only: the transposed rows, one owner per row of Y (a collapse without atomics)
    int32_t* d_colcells = nullptr;        // variant 4: cells sorted by colour (cells of one colour share no node)
    std::vector<int64_t> colour_off;      //   colour c = cells [colour_off[c], colour_off[c+1])
    double *d_Xh = nullptr, *d_Yh = nullptr;  // (N_all - N) * hcap: expanded hanging values / their scatter target
    double* d_grecU = nullptr;  // fe_apply_potential on a general mesh: records with zero metric and WV = w |J| U
    // general mesh whose cells are all axis-aligned boxes (octree leaves of a box): the 10-sweep kernel of fe_gbox.cuh
    bool gbox = false, gbox_off = false;  // gbox_off: fe_apply_potential borrows the generic kernel (records with zero metric)
    double* d_gbrec = nullptr;            // ncells * gbox_rec_doubles(n)
    EOTab bxN, bxNT, bxG;                 // folded tables N', N'^T, G' (as on box meshes)
    int hcap = 0;
    int sms = 0;  // multiprocessors of the device (persistent grid size)
    int64_t launches = 0;
};

const char* fe_last_error(void) { return g_err; }

// even-odd split of a centro-symmetric n x n matrix (row-major M[i*n+k]); transpose selects M^T
static void make_eo(const double* M, int n, bool transpose, EOTab* T)
{
    const int h = n / 2, c = (n + 1) / 2;
    memset(T, 0, sizeof(*T));
    auto at = [&](int i, int k) { return transpose ? M[k * n + i] : M[i * n + k]; };
    for (int i = 0; i < c; ++i) {
        for (int k = 0; k < h; ++k) {
            T->S[i * h + k] = 0.5 * (at(i, k) + at(i, n - 1 - k));
            if (i < h) T->A[i * h + k] = 0.5 * (at(i, k) - at(i, n - 1 - k));
        }
        if (n % 2 == 1) T->Mid[i] = at(i, h);
    }
}

static int small_tile(int n) { return 3 * n * n * (n + (n & 1)) + 8; }  // REC of fe_apply_tma.cuh

// Gauss weights folded into the 1-D tables (fe_apply_tma.cuh): N' = diag(sqrt w) N, G' = diag(w^-1/2) G diag(w^-1/2)
static void build_folded_tables(const fe_mesh* m, EOTab* eoN, EOTab* eoNT, EOTab* eoG)
{
    const int n = m->n;
    double Np[kMaxN * kMaxN], Gp[kMaxN * kMaxN];
    for (int q = 0; q < n; ++q)
        for (int a = 0; a < n; ++a) {
            Np[q * n + a] = std::sqrt(m->tab.gl_w[q]) * m->tab.N[q * n + a];
            Gp[q * n + a] = m->tab.G[q * n + a] / std::sqrt(m->tab.gl_w[q] * m->tab.gl_w[a]);
        }
    make_eo(Np, n, false, eoN);
    make_eo(Np, n, true, eoNT);
    make_eo(Gp, n, false, eoG);
}

static void axis_mass(const std::vector<double>& e, int c, int p, const Tables1D& t, std::vector<double>& m)
{
    m.assign((size_t)c * p + 1, 0.0);
    for (int ec = 0; ec < c; ++ec)
        for (int a = 0; a <= p; ++a) m[(size_t)ec * p + a] += 0.5 * (e[ec + 1] - e[ec]) * t.gll_w[a];
}

static int upload(double** dst, const std::vector<double>& src)
{
    CUDA_TRY(cudaMalloc((void**)dst, src.size() * sizeof(double)));
    CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(double), cudaMemcpyHostToDevice));
    return FE_OK;
}

int fe_mesh_create(const double* xe, int cx, const double* ye, int cy, const double* ze, int cz, int p,
                   int cuda_device, fe_mesh** out)
{
    if (!out) return fail(FE_ERR_INVALID, "fe_mesh_create: out is NULL");
    *out = nullptr;
    if (!xe || !ye || !ze) return fail(FE_ERR_INVALID, "fe_mesh_create: NULL edge array");
    if (p < 1 || p > 8) return fail(FE_ERR_INVALID, "fe_mesh_create: order p=%d outside 1..8", p);
    if (cx < 1 || cy < 1 || cz < 1) return fail(FE_ERR_INVALID, "fe_mesh_create: need at least one cell per axis");
    const double* ed[3] = {xe, ye, ze};
    const int cc[3] = {cx, cy, cz};
    for (int d = 0; d < 3; ++d)
        for (int i = 0; i < cc[d]; ++i)
            if (!(ed[d][i + 1] > ed[d][i]) || !std::isfinite(ed[d][i]) || !std::isfinite(ed[d][i + 1]))
                return fail(FE_ERR_INVALID, "fe_mesh_create: edges of axis %d not strictly increasing at %d", d, i);
    const int64_t Nx = (int64_t)cx * p + 1, Ny = (int64_t)cy * p + 1, Nz = (int64_t)cz * p + 1;
    if ((double)Nx * (double)Ny * (double)Nz > 2147483647.0)
        return fail(FE_ERR_INVALID, "fe_mesh_create: more than 2^31-1 nodes (int32 l2g, R3)");
    int ndev = 0;
    CUDA_TRY(cudaGetDeviceCount(&ndev));
    if (cuda_device < 0 || cuda_device >= ndev) return fail(FE_ERR_INVALID, "fe_mesh_create: no CUDA device %d", cuda_device);
    CUDA_TRY(cudaSetDevice(cuda_device));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, cuda_device));
    if (prop.major < 10) return fail(FE_ERR_CUDA, "fe_mesh_create: device %d is sm_%d%d; this library is built for sm_100a only", cuda_device, prop.major, prop.minor);

    fe_mesh* m = new (std::nothrow) fe_mesh;
    if (!m) return fail(FE_ERR_NOMEM, "fe_mesh_create: host allocation failed");
    m->p = p; m->n = p + 1; m->cx = cx; m->cy = cy; m->cz = cz; m->device = cuda_device;
    m->nc = m->n * m->n * m->n;
    m->sms = prop.multiProcessorCount;
    m->Nx = Nx; m->Ny = Ny; m->Nz = Nz; m->N = Nx * Ny * Nz; m->ncells = (int64_t)cx * cy * cz;
    m->xe.assign(xe, xe + cx + 1); m->ye.assign(ye, ye + cy + 1); m->ze.assign(ze, ze + cz + 1);
    build_tables(p, &m->tab);
    axis_mass(m->xe, cx, p, m->tab, m->mx);
    axis_mass(m->ye, cy, p, m->tab, m->my);
    axis_mass(m->ze, cz, p, m->tab, m->mz);

    // per-axis M^{-1/2} with the Dirichlet mask folded in (R5, R6), and per-axis cell sizes
    std::vector<double> s[3], h[3];
    const std::vector<double>* mm[3] = {&m->mx, &m->my, &m->mz};
    const std::vector<double>* ee[3] = {&m->xe, &m->ye, &m->ze};
    for (int d = 0; d < 3; ++d) {
        size_t nn = mm[d]->size();
        s[d].resize(nn);
        for (size_t i = 0; i < nn; ++i) s[d][i] = (i == 0 || i == nn - 1) ? 0.0 : 1.0 / std::sqrt((*mm[d])[i]);
        h[d].resize(cc[d]);
        for (int i = 0; i < cc[d]; ++i) h[d][i] = (*ee[d])[i + 1] - (*ee[d])[i];
    }
    int rc = FE_OK;
    auto cleanup = [&](int code) {
        if (code != FE_OK) fe_mesh_destroy(m);
        return code;
    };
    if ((rc = upload(&m->d_sx, s[0])) || (rc = upload(&m->d_sy, s[1])) || (rc = upload(&m->d_sz, s[2]))) return cleanup(rc);
    if ((rc = upload(&m->d_hx, h[0])) || (rc = upload(&m->d_hy, h[1])) || (rc = upload(&m->d_hz, h[2]))) return cleanup(rc);
    cudaError_t ce = cudaMalloc((void**)&m->d_sm, (size_t)m->N * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&m->d_WV, (size_t)m->ncells * m->nc * sizeof(double));
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&m->d_VZ, (size_t)m->ncells * small_tile(m->n) * sizeof(double));
    if (ce != cudaSuccess) return cleanup(fail(FE_ERR_NOMEM, "fe_mesh_create: device allocation failed: %s", cudaGetErrorString(ce)));
    ce = cudaMemset(m->d_VZ, 0, (size_t)m->ncells * small_tile(m->n) * sizeof(double));
    if (ce != cudaSuccess) return cleanup(fail(FE_ERR_CUDA, "fe_mesh_create: memset failed: %s", cudaGetErrorString(ce)));
    k_build_records<<<m->sms * 8, 256>>>(m->d_VZ, m->n, m->cx, m->cy, m->ncells, m->d_sx, m->d_sy, m->d_sz, m->d_hx, m->d_hy, m->d_hz);
    m->launches += 1;
    launch_build_scaling(m->d_sx, m->d_sy, m->d_sz, m->Nx, m->Ny, m->Nz, m->d_sm, m->sms, 0);
    m->launches += 1;
    ce = cudaDeviceSynchronize();
    if (ce != cudaSuccess) return cleanup(fail(FE_ERR_CUDA, "fe_mesh_create: scaling kernel failed: %s", cudaGetErrorString(ce)));
    build_folded_tables(m, &m->eoN, &m->eoNT, &m->eoG);
    *out = m;
    return cleanup(FE_OK);
}

int fe_mesh_destroy(fe_mesh* m)
{
    if (!m) return FE_OK;
    if (m->device >= 0) cudaSetDevice(m->device);
    cudaFree(m->d_sm); cudaFree(m->d_hx); cudaFree(m->d_hy); cudaFree(m->d_hz); cudaFree(m->d_WV);
    cudaFree(m->d_host); cudaFree(m->d_WU); cudaFree(m->d_VZU);
    for (cudaStream_t s : m->hstream) if (s) cudaStreamDestroy(s);
    cudaFree(m->d_small); cudaFree(m->d_minv); cudaFree(m->d_mask); cudaFree(m->d_scal);
    cudaFree(m->d_VZ); cudaFree(m->d_sx); cudaFree(m->d_sy); cudaFree(m->d_sz);
    cudaFree(m->d_gl2g); cudaFree(m->d_gmetric); cudaFree(m->d_gwdet); cudaFree(m->d_gsc);
    cudaFree(m->d_Xh); cudaFree(m->d_Yh); cudaFree(m->d_grecU); cudaFree(m->d_gbrec);
    cudaFree(m->gexp.bptr); cudaFree(m->gexp.bcol); cudaFree(m->gexp.brow); cudaFree(m->gexp.out); cudaFree(m->gexp.bw);
    cudaFree(m->gtr.bptr); cudaFree(m->gtr.bcol); cudaFree(m->gtr.brow); cudaFree(m->gtr.out); cudaFree(m->gtr.bw);
    cudaFree(m->d_colcells);
    delete m->gh;
    delete m;
    return FE_OK;
}

int64_t fe_num_nodes(const fe_mesh* m) { return m ? m->N : FE_ERR_INVALID; }
int64_t fe_num_free(const fe_mesh* m)
{
    if (!m) return FE_ERR_INVALID;
    if (m->kind == 0) return (m->Nx - 2) * (m->Ny - 2) * (m->Nz - 2);
    int64_t k = 0;
    for (uint8_t f : m->gh->mask) k += f;
    return k;
}
int64_t fe_num_all_nodes(const fe_mesh* m) { return m ? (m->kind ? m->gh->N_all : m->N) : FE_ERR_INVALID; }
int64_t fe_num_constraint_entries(const fe_mesh* m) { return m ? (m->kind ? (int64_t)m->gh->ccol.size() : 0) : FE_ERR_INVALID; }
int64_t fe_num_cells(const fe_mesh* m) { return m ? m->ncells : FE_ERR_INVALID; }
int fe_nodes_per_cell(const fe_mesh* m) { return m ? m->nc : FE_ERR_INVALID; }
int fe_quad_per_cell(const fe_mesh* m) { return m ? m->nc : FE_ERR_INVALID; }
int64_t fe_launch_count(const fe_mesh* m) { return m ? m->launches : FE_ERR_INVALID; }

int fe_get_l2g(const fe_mesh* m, int32_t* l2g)
{
    if (!m || !l2g) return fail(FE_ERR_INVALID, "fe_get_l2g: NULL argument");
    if (m->kind) { memcpy(l2g, m->gh->l2g.data(), m->gh->l2g.size() * sizeof(int32_t)); return FE_OK; }
    const int n = m->n, p = m->p;
    for (int64_t ez = 0; ez < m->cz; ++ez)
        for (int64_t ey = 0; ey < m->cy; ++ey)
            for (int64_t ex = 0; ex < m->cx; ++ex) {
                int32_t* row = l2g + (ex + m->cx * (ey + m->cy * ez)) * m->nc;
                const int64_t base = ex * p + m->Nx * (ey * p + m->Ny * (ez * p));
                for (int az = 0; az < n; ++az)
                    for (int ay = 0; ay < n; ++ay)
                        for (int ax = 0; ax < n; ++ax)
                            row[ax + n * (ay + n * az)] = (int32_t)(base + ax + m->Nx * (ay + m->Ny * az));
            }
    return FE_OK;
}

// R4: x = lo + 0.5 (xi+1) (hi-lo); the last GLL node of a cell is exactly the upper edge
static void axis_coords(const std::vector<double>& e, int c, int p, const double* xi, bool lobatto, std::vector<double>& out)
{
    const int n = p + 1;
    out.resize(lobatto ? (size_t)c * p + 1 : (size_t)c * n);
    for (int ec = 0; ec < c; ++ec)
        for (int a = 0; a < n; ++a) {
            double v = (lobatto && a == p) ? e[ec + 1] : e[ec] + 0.5 * (xi[a] + 1.0) * (e[ec + 1] - e[ec]);
            out[lobatto ? (size_t)ec * p + a : (size_t)ec * n + a] = v;
        }
}

int fe_get_node_coords(const fe_mesh* m, double* xyz)
{
    if (!m || !xyz) return fail(FE_ERR_INVALID, "fe_get_node_coords: NULL argument");
    if (m->kind) { memcpy(xyz, m->gh->node_xyz.data(), m->gh->node_xyz.size() * sizeof(double)); return FE_OK; }
    std::vector<double> X, Y, Z;
    axis_coords(m->xe, m->cx, m->p, m->tab.gll_x, true, X);
    axis_coords(m->ye, m->cy, m->p, m->tab.gll_x, true, Y);
    axis_coords(m->ze, m->cz, m->p, m->tab.gll_x, true, Z);
    for (int64_t gz = 0; gz < m->Nz; ++gz)
        for (int64_t gy = 0; gy < m->Ny; ++gy)
            for (int64_t gx = 0; gx < m->Nx; ++gx) {
                double* o = xyz + 3 * (gx + m->Nx * (gy + m->Ny * gz));
                o[0] = X[gx]; o[1] = Y[gy]; o[2] = Z[gz];
            }
    return FE_OK;
}

int fe_get_quad_coords(const fe_mesh* m, double* xyz)
{
    if (!m || !xyz) return fail(FE_ERR_INVALID, "fe_get_quad_coords: NULL argument");
    if (m->kind) { memcpy(xyz, m->gh->quad_xyz.data(), m->gh->quad_xyz.size() * sizeof(double)); return FE_OK; }
    const int n = m->n;
    std::vector<double> X, Y, Z;
    axis_coords(m->xe, m->cx, m->p, m->tab.gl_x, false, X);
    axis_coords(m->ye, m->cy, m->p, m->tab.gl_x, false, Y);
    axis_coords(m->ze, m->cz, m->p, m->tab.gl_x, false, Z);
    for (int64_t ez = 0; ez < m->cz; ++ez)
        for (int64_t ey = 0; ey < m->cy; ++ey)
            for (int64_t ex = 0; ex < m->cx; ++ex) {
                double* o = xyz + 3 * (ex + m->cx * (ey + m->cy * ez)) * m->nc;
                for (int qz = 0; qz < n; ++qz)
                    for (int qy = 0; qy < n; ++qy)
                        for (int qx = 0; qx < n; ++qx) {
                            double* q = o + 3 * (qx + n * (qy + n * qz));
                            q[0] = X[ex * n + qx]; q[1] = Y[ey * n + qy]; q[2] = Z[ez * n + qz];
                        }
            }
    return FE_OK;
}

int fe_get_mass(const fe_mesh* m, double* Mdiag)
{
    if (!m || !Mdiag) return fail(FE_ERR_INVALID, "fe_get_mass: NULL argument");
    if (m->kind) { memcpy(Mdiag, m->gh->mass.data(), m->gh->mass.size() * sizeof(double)); return FE_OK; }
    for (int64_t gz = 0; gz < m->Nz; ++gz)
        for (int64_t gy = 0; gy < m->Ny; ++gy)
            for (int64_t gx = 0; gx < m->Nx; ++gx) Mdiag[gx + m->Nx * (gy + m->Ny * gz)] = m->mx[gx] * m->my[gy] * m->mz[gz];
    return FE_OK;
}

int fe_get_dirichlet_mask(const fe_mesh* m, uint8_t* mask)
{
    if (!m || !mask) return fail(FE_ERR_INVALID, "fe_get_dirichlet_mask: NULL argument");
    if (m->kind) { memcpy(mask, m->gh->mask.data(), m->gh->mask.size()); return FE_OK; }
    for (int64_t gz = 0; gz < m->Nz; ++gz)
        for (int64_t gy = 0; gy < m->Ny; ++gy)
            for (int64_t gx = 0; gx < m->Nx; ++gx)
                mask[gx + m->Nx * (gy + m->Ny * gz)] =
                    (gx == 0 || gx == m->Nx - 1 || gy == 0 || gy == m->Ny - 1 || gz == 0 || gz == m->Nz - 1) ? 0 : 1;
    return FE_OK;
}

static void fill_params(const fe_mesh* m, ApplyParams* prm)
{
    memset(prm, 0, sizeof(*prm));
    prm->sm = m->d_sm; prm->WV = m->d_WV; prm->hx = m->d_hx; prm->hy = m->d_hy; prm->hz = m->d_hz;
    prm->cx = m->cx; prm->cy = m->cy; prm->cz = m->cz;
    prm->Nx = m->Nx; prm->NxNy = m->Nx * m->Ny;
    const int n = m->n;
    for (int q = 0; q < n; ++q) prm->w[q] = m->tab.gl_w[q];
    make_eo(m->tab.N, n, false, &prm->eoN);
    make_eo(m->tab.N, n, true, &prm->eoNT);
    make_eo(m->tab.G, n, false, &prm->eoG);
}

int fe_set_potential(fe_mesh* m, const double* Vq_dev, int copy, void* cuda_stream)
{
    (void)copy;
    if (!m || !Vq_dev) return fail(FE_ERR_INVALID, "fe_set_potential: NULL argument");
    if (m->device < 0) return fail(FE_ERR_STATE, "fe_set_potential: the handle was created without a device (tables only)");
    CUDA_TRY(cudaSetDevice(m->device));
    if (m->kind) {
        k_gen_weight_potential<<<m->sms * 8, 256, 0, (cudaStream_t)cuda_stream>>>(m->d_gmetric, Vq_dev, m->d_gwdet, m->ncells, m->nc,
                                                                                  gen_rec_doubles(m->n));
        CUDA_TRY(cudaGetLastError());
        m->launches += 1;
        if (m->gbox) {
            k_gbox_weight_potential<<<m->sms * 8, 256, 0, (cudaStream_t)cuda_stream>>>(m->d_gbrec, Vq_dev, m->ncells, m->n);
            CUDA_TRY(cudaGetLastError());
            m->launches += 1;
        }
        m->have_V = true;
        return FE_OK;
    }
    ApplyParams prm;
    fill_params(m, &prm);
    launch_weight_potential(prm, m->p, Vq_dev, m->d_WV, m->d_VZ, m->ncells, m->sms, (cudaStream_t)cuda_stream);
    CUDA_TRY(cudaGetLastError());
    m->launches += 1;
    m->have_V = true;
    return FE_OK;
}

int fe_set_variant(fe_mesh* m, int variant)
{
    if (!m) return fail(FE_ERR_INVALID, "fe_set_variant: NULL mesh");
    if (!variant_supported(m->p, variant)) return fail(FE_ERR_INVALID, "fe_set_variant: variant %d not available for p=%d", variant, m->p);
    m->variant = variant;
    return FE_OK;
}

// one fused operator launch: Y = mu (alpha (S sum_e P_e^T y_e - (c + eps) X) + beta Z)
static int general_step(fe_mesh* m, const double* X, const double* Z, double* Y, int B, const double* eps,
                        double alpha, double beta, double c, cudaStream_t st, double* W = nullptr, double beta_next = 0.0,
                        bool y_ready = false);
static int general_expand(fe_mesh* m, const double* X, int B, cudaStream_t st);

static int operator_step(fe_mesh* m, const double* X, const double* Z, double* Y, int B, const double* eps,
                         double alpha, double beta, double c, cudaStream_t st)
{
    if (m->kind) return general_step(m, X, Z, Y, B, eps, alpha, beta, c, st);
    ApplyParams prm;
    fill_params(m, &prm);
    prm.X = X; prm.Z = Z; prm.Y = Y; prm.eps = eps; prm.B = B;
    prm.alpha = alpha; prm.beta = beta; prm.c = c;
    int nl = 0;
    cudaError_t e = launch_apply(prm, m->p, m->variant, m->N, m->ncells, st, &nl);
    if (e != cudaSuccess) return fail(FE_ERR_CUDA, "operator launch failed: %s", cudaGetErrorString(e));
    m->launches += nl;
    return FE_OK;
}

// ---- general hexahedral meshes with hanging nodes (NEXT-3; fe_general.h / fe_general.cuh) ---------------------------------------
template <class T>
static int upload_vec(T** dst, const std::vector<T>& src)
{
    if (src.empty()) { *dst = nullptr; return FE_OK; }
    CUDA_TRY(cudaMalloc((void**)dst, src.size() * sizeof(T)));
    CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return FE_OK;
}

// sort sparse rows by column list and pack rows with identical lists into bundles for k_gen_rows_times_block / k_gen_collapse
static int pack_bundles(const std::vector<std::vector<std::pair<int32_t, double>>>& rws, const std::vector<int32_t>& dst_of,
                    fe_mesh::GenBundlesDev* dev)
{
    const int64_t nr = (int64_t)rws.size();
    std::vector<int32_t> order((size_t)nr);
    for (int64_t i = 0; i < nr; ++i) order[i] = (int32_t)i;
    auto same_cols = [&](int32_t a, int32_t b) {
        if (rws[a].size() != rws[b].size()) return false;
        for (size_t k = 0; k < rws[a].size(); ++k)
            if (rws[a][k].first != rws[b][k].first) return false;
        return true;
    };
    std::sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
        if (rws[a].size() != rws[b].size()) return rws[a].size() < rws[b].size();
        for (size_t k = 0; k < rws[a].size(); ++k)
            if (rws[a][k].first != rws[b][k].first) return rws[a][k].first < rws[b][k].first;
        return a < b;
    });
    std::vector<long long> bptr{0};
    std::vector<int32_t> bcol, brow{0}, out;
    std::vector<double> bw;
    for (int64_t i = 0; i < nr;) {
        int64_t e = i + 1;
        while (e < nr && e - i < kGenBundle && same_cols(order[i], order[e])) ++e;
        const auto& first = rws[order[i]];
        for (size_t k = 0; k < first.size(); ++k) {
            // an entry whose weights are 0 for every row of the bundle (a Dirichlet node: the weights carry s = 0) is dropped, so
            // the kernels never read such a row of the block -- whatever it holds (R5) -- and need no per-weight test
            bool any = false;
            for (int64_t q = i; q < e; ++q) any = any || rws[order[q]][k].second != 0.0;
            if (!any) continue;
            bcol.push_back(first[k].first);
            for (int u = 0; u < kGenBundle; ++u) bw.push_back(i + u < e ? rws[order[i + u]][k].second : 0.0);
        }
        for (int64_t q = i; q < e; ++q) out.push_back(dst_of[order[q]]);
        bptr.push_back((long long)bcol.size());
        brow.push_back((int32_t)out.size());
        i = e;
    }
    dev->nb = (long long)bptr.size() - 1;
    int r;
    if ((r = upload_vec(&dev->bptr, bptr)) || (r = upload_vec(&dev->bcol, bcol)) || (r = upload_vec(&dev->brow, brow)) ||
        (r = upload_vec(&dev->out, out)) || (r = upload_vec(&dev->bw, bw)))
        return r;
    return FE_OK;
}

int fe_mesh_create_general(int cx, int cy, int cz, const int32_t* cells, int64_t ncells, const double* verts, int p,
                           int cuda_device, fe_mesh** out)
{
    if (!out) return fail(FE_ERR_INVALID, "fe_mesh_create_general: out is NULL");
    *out = nullptr;
    if (!cells || !verts) return fail(FE_ERR_INVALID, "fe_mesh_create_general: NULL array");
    if (p < 1 || p > 8) return fail(FE_ERR_INVALID, "fe_mesh_create_general: order p=%d outside 1..8", p);
    if (cx < 1 || cy < 1 || cz < 1 || ncells < 1) return fail(FE_ERR_INVALID, "fe_mesh_create_general: empty mesh");
    for (int64_t i = 0; i < ncells * 24; ++i)
        if (!std::isfinite(verts[i])) return fail(FE_ERR_INVALID, "fe_mesh_create_general: corner coordinate %lld is not finite", (long long)i);
    fe_mesh* m = new (std::nothrow) fe_mesh;
    if (!m) return fail(FE_ERR_NOMEM, "fe_mesh_create_general: host allocation failed");
    m->gh = new (std::nothrow) GeneralHost;
    if (!m->gh) { delete m; return fail(FE_ERR_NOMEM, "fe_mesh_create_general: host allocation failed"); }
    m->kind = 1; m->p = p; m->n = p + 1; m->nc = m->n * m->n * m->n; m->cx = cx; m->cy = cy; m->cz = cz;
    build_tables(p, &m->tab);
    char msg[400];
    if (build_general_mesh(cx, cy, cz, cells, ncells, verts, p, m->tab, m->gh, msg, sizeof(msg))) {
        fe_mesh_destroy(m);
        return fail(FE_ERR_INVALID, "%s", msg);
    }
    const GeneralHost& g = *m->gh;
    m->N = g.N; m->ncells = ncells;
    if (cuda_device == -1) {  // tables only (numbering, constraints, coordinates, mass): no device, no operator
        m->device = -1;
        *out = m;
        return FE_OK;
    }
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) {
        fe_mesh_destroy(m);
        return ce != cudaSuccess ? fail(FE_ERR_CUDA, "fe_mesh_create_general: %s", cudaGetErrorString(ce))
                                 : fail(FE_ERR_INVALID, "fe_mesh_create_general: no CUDA device %d", cuda_device);
    }
    m->device = cuda_device;
    cudaDeviceProp prop;
    if (cudaSetDevice(cuda_device) != cudaSuccess || cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess || prop.major < 10) {
        fe_mesh_destroy(m);
        return fail(FE_ERR_CUDA, "fe_mesh_create_general: device %d is not an sm_100 device", cuda_device);
    }
    m->sms = prop.multiProcessorCount;
    // s_g = mu_g M_c,gg^{-1/2} (Eq. 19 with the constrained lumped mass, R25); metric split into its tensor and weight parts
    const int grec = gen_rec_doubles(m->n);
    std::vector<double> sv((size_t)g.N), met((size_t)ncells * grec, 0.0), wdet((size_t)ncells * m->nc);
    for (int64_t i = 0; i < g.N; ++i) sv[i] = g.mask[i] ? 1.0 / std::sqrt(g.mass[i]) : 0.0;
    for (int64_t e = 0; e < ncells; ++e) {
        memcpy(&met[(size_t)e * grec], &g.metric[(size_t)e * 7 * m->nc], (size_t)6 * m->nc * sizeof(double));
        memcpy(&wdet[(size_t)e * m->nc], &g.metric[((size_t)e * 7 + 6) * m->nc], (size_t)m->nc * sizeof(double));
    }
    std::vector<double> scv(g.l2g.size()), csv(g.cval.size());
    for (size_t i = 0; i < scv.size(); ++i) scv[i] = g.l2g[i] < g.N ? sv[g.l2g[i]] : 1.0;
    for (size_t k = 0; k < csv.size(); ++k) csv[k] = g.cval[k] * sv[g.ccol[k]];  // constraint weight times s of its node
    {   // plain (unfolded) tables for the general kernel; D is centro-antisymmetric: its middle row goes to row h of S
        const int n = m->n, h = n / 2;
        double Dt[kMaxN * kMaxN];
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) Dt[a * n + b] = m->tab.D[b * n + a];
        make_eo(m->tab.N, n, false, &m->eoN);
        make_eo(m->tab.N, n, true, &m->eoNT);
        make_eo(m->tab.D, n, false, &m->eoD);
        make_eo(Dt, n, false, &m->eoDT);
        if (n % 2 == 1)
            for (int k = 0; k < h; ++k) { m->eoD.S[h * h + k] = m->tab.D[h * n + k]; m->eoDT.S[h * h + k] = Dt[h * n + k]; }
    }
    // the constraint rows and their transpose, sorted by column list and packed into bundles of rows with identical lists
    int rc = FE_OK;
    {
        const int64_t nh = g.N_all - g.N;
        std::vector<std::vector<std::pair<int32_t, double>>> fw((size_t)nh);
        std::vector<int32_t> fdst((size_t)nh);
        for (int64_t r = 0; r < nh; ++r) {
            fdst[r] = (int32_t)r;
            for (int64_t k = g.crow[r]; k < g.crow[r + 1]; ++k) fw[r].push_back({g.ccol[k], csv[k]});
        }
        if ((rc = pack_bundles(fw, fdst, &m->gexp))) { fe_mesh_destroy(m); return rc; }
    }
    if ((rc = upload_vec(&m->d_gsc, scv)) || (rc = upload_vec(&m->d_sm, sv)) || (rc = upload_vec(&m->d_gl2g, g.l2g)) || (rc = upload_vec(&m->d_gmetric, met)) ||
        (rc = upload_vec(&m->d_gwdet, wdet))) {
        fe_mesh_destroy(m);
        return rc;
    }
    // Octree leaves of an undeformed box (the paper's adaptive meshes, l.273): every cell is an axis-aligned box, the metric
    // is diagonal and constant per cell, and the 10-sweep kernel of fe_gbox.cuh applies.  Corner v = vx + 2 (vy + 2 vz).
    if (gbox_supported(p)) {
        const int n = m->n, NP = n + (n & 1), SMALL = n * n * NP, brec = gbox_rec_doubles(n);
        std::vector<double> br((size_t)ncells * brec, 0.0);
        std::vector<char> owned((size_t)g.N, 0);  // owner cell of an unconstrained node = the first cell that lists it
        bool all_boxes = true;
        for (int64_t e = 0; e < ncells && all_boxes; ++e) {
            const double* c = verts + e * 24;
            double lo[3], h[3];
            for (int d = 0; d < 3; ++d) { lo[d] = c[d]; h[d] = c[3 * (1 << d) + d] - c[d]; }
            for (int v = 0; v < 8 && all_boxes; ++v)
                for (int d = 0; d < 3; ++d) {
                    const double want = lo[d] + (((v >> d) & 1) ? h[d] : 0.0);
                    if (!(h[d] > 0.0) || std::fabs(c[3 * v + d] - want) > 1e-13 * (std::fabs(want) + h[d])) all_boxes = false;
                }
            if (!all_boxes) break;
            double* r = &br[(size_t)e * brec];
            const double kz = 0.25 * h[0] * h[1] / h[2];  // 2J/hz^2, J = hx hy hz / 8
            bool dirichlet = false;
            for (int az = 0; az < n; ++az)
                for (int ay = 0; ay < n; ++ay)
                    for (int ax = 0; ax < n; ++ax) {
                        const double sc = scv[(size_t)e * m->nc + ax + n * (ay + n * az)];
                        r[SMALL + (az * n + ay) * NP + ax] = sc;
                        r[2 * SMALL + 8 + (az * n + ay) * NP + ax] = kz * sc;
                        dirichlet = dirichlet || sc == 0.0;
                    }
            r[2 * SMALL + 0] = (h[0] * h[0]) / (h[1] * h[1]);
            r[2 * SMALL + 1] = (h[2] * h[2]) / (h[0] * h[0]);
            r[2 * SMALL + 2] = kz;
            r[2 * SMALL + 3] = 0.5 * h[2] * h[2];
            r[2 * SMALL + 4] = dirichlet ? 1.0 : 0.0;
            int32_t* ids = reinterpret_cast<int32_t*>(r + 3 * SMALL + 8);
            for (int a = 0; a < m->nc; ++a) {
                const int32_t id = g.l2g[(size_t)e * m->nc + a];
                ids[a] = id;
                if (id < g.N && !owned[id]) { owned[id] = 1; ids[a] = (int32_t)((uint32_t)id | 0x80000000u); }  // bit 31: owner
            }
        }
        if (all_boxes) {
            if ((rc = upload_vec(&m->d_gbrec, br))) { fe_mesh_destroy(m); return rc; }
            build_folded_tables(m, &m->bxN, &m->bxNT, &m->bxG);
            m->gbox = true;
        }
    }
    *out = m;
    return FE_OK;
}

int fe_get_constraints(const fe_mesh* m, int64_t* row_ptr, int32_t* col, double* val)
{
    if (!m || !row_ptr) return fail(FE_ERR_INVALID, "fe_get_constraints: NULL argument");
    if (!m->kind) { row_ptr[0] = 0; return FE_OK; }
    const GeneralHost& g = *m->gh;
    memcpy(row_ptr, g.crow.data(), g.crow.size() * sizeof(int64_t));
    if (!g.ccol.empty()) {
        if (!col || !val) return fail(FE_ERR_INVALID, "fe_get_constraints: NULL argument");
        memcpy(col, g.ccol.data(), g.ccol.size() * sizeof(int32_t));
        memcpy(val, g.cval.data(), g.cval.size() * sizeof(double));
    }
    return FE_OK;
}

// hanging values X_h = C_h (s . X) of a block into the handle's scratch (grown to B columns on demand)
static int general_expand(fe_mesh* m, const double* X, int B, cudaStream_t st)
{
    const GeneralHost& g = *m->gh;
    const long long nh = g.N_all - g.N;
    if (nh <= 0) return FE_OK;
    if (m->hcap < B) {
        cudaFree(m->d_Xh); cudaFree(m->d_Yh);
        m->d_Xh = m->d_Yh = nullptr; m->hcap = 0;
        CUDA_TRY(cudaMalloc((void**)&m->d_Xh, (size_t)nh * B * sizeof(double)));
        CUDA_TRY(cudaMalloc((void**)&m->d_Yh, (size_t)nh * B * sizeof(double)));
        m->hcap = B;
    }
    k_gen_rows_times_block<<<m->sms * 8, dim3(32, kGenRows), 0, st>>>(m->d_Xh, X, m->gexp.bptr, m->gexp.bcol, m->gexp.bw, m->gexp.brow,
                                                                      m->gexp.out, m->gexp.nb, B, 1.0, 0, m->d_Yh);  // also clears Y_h
    CUDA_TRY(cudaGetLastError());
    m->launches += 1;
    return FE_OK;
}

// Colour-ordered (deterministic) scatter on a general mesh (variant 4; S8(a) a3 "atomic or colour-ordered"): cells are
// coloured greedily so that no two cells of a colour share a node (unconstrained or hanging); the cell kernel is launched
// colour by colour, and the collapse runs over the transposed constraint rows (one owner per row of Y), so every sum has a
// fixed order and the result is bit-reproducible.  Built on first use.
static int ensure_general_colours(fe_mesh* m)
{
    if (m->d_colcells) return FE_OK;
    const GeneralHost& g = *m->gh;
    const int nc = m->nc;
    std::vector<int64_t> cnt((size_t)g.N_all + 1, 0);
    for (int32_t id : g.l2g) cnt[(size_t)id + 1] += 1;
    for (int64_t i = 0; i < g.N_all; ++i) cnt[i + 1] += cnt[i];
    std::vector<int32_t> cells_of((size_t)g.l2g.size());
    {
        std::vector<int64_t> pos(cnt.begin(), cnt.end() - 1);
        for (int64_t e = 0; e < g.ncells; ++e)
            for (int a = 0; a < nc; ++a) cells_of[pos[g.l2g[(size_t)e * nc + a]]++] = (int32_t)e;
    }
    std::vector<int> colour((size_t)g.ncells, -1);
    int ncol = 0;
    std::vector<char> used;
    for (int64_t e = 0; e < g.ncells; ++e) {
        used.assign((size_t)ncol + 1, 0);
        for (int a = 0; a < nc; ++a) {
            const int32_t id = g.l2g[(size_t)e * nc + a];
            for (int64_t q = cnt[id]; q < cnt[id + 1]; ++q) {
                const int c = colour[cells_of[q]];
                if (c >= 0) used[c] = 1;
            }
        }
        int c = 0;
        while (c < ncol && used[c]) ++c;
        colour[e] = c;
        if (c == ncol) ++ncol;
    }
    std::vector<int32_t> sorted;
    m->colour_off.assign(1, 0);
    for (int c = 0; c < ncol; ++c) {
        for (int64_t e = 0; e < g.ncells; ++e)
            if (colour[e] == c) sorted.push_back((int32_t)e);
        m->colour_off.push_back((int64_t)sorted.size());
    }
    // transposed constraint rows: for every unconstrained node with hanging dependents, (hanging row, weight * s)
    const int64_t nh = g.N_all - g.N;
    std::vector<std::vector<std::pair<int32_t, double>>> tr;
    std::vector<int32_t> tdst, tindex((size_t)g.N, -1);
    for (int64_t r = 0; r < nh; ++r)
        for (int64_t k = g.crow[r]; k < g.crow[r + 1]; ++k) {
            int32_t& ti = tindex[g.ccol[k]];
            if (ti < 0) { ti = (int32_t)tr.size(); tr.emplace_back(); tdst.push_back(g.ccol[k]); }
            const double sk = g.mask[g.ccol[k]] ? 1.0 / std::sqrt(g.mass[g.ccol[k]]) : 0.0;
            tr[ti].push_back({(int32_t)r, g.cval[k] * sk});
        }
    int rc;
    if (!tr.empty() && (rc = pack_bundles(tr, tdst, &m->gtr))) return rc;
    return upload_vec(&m->d_colcells, sorted);
}

// one fused operator step on a general mesh: diagonal terms (k_gen_init), expansion of the hanging values, the cell kernel,
// the transposed expansion
// Box-cell kernel only (general_fused): y_ready = Y already holds beta Y_{k-1} (written by the previous step's
// pre-initialisation; Z is not read), W != NULL = this step stores beta_next X into W for the step after it
static bool general_fused(const fe_mesh* m) { return m->kind && m->gbox && !m->gbox_off && m->variant != 9 && m->variant != 4; }

static int general_step(fe_mesh* m, const double* X, const double* Z, double* Y, int B, const double* eps,
                        double alpha, double beta, double c, cudaStream_t st, double* W, double beta_next, bool y_ready)
{
    const GeneralHost& g = *m->gh;
    const long long nh = g.N_all - g.N;
    int rc = general_expand(m, X, B, st);
    if (rc) return rc;
    const int grid = m->sms * 8;
    const dim3 rows(32, kGenRows);
    // box-cell kernel without a Z block: the shift term kappa_j X comes from the owner cells inside the kernel
    const bool fuse = general_fused(m) && !Z;
    if ((W || y_ready) && !fuse) return fail(FE_ERR_STATE, "general_step: pre-initialisation needs the box-cell kernel");
    bool init_kernel = false;
    if (y_ready) {
        // Y was pre-initialised by the previous step
    } else if (fuse || (!Z && !eps && c == 0.0))  // nothing diagonal to write here: Y is just cleared
        CUDA_TRY(cudaMemsetAsync(Y, 0, (size_t)g.N * B * sizeof(double), st));
    else {
        k_gen_init<<<grid, rows, 0, st>>>(Y, X, Z, m->d_sm, eps, alpha, beta, c, g.N, B);
        init_kernel = true;
    }
    // Y_h (the scatter target of the hanging nodes) was cleared by the expansion kernel: every hanging row is in one bundle
    // all cells axis-aligned boxes: the 10-sweep kernel (variant 9 keeps the generic 12-sweep kernel as a cross-check)
    const bool box = m->gbox && !m->gbox_off && m->variant != 9;
    GenParams prm;
    memset(&prm, 0, sizeof(prm));
    prm.X = X; prm.Xh = m->d_Xh ? m->d_Xh : X; prm.Y = Y; prm.Yh = m->d_Yh ? m->d_Yh : Y; prm.sc = m->d_gsc; prm.l2g = m->d_gl2g;
    prm.rec = m->d_gmetric; prm.N = g.N; prm.ncells = m->ncells; prm.B = B; prm.alpha = alpha;
    prm.eoN = m->eoN; prm.eoNT = m->eoNT; prm.eoD = m->eoD; prm.eoDT = m->eoDT;
    GBoxParams bp;
    if (box) {
        memset(&bp, 0, sizeof(bp));
        bp.X = prm.X; bp.Xh = prm.Xh; bp.Y = prm.Y; bp.Yh = prm.Yh; bp.rec = m->d_gbrec; bp.N = g.N; bp.ncells = m->ncells; bp.B = B;
        bp.eoN = m->bxN; bp.eoNT = m->bxNT; bp.eoG = m->bxG; bp.eoNTa = m->bxNT;
        for (double& x : bp.eoNTa.S) x *= alpha;
        for (double& x : bp.eoNTa.A) x *= alpha;
        for (double& x : bp.eoNTa.Mid) x *= alpha;
        if (fuse) {
            bp.W = W; bp.beta_next = beta_next; bp.eps = eps; bp.alpha = alpha; bp.c = c;
            bp.owner = (eps != nullptr || c != 0.0) ? 1 : 0;
        }
    }
    // the box kernel delivers alpha yhat to the hanging targets too (alpha sits in its last table): the collapse runs with 1
    const double alpha_h = box ? 1.0 : alpha;
    if (m->variant == 4) {  // colour-ordered, bit-reproducible
        if ((rc = ensure_general_colours(m))) return rc;
        for (size_t c = 0; c + 1 < m->colour_off.size(); ++c) {
            prm.cell_list = bp.cell_list = m->d_colcells + m->colour_off[c];
            prm.ncells = bp.ncells = m->colour_off[c + 1] - m->colour_off[c];
            cudaError_t ec = box ? launch_apply_gbox(bp, m->p, bp.ncells, m->sms, st) : launch_apply_gen(prm, m->p, prm.ncells, m->sms, st);
            if (ec != cudaSuccess) return fail(FE_ERR_CUDA, "operator launch (general mesh) failed: %s", cudaGetErrorString(ec));
        }
        if (nh > 0)
            k_gen_rows_times_block<<<grid, rows, 0, st>>>(Y, m->d_Yh, m->gtr.bptr, m->gtr.bcol, m->gtr.bw, m->gtr.brow, m->gtr.out,
                                                          m->gtr.nb, B, alpha_h, 1, nullptr);
        CUDA_TRY(cudaGetLastError());
        m->launches += (int64_t)m->colour_off.size() - 1 + (nh > 0 ? 1 : 0) + (init_kernel ? 1 : 0);
        return FE_OK;
    }
    cudaError_t e = box ? launch_apply_gbox(bp, m->p, m->ncells, m->sms, st) : launch_apply_gen(prm, m->p, m->ncells, m->sms, st);
    if (e != cudaSuccess) return fail(FE_ERR_CUDA, "operator launch (general mesh) failed: %s", cudaGetErrorString(e));
    if (nh > 0)
        k_gen_collapse<<<grid, rows, 0, st>>>(Y, m->d_Yh, m->gexp.bptr, m->gexp.bcol, m->gexp.bw, m->gexp.brow, m->gexp.out, m->gexp.nb, B,
                                              alpha_h);
    CUDA_TRY(cudaGetLastError());
    m->launches += (nh > 0 ? 2 : 1) + (init_kernel ? 1 : 0);  // cell kernel, collapse, k_gen_init (memsets are not counted)
    return FE_OK;
}

// ---- TMA path (fe_apply_tma.cuh) -----------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        cudaDriverEntryPointQueryResult qr;
        void* p = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// the block as a 4-D tensor (j, gx, gy, gz) of doubles with a box of (bt, bx, by, bz) elements
static int make_map(CUtensorMap* out, const fe_mesh* m, const double* base, int B, int bt, int bx, int by, int bz)
{
    EncodeTiledFn enc = encode_fn();
    if (!enc) return fail(FE_ERR_CUDA, "cuTensorMapEncodeTiled not available from this driver");
    cuuint64_t dims[4] = {(cuuint64_t)B, (cuuint64_t)m->Nx, (cuuint64_t)m->Ny, (cuuint64_t)m->Nz};
    cuuint64_t strides[3] = {(cuuint64_t)B * 8, (cuuint64_t)B * 8 * m->Nx, (cuuint64_t)B * 8 * m->Nx * m->Ny};
    cuuint32_t box[4] = {(cuuint32_t)bt, (cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz}, es[4] = {1, 1, 1, 1};
    CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)base, dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(FE_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
    return FE_OK;
}

// the three views of one block the TMA kernel uses
struct BlockMaps {
    CUtensorMap n3, h1, h2, p1;  // tile load; the two row halves of an output plane; owner sub-plane
};

static int make_block_maps(BlockMaps* bm, const fe_mesh* m, const double* base, int B)
{
    const int bt = tma_bt(m->p, m->variant, B), n = m->n, p = m->p;
    int rc;
    if ((rc = make_map(&bm->n3, m, base, B, bt, n, n, n))) return rc;
    if ((rc = make_map(&bm->h1, m, base, B, bt, n, (n + 1) / 2, 1))) return rc;
    if ((rc = make_map(&bm->h2, m, base, B, bt, n, n / 2 > 0 ? n / 2 : 1, 1))) return rc;
    return make_map(&bm->p1, m, base, B, bt, p, p, 1);
}

// bulk tensor copies need 16-byte aligned bases and row pitches (B even)
static bool tma_eligible(const fe_mesh* m, int B, const void* a, const void* b, const void* c)
{
    if (m->kind || m->variant == 3 || m->variant == 4) return false;
    if (B % 2 != 0 || !encode_fn()) return false;
    return (((uintptr_t)a | (uintptr_t)b | (uintptr_t)c) & 15) == 0;
}

static void fill_tma_params(const fe_mesh* m, TmaParams* prm, int B)
{
    memset(prm, 0, sizeof(*prm));
    prm->rec = m->d_VZ;
    prm->B = B; prm->cx = m->cx; prm->cy = m->cy; prm->cz = m->cz;
    // blocked walk (fe_apply_tma.cuh: walk_cell): the largest block edge T in {8, 4, 2} that divides cy and cz and keeps
    // T rows of cells (their X and Y tiles) within about half of the 126 MB L2; T = 1 when a whole x-y slab fits anyway
    const double cell_bytes = (double)m->nc * B * 16.0;
    prm->blk = 1;
    if ((double)m->cx * m->cy * cell_bytes > 64.0e6)
        for (int T = 8; T >= 2; T /= 2)
            if (m->cy % T == 0 && m->cz % T == 0 && (double)T * m->cx * cell_bytes <= 64.0e6) { prm->blk = T; break; }
    prm->eoN = m->eoN; prm->eoNT = m->eoNT; prm->eoG = m->eoG;
}

// Y += alpha s sum_e yhat_e(X) + kappa X (owner),  W = beta_next X (pre-initialisation of the next target), one launch
static int tma_step(fe_mesh* m, const BlockMaps& X, const BlockMaps& Y, const BlockMaps* W, int B, const double* eps,
                    double alpha, double c, bool owner, double beta_next, bool first, cudaStream_t st,
                    double* dots = nullptr)
{
    TmaParams prm;
    fill_tma_params(m, &prm, B);
    prm.dots = dots;
    prm.mXn = X.n3; prm.mYh1 = Y.h1; prm.mYh2 = Y.h2; prm.mYp1 = Y.p1; prm.mWp1 = W ? W->p1 : Y.p1;
    prm.eps = eps; prm.alpha = alpha; prm.c = c; prm.owner = owner ? 1 : 0;
    prm.preinit = W ? 1 : 0; prm.beta_next = beta_next;
    prm.eoNTa = m->eoNT;
    for (double& x : prm.eoNTa.S) x *= alpha;
    for (double& x : prm.eoNTa.A) x *= alpha;
    for (double& x : prm.eoNTa.Mid) x *= alpha;
    cudaError_t e = launch_apply_tma(prm, m->p, m->ncells, first, st, m->variant, m->sms);
    if (e != cudaSuccess) return fail(FE_ERR_CUDA, "operator launch failed: %s", cudaGetErrorString(e));
    m->launches += 1;
    return FE_OK;
}

__global__ void k_zero_masked_rows(double* __restrict__ Y, const double* __restrict__ s, long long N, int B)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N * B; i += (long long)gridDim.x * blockDim.x)
        if (s[i / B] == 0.0) Y[i] = 0.0;
}

static int zero_faces(fe_mesh* m, double* Y, int B, cudaStream_t st)
{
    if (m->kind) {  // no tensor structure: the Dirichlet rows are those with s_g = 0
        k_zero_masked_rows<<<m->sms * 8, 256, 0, st>>>(Y, m->d_sm, m->N, B);
        CUDA_TRY(cudaGetLastError());
        m->launches += 1;
        return FE_OK;
    }
    k_zero_faces<<<m->sms * 4, 256, 0, st>>>(Y, m->Nx, m->Ny, m->Nz, B);
    CUDA_TRY(cudaGetLastError());
    m->launches += 1;
    return FE_OK;
}

static bool overlap(const double* a, size_t na, const double* b, size_t nb)
{
    return a < b + nb && b < a + na;
}

int fe_apply_H(fe_mesh* m, const double* X, double* Y, int B, const double* eps_dev, void* cuda_stream)
{
    if (!m || !X || !Y) return fail(FE_ERR_INVALID, "fe_apply_H: NULL argument");
    if (B < 1) return fail(FE_ERR_INVALID, "fe_apply_H: B=%d < 1", B);
    if (!m->have_V) return fail(FE_ERR_STATE, "fe_apply_H: call fe_set_potential first");
    const size_t len = (size_t)m->N * B;
    if (overlap(X, len, Y, len)) return fail(FE_ERR_INVALID, "fe_apply_H: X and Y overlap");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (tma_eligible(m, B, X, Y, eps_dev)) {
        BlockMaps mx, my;
        int rc;
        if ((rc = make_block_maps(&mx, m, X, B)) || (rc = make_block_maps(&my, m, Y, B))) return rc;
        // The zero-fill stays a plain memset in front of the kernel.  Measured (cfg 5): clearing Y chunk by
        // chunk from a concurrent kernel (programmatic dependent launch + per-chunk flags) gave no overlap at all, and even a
        // memset on an unrelated stream costs the operator kernel 18 of its own 22 us -- the two contend for HBM, so the
        // zero-fill can only be removed as BYTES, not hidden.
        CUDA_TRY(cudaMemsetAsync(Y, 0, len * sizeof(double), st));
        return tma_step(m, mx, my, nullptr, B, eps_dev, 1.0, 0.0, eps_dev != nullptr, 0.0, true, st);
    }
    return operator_step(m, X, nullptr, Y, B, eps_dev, 1.0, 0.0, 0.0, st);
}

// fe_apply_H into a block the caller has already cleared (the library's own loops let the elementwise kernel that reads a
// block last also clear it, so the separate zero-fill pass disappears); falls back to fe_apply_H when the TMA path is not taken
// dots_dev (B doubles, zero on entry) receives the column-wise x_j . y_j: from the operator kernel itself on the TMA path
// (cell-local terms, fe_apply_tma.cuh DOTS), from one extra pass otherwise
static int apply_into_cleared(fe_mesh* m, const double* X, double* Y, int B, const double* eps_dev, double* dots_dev,
                              void* cuda_stream)
{
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!tma_eligible(m, B, X, Y, eps_dev)) {
        // general mesh of box cells: the cell kernel adds into the cleared block (owner terms inside), no second zero-fill
        int rc = general_fused(m) ? general_step(m, X, nullptr, Y, B, eps_dev, 1.0, 0.0, 0.0, st, nullptr, 0.0, true)
                                  : fe_apply_H(m, X, Y, B, eps_dev, cuda_stream);
        if (rc || !dots_dev) return rc;
        k_col_dot<<<m->sms * 8, dim3(kMRx, kMRy), 0, st>>>(X, Y, m->N, B, dots_dev);
        CUDA_TRY(cudaGetLastError());
        m->launches += 1;
        return FE_OK;
    }
    BlockMaps mx, my;
    int rc;
    if ((rc = make_block_maps(&mx, m, X, B)) || (rc = make_block_maps(&my, m, Y, B))) return rc;
    return tma_step(m, mx, my, nullptr, B, eps_dev, 1.0, 0.0, eps_dev != nullptr, 0.0, true, st, dots_dev);
}

int fe_apply_H_chain(fe_mesh* m, const double* X, double* Y, double* Ynext, int B, const double* eps_dev, int y_is_clear,
                     void* cuda_stream)
{
    if (!m || !X || !Y) return fail(FE_ERR_INVALID, "fe_apply_H_chain: NULL argument");
    if (B < 1) return fail(FE_ERR_INVALID, "fe_apply_H_chain: B=%d < 1", B);
    if (!m->have_V) return fail(FE_ERR_STATE, "fe_apply_H_chain: call fe_set_potential first");
    const size_t len = (size_t)m->N * B;
    if (overlap(X, len, Y, len) || (Ynext && (overlap(X, len, Ynext, len) || overlap(Y, len, Ynext, len))))
        return fail(FE_ERR_INVALID, "fe_apply_H_chain: X, Y and Ynext must not overlap");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (m->kind == 0 && tma_eligible(m, B, X, Y, eps_dev) && (!Ynext || tma_eligible(m, B, Ynext, Ynext, Ynext))) {
        // the clearing of the NEXT target rides on this launch as the pre-initialisation store (beta' = 0) of the owner boxes;
        // the far boundary faces, which no owner box covers, are cleared by k_zero_faces
        BlockMaps mx, my, mw;
        int rc;
        if ((rc = make_block_maps(&mx, m, X, B)) || (rc = make_block_maps(&my, m, Y, B))) return rc;
        if (Ynext && (rc = make_block_maps(&mw, m, Ynext, B))) return rc;
        if (!y_is_clear) CUDA_TRY(cudaMemsetAsync(Y, 0, len * sizeof(double), st));
        if (Ynext && (rc = zero_faces(m, Ynext, B, st))) return rc;
        return tma_step(m, mx, my, Ynext ? &mw : nullptr, B, eps_dev, 1.0, 0.0, eps_dev != nullptr, 0.0, true, st);
    }
    if (general_fused(m)) {
        // general mesh of box cells: the owner cells of k_apply_gbox store 0 into every row of the next target (beta' = 0)
        if (!y_is_clear) CUDA_TRY(cudaMemsetAsync(Y, 0, len * sizeof(double), st));
        return general_step(m, X, nullptr, Y, B, eps_dev, 1.0, 0.0, 0.0, st, Ynext, 0.0, true);
    }
    // other paths (general meshes with deformed cells, odd B, unaligned blocks): plain apply, then clear the next target
    int rc = fe_apply_H(m, X, Y, B, eps_dev, cuda_stream);
    if (rc) return rc;
    if (Ynext) CUDA_TRY(cudaMemsetAsync(Ynext, 0, len * sizeof(double), st));
    return FE_OK;
}

int cheb_filter(fe_mesh* m, double* X, int B, int deg, double a, double b, double a0, double* work, void* cuda_stream)
{
    if (!m || !X || !work) return fail(FE_ERR_INVALID, "cheb_filter: NULL argument");
    if (B < 1 || deg < 1) return fail(FE_ERR_INVALID, "cheb_filter: need B >= 1 and degree >= 1 (B=%d, m=%d)", B, deg);
    if (!(a0 < a && a < b) || !std::isfinite(a0) || !std::isfinite(b))
        return fail(FE_ERR_INVALID, "cheb_filter: need a0 < a < b (a0=%g a=%g b=%g)", a0, a, b);
    if (!m->have_V) return fail(FE_ERR_STATE, "cheb_filter: call fe_set_potential first");
    const size_t len = (size_t)m->N * B;
    if (overlap(X, len, work, 2 * len)) return fail(FE_ERR_INVALID, "cheb_filter: work overlaps X");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // l.208-210 / R7.  Three blocks rotate: Y_k lives in buf[k % 3], buf = {X, work, work + N*B}.
    double* buf[3] = {X, work, work + len};
    const double e = 0.5 * (b - a), c = 0.5 * (b + a);
    const double sigma1 = e / (a0 - c);
    double sigma = sigma1;
    if (tma_eligible(m, B, X, work, work + len)) {
        // Pre-initialised recurrence: step k adds alpha_k (H~ - c) Y_k into buf[(k+1)%3], which step k-1 filled with
        // beta_k Y_{k-1}; it stores beta_{k+1} Y_k into buf[(k+2)%3].  No zero-fill or read of Y_{k-1} per step.
        BlockMaps bm[3];
        int rc;
        for (int i = 0; i < 3; ++i)
            if ((rc = make_block_maps(&bm[i], m, buf[i], B))) return rc;
        CUDA_TRY(cudaMemsetAsync(buf[1], 0, len * sizeof(double), st));
        if ((rc = zero_faces(m, buf[0], B, st)) || (rc = zero_faces(m, buf[2], B, st))) return rc;
        double s_cur = sigma1;  // sigma_{k+1} at iteration k
        for (int k = 0; k < deg; ++k) {
            const double s_next = 1.0 / (2.0 / sigma1 - s_cur);  // sigma_{k+2}
            const double alpha = (k == 0) ? s_cur / e : 2.0 * s_cur / e;
            const bool pre = k + 1 < deg;  // beta_{k+1} = -sigma_{k+1} sigma_{k+2}
            rc = tma_step(m, bm[k % 3], bm[(k + 1) % 3], pre ? &bm[(k + 2) % 3] : nullptr, B, nullptr, alpha, c, true,
                          -s_cur * s_next, k == 0, st);
            if (rc) return rc;
            s_cur = s_next;
        }
        if (deg % 3 != 0) CUDA_TRY(cudaMemcpyAsync(X, buf[deg % 3], len * sizeof(double), cudaMemcpyDeviceToDevice, st));
        return FE_OK;
    }
    if (general_fused(m)) {
        // general mesh of box cells: the pre-initialised recurrence of the TMA path through the owner cells of k_apply_gbox
        // (every unconstrained node has an owner, Dirichlet rows are stored as 0: no face clears)
        double s_cur = sigma1;
        for (int k = 0; k < deg; ++k) {  // step 0 clears its own target
            const double s_next = 1.0 / (2.0 / sigma1 - s_cur);
            const double alpha = (k == 0) ? s_cur / e : 2.0 * s_cur / e;
            const bool pre = k + 1 < deg;
            int rcg = general_step(m, buf[k % 3], nullptr, buf[(k + 1) % 3], B, nullptr, alpha, 0.0, c, st,
                                   pre ? buf[(k + 2) % 3] : nullptr, -s_cur * s_next, k > 0);
            if (rcg) return rcg;
            s_cur = s_next;
        }
        if (deg % 3 != 0) CUDA_TRY(cudaMemcpyAsync(X, buf[deg % 3], len * sizeof(double), cudaMemcpyDeviceToDevice, st));
        return FE_OK;
    }
    int rc = operator_step(m, buf[0], nullptr, buf[1], B, nullptr, sigma1 / e, 0.0, c, st);
    if (rc) return rc;
    for (int k = 1; k < deg; ++k) {
        const double sigma_next = 1.0 / (2.0 / sigma1 - sigma);
        rc = operator_step(m, buf[k % 3], buf[(k - 1) % 3], buf[(k + 1) % 3], B, nullptr, 2.0 * sigma_next / e,
                           -sigma * sigma_next, c, st);
        if (rc) return rc;
        sigma = sigma_next;
    }
    if (deg % 3 != 0) CUDA_TRY(cudaMemcpyAsync(X, buf[deg % 3], len * sizeof(double), cudaMemcpyDeviceToDevice, st));
    return FE_OK;
}

// ---- Rayleigh-Ritz (NEXT-1; Eq. 23-24 l.210-219; readings R8, R9) ------------------------------------------
// small dense helpers on the host (B <= 128): Cholesky S = L L^T, R = L^{-T}, tridiagonal QR for the symmetric B x B problem
static bool chol_lower(std::vector<double>& S, int B)
{
    for (int j = 0; j < B; ++j) {
        double d = S[(size_t)j * B + j];
        for (int k = 0; k < j; ++k) d -= S[(size_t)j * B + k] * S[(size_t)j * B + k];
        if (!(d > 0.0)) return false;
        d = std::sqrt(d);
        S[(size_t)j * B + j] = d;
        for (int i = j + 1; i < B; ++i) {
            double v = S[(size_t)i * B + j];
            for (int k = 0; k < j; ++k) v -= S[(size_t)i * B + k] * S[(size_t)j * B + k];
            S[(size_t)i * B + j] = v / d;
        }
    }
    return true;
}

// R = L^{-T} (upper triangular, row-major R[i*B+j]) from the lower factor stored in the lower triangle of L
static void inv_lower_transposed(const std::vector<double>& L, int B, std::vector<double>& R)
{
    std::vector<double> Li((size_t)B * B, 0.0);  // L^{-1}, lower
    for (int c = 0; c < B; ++c) {
        Li[(size_t)c * B + c] = 1.0 / L[(size_t)c * B + c];
        for (int i = c + 1; i < B; ++i) {
            double v = 0.0;
            for (int k = c; k < i; ++k) v -= L[(size_t)i * B + k] * Li[(size_t)k * B + c];
            Li[(size_t)i * B + c] = v / L[(size_t)i * B + i];
        }
    }
    R.assign((size_t)B * B, 0.0);
    for (int i = 0; i < B; ++i)
        for (int j = i; j < B; ++j) R[(size_t)i * B + j] = Li[(size_t)j * B + i];
}

// Symmetric B x B eigenproblem on the host: Householder reduction to tridiagonal form, then implicit-shift QR sweeps
// (Wilkinson shift, deflation from the bottom) with the rotations accumulated.  Eigenvalues ascending in w,
// eigenvectors in the COLUMNS of V (row-major V[i*B+k] = component i of vector k).  O(B^3), ~10x fewer flops than
// cyclic Jacobi, which dominated fe_rayleigh_ritz at B = 64.
static void sym_eigh(std::vector<double> A, int n, std::vector<double>& w, std::vector<double>& V)
{
    std::vector<double> Zt((size_t)n * n, 0.0);  // Zt[k*n + i] = component i of basis vector k
    for (int i = 0; i < n; ++i) Zt[(size_t)i * n + i] = 1.0;
    std::vector<double> v(n), pv(n);
    for (int k = 0; k + 2 < n; ++k) {  // reflector acting on indices k+1..n-1 zeroes A[k+2.., k]
        double nrm = 0.0;
        for (int i = k + 1; i < n; ++i) nrm += A[(size_t)i * n + k] * A[(size_t)i * n + k];
        nrm = std::sqrt(nrm);
        if (nrm == 0.0) continue;
        const double x0 = A[(size_t)(k + 1) * n + k];
        const double alpha = x0 > 0.0 ? -nrm : nrm;
        double vn = 0.0;
        for (int i = k + 1; i < n; ++i) {
            v[i] = A[(size_t)i * n + k] - (i == k + 1 ? alpha : 0.0);
            vn += v[i] * v[i];
        }
        if (vn == 0.0) continue;
        const double inv = 1.0 / std::sqrt(vn);
        for (int i = k + 1; i < n; ++i) v[i] *= inv;
        // A <- H A H, H = I - 2 v v^T: p = A v, K = v.p, q = p - K v, A -= 2 (v q^T + q v^T)
        double K = 0.0;
        for (int i = k; i < n; ++i) {
            double t = 0.0;
            for (int jx = k + 1; jx < n; ++jx) t += A[(size_t)i * n + jx] * v[jx];
            pv[i] = t;
        }
        for (int i = k + 1; i < n; ++i) K += v[i] * pv[i];
        // column/row k: only the reflector's action on A[k+1.., k] matters: it becomes (alpha, 0, ..., 0)
        for (int i = k + 1; i < n; ++i) {
            const double val = (i == k + 1) ? alpha : 0.0;
            A[(size_t)i * n + k] = val;
            A[(size_t)k * n + i] = val;
        }
        for (int i = k + 1; i < n; ++i) pv[i] -= K * v[i];
        for (int i = k + 1; i < n; ++i)
            for (int jx = k + 1; jx < n; ++jx) A[(size_t)i * n + jx] -= 2.0 * (v[i] * pv[jx] + pv[i] * v[jx]);
        // Z <- Z H on the basis:  Z[:, j] -= 2 (Z v) v_j
        for (int i = 0; i < n; ++i) pv[i] = 0.0;
        for (int jx = k + 1; jx < n; ++jx)
            for (int i = 0; i < n; ++i) pv[i] += Zt[(size_t)jx * n + i] * v[jx];
        for (int jx = k + 1; jx < n; ++jx)
            for (int i = 0; i < n; ++i) Zt[(size_t)jx * n + i] -= 2.0 * pv[i] * v[jx];
    }
    std::vector<double> d(n), e(n > 1 ? n - 1 : 0);
    for (int i = 0; i < n; ++i) d[i] = A[(size_t)i * n + i];
    for (int i = 0; i + 1 < n; ++i) e[i] = A[(size_t)(i + 1) * n + i];
    const double eps = 2.220446049250313e-16;
    int hi = n - 1, guard = 0;
    while (hi > 0 && guard < 100 * n) {
        if (std::fabs(e[hi - 1]) <= eps * (std::fabs(d[hi - 1]) + std::fabs(d[hi]))) {
            e[hi - 1] = 0.0;
            --hi;
            continue;
        }
        ++guard;
        int lo = hi - 1;
        while (lo > 0 && std::fabs(e[lo - 1]) > eps * (std::fabs(d[lo - 1]) + std::fabs(d[lo]))) --lo;
        const double dd = 0.5 * (d[hi - 1] - d[hi]), eh = e[hi - 1];
        const double mu = d[hi] - eh * eh / (dd + (dd >= 0.0 ? 1.0 : -1.0) * std::hypot(dd, eh));
        double x = d[lo] - mu, z = e[lo];
        for (int k = lo; k < hi; ++k) {
            const double r = std::hypot(x, z);
            const double c = r > 0.0 ? x / r : 1.0, sn = r > 0.0 ? z / r : 0.0;
            if (k > lo) e[k - 1] = r;
            const double a = d[k], b = e[k], dn = d[k + 1];
            d[k] = c * c * a + 2.0 * c * sn * b + sn * sn * dn;
            d[k + 1] = sn * sn * a - 2.0 * c * sn * b + c * c * dn;
            e[k] = c * sn * (dn - a) + (c * c - sn * sn) * b;
            x = e[k];
            if (k + 1 < hi) {
                z = sn * e[k + 1];
                e[k + 1] = c * e[k + 1];
            }
            double* q0 = &Zt[(size_t)k * n];
            double* q1 = &Zt[(size_t)(k + 1) * n];
            for (int i = 0; i < n; ++i) {
                const double u0 = q0[i], u1 = q1[i];
                q0[i] = c * u0 + sn * u1;
                q1[i] = -sn * u0 + c * u1;
            }
        }
    }
    std::vector<int> idx(n);
    for (int i = 0; i < n; ++i) idx[i] = i;
    std::sort(idx.begin(), idx.end(), [&](int a, int b) { return d[a] < d[b]; });
    w.resize(n);
    V.assign((size_t)n * n, 0.0);
    for (int k = 0; k < n; ++k) {
        w[k] = d[idx[k]];
        for (int i = 0; i < n; ++i) V[(size_t)i * n + k] = Zt[(size_t)idx[k] * n + i];
    }
}

// one CholQR pass: S = Y^T Y (device) -> L, R = L^{-T} (host) -> Y <- Y R (device)
static int cholqr_pass(fe_mesh* m, double* Y, int B, cudaStream_t st)
{
    const size_t bb = (size_t)B * B;
    CUDA_TRY(cudaMemsetAsync(m->d_small, 0, bb * sizeof(double), st));
    CUDA_TRY(launch_gram(Y, Y, m->N, B, m->d_small, m->sms, st));
    std::vector<double> S(bb), R;
    CUDA_TRY(cudaMemcpyAsync(S.data(), m->d_small, bb * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    for (int i = 0; i < B; ++i)
        for (int j = 0; j < i; ++j) S[(size_t)i * B + j] = S[(size_t)j * B + i] = 0.5 * (S[(size_t)i * B + j] + S[(size_t)j * B + i]);
    if (!chol_lower(S, B)) return fail(FE_ERR_STATE, "fe_rayleigh_ritz: Y^T Y is not positive definite (rank-deficient block)");
    inv_lower_transposed(S, B, R);
    CUDA_TRY(cudaMemcpyAsync(m->d_small + bb, R.data(), bb * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(launch_rightmul(Y, m->d_small + bb, Y, 0, m->N, B, m->sms, st));
    CUDA_TRY(cudaStreamSynchronize(st));  // R is a host temporary
    m->launches += 2;
    return FE_OK;
}

int fe_rayleigh_ritz(fe_mesh* m, double* Y, int B, double* theta_host, double* work, void* cuda_stream)
{
    if (!m || !Y || !theta_host || !work) return fail(FE_ERR_INVALID, "fe_rayleigh_ritz: NULL argument");
    if (B < 1 || B > 128) return fail(FE_ERR_INVALID, "fe_rayleigh_ritz: B=%d outside 1..128", B);
    if (!m->have_V) return fail(FE_ERR_STATE, "fe_rayleigh_ritz: call fe_set_potential first");
    const size_t len = (size_t)m->N * B, bb = (size_t)B * B;
    if (overlap(Y, len, work, len)) return fail(FE_ERR_INVALID, "fe_rayleigh_ritz: work overlaps Y");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!m->d_small) CUDA_TRY(cudaMalloc((void**)&m->d_small, 2 * 128 * 128 * sizeof(double)));
    int rc;
    if ((rc = zero_faces(m, Y, B, st))) return rc;                          // R5: Dirichlet rows do not take part
    if ((rc = cholqr_pass(m, Y, B, st)) || (rc = cholqr_pass(m, Y, B, st))) return rc;  // R9: CholQR2, Y is now Q
    if ((rc = fe_apply_H(m, Y, work, B, nullptr, cuda_stream))) return rc;  // H~ Q
    CUDA_TRY(cudaMemsetAsync(m->d_small, 0, bb * sizeof(double), st));
    CUDA_TRY(launch_gram(Y, work, m->N, B, m->d_small, m->sms, st));        // R8: H~_Y = Q^T H~ Q
    std::vector<double> G(bb), w, V;
    CUDA_TRY(cudaMemcpyAsync(G.data(), m->d_small, bb * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    for (int i = 0; i < B; ++i)
        for (int j = 0; j < i; ++j) G[(size_t)i * B + j] = G[(size_t)j * B + i] = 0.5 * (G[(size_t)i * B + j] + G[(size_t)j * B + i]);
    sym_eigh(G, B, w, V);
    for (int k = 0; k < B; ++k) theta_host[k] = w[k];
    CUDA_TRY(cudaMemcpyAsync(m->d_small + bb, V.data(), bb * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(launch_rightmul(Y, m->d_small + bb, Y, 0, m->N, B, m->sms, st));     // X = Q V
    CUDA_TRY(cudaStreamSynchronize(st));
    m->launches += 2;
    return FE_OK;
}

// ---- block preconditioned MINRES around the shifted apply (NEXT-2; Eq. 20 l.183) ----------------
// per-axis diagonals of the Gauss-quadrature 1-D stiffness (2/h) N^T G N and mass (h/2) N^T W N, assembled over cells
static void axis_diagonals(const fe_mesh* m, const std::vector<double>& e, int c, std::vector<double>& kd, std::vector<double>& md)
{
    const int n = m->n, p = m->p;
    std::vector<double> kh(n, 0.0), mh(n, 0.0);
    for (int a = 0; a < n; ++a)
        for (int q = 0; q < n; ++q) {
            mh[a] += m->tab.gl_w[q] * m->tab.N[q * n + a] * m->tab.N[q * n + a];
            for (int r = 0; r < n; ++r) kh[a] += m->tab.N[q * n + a] * m->tab.G[q * n + r] * m->tab.N[r * n + a];
        }
    kd.assign((size_t)c * p + 1, 0.0);
    md.assign((size_t)c * p + 1, 0.0);
    for (int ec = 0; ec < c; ++ec) {
        const double h = e[ec + 1] - e[ec];
        for (int a = 0; a < n; ++a) {
            kd[(size_t)ec * p + a] += 2.0 / h * kh[a];
            md[(size_t)ec * p + a] += 0.5 * h * mh[a];
        }
    }
}

__global__ void k_nonzero_to_one(double* __restrict__ a, long long n)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        a[i] = a[i] != 0.0 ? 1.0 : 0.0;
}

// general mesh (reading R27): Minv_i = M_c,ii / d_i with d_i = kd_i + sum_h C_hi^2 kd_h, kd the diagonal of the assembled
// kinetic matrix 1/2 K over all nodes -- the diagonal of C^T (1/2 K) C without the couplings between hanging nodes
static int ensure_minres_tables_general(fe_mesh* m)
{
    const GeneralHost& g = *m->gh;
    const int n = m->n;
    GenDiagTables tb;
    memset(&tb, 0, sizeof(tb));
    for (int q = 0; q < n; ++q)
        for (int a = 0; a < n; ++a) {
            tb.Nt[q * n + a] = m->tab.N[q * n + a];
            double d = 0.0;
            for (int r = 0; r < n; ++r) d += m->tab.D[q * n + r] * m->tab.N[r * n + a];  // l_a'(gl_q)
            tb.DNt[q * n + a] = d;
        }
    double* d_kd = nullptr;
    CUDA_TRY(cudaMalloc((void**)&d_kd, (size_t)g.N_all * sizeof(double)));
    cudaError_t ce = cudaMemset(d_kd, 0, (size_t)g.N_all * sizeof(double));
    std::vector<double> kd((size_t)g.N_all), minv((size_t)g.N), mask((size_t)g.N);
    if (ce == cudaSuccess) {
        k_gen_kinetic_diag<<<m->sms * 8, 256>>>(d_kd, m->d_gmetric, m->d_gl2g, m->ncells, n, gen_rec_doubles(n), tb);
        ce = cudaMemcpy(kd.data(), d_kd, kd.size() * sizeof(double), cudaMemcpyDeviceToHost);
    }
    cudaFree(d_kd);
    if (ce != cudaSuccess) return fail(FE_ERR_CUDA, "fe_minres_shifted: building the preconditioner failed: %s", cudaGetErrorString(ce));
    m->launches += 1;
    std::vector<double> d(kd.begin(), kd.begin() + g.N);
    for (int64_t r = 0; r < g.N_all - g.N; ++r)
        for (int64_t k = g.crow[r]; k < g.crow[r + 1]; ++k) d[g.ccol[k]] += g.cval[k] * g.cval[k] * kd[g.N + r];
    for (int64_t i = 0; i < g.N; ++i) {
        mask[i] = g.mask[i] ? 1.0 : 0.0;
        minv[i] = g.mask[i] ? g.mass[i] / d[i] : 0.0;
    }
    int rc;
    if ((rc = upload(&m->d_minv, minv)) || (rc = upload(&m->d_mask, mask))) return rc;
    CUDA_TRY(cudaMalloc((void**)&m->d_scal, 21 * 128 * sizeof(double)));
    return FE_OK;
}

static int ensure_minres_tables(fe_mesh* m)
{
    if (m->d_minv) return FE_OK;
    if (m->kind) return ensure_minres_tables_general(m);
    std::vector<double> k[3], md[3];
    axis_diagonals(m, m->xe, m->cx, k[0], md[0]);
    axis_diagonals(m, m->ye, m->cy, k[1], md[1]);
    axis_diagonals(m, m->ze, m->cz, k[2], md[2]);
    double* d[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int rc = FE_OK;
    for (int i = 0; i < 3 && !rc; ++i) {
        rc = upload(&d[i], k[i]);
        if (!rc) rc = upload(&d[3 + i], md[i]);
    }
    cudaError_t ce = cudaSuccess;
    if (!rc) ce = cudaMalloc((void**)&m->d_minv, (size_t)m->N * sizeof(double));
    if (!rc && ce == cudaSuccess) ce = cudaMalloc((void**)&m->d_mask, (size_t)m->N * sizeof(double));
    if (!rc && ce == cudaSuccess) ce = cudaMalloc((void**)&m->d_scal, 21 * 128 * sizeof(double));
    if (!rc && ce == cudaSuccess) {
        k_build_precond<<<m->sms * 8, 256>>>(m->d_minv, m->Nx, m->Ny, m->Nz, d[0], d[1], d[2], d[3], d[4], d[5], m->d_sx, m->d_sy, m->d_sz);
        k_build_scaling<<<m->sms * 8, 256>>>(m->d_sx, m->d_sy, m->d_sz, m->Nx, m->Ny, m->Nz, m->d_mask);
        k_nonzero_to_one<<<m->sms * 4, 256>>>(m->d_mask, m->N);  // mu M^{-1/2} -> {0, 1}
        ce = cudaDeviceSynchronize();
        m->launches += 2;
    }
    for (double* q : d) cudaFree(q);
    if (rc) return rc;
    if (ce != cudaSuccess) return fail(FE_ERR_CUDA, "fe_minres_shifted: building the preconditioner failed: %s", cudaGetErrorString(ce));
    return FE_OK;
}

int fe_minres_shifted(fe_mesh* m, const double* G, double* X, int B, const double* eps_dev, int maxit, double tol,
                      int precondition, double* relres_host, int* iters_host, double* work, void* cuda_stream)
{
    if (!m || !G || !X || !work) return fail(FE_ERR_INVALID, "fe_minres_shifted: NULL argument");
    if (B < 1 || B > 128) return fail(FE_ERR_INVALID, "fe_minres_shifted: B=%d outside 1..128", B);
    if (maxit < 1 || !(tol >= 0.0)) return fail(FE_ERR_INVALID, "fe_minres_shifted: need maxit >= 1 and tol >= 0");
    if (!m->have_V) return fail(FE_ERR_STATE, "fe_minres_shifted: call fe_set_potential first");
    const size_t len = (size_t)m->N * B;
    if (overlap(X, len, work, 6 * len) || overlap(G, len, work, 6 * len) || overlap(G, len, X, len))
        return fail(FE_ERR_INVALID, "fe_minres_shifted: G, X and work must not overlap");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = ensure_minres_tables(m);
    if (rc) return rc;
    const double* Minv = precondition ? m->d_minv : m->d_mask;
    double *R1 = work, *R2 = work + len, *Y = work + 2 * len, *HY = work + 3 * len, *W1 = work + 4 * len, *W2 = work + 5 * len;
    MinresScalars q;
    double* s = m->d_scal;
    double** f[] = {&q.beta, &q.oldb, &q.alfa, &q.betasq, &q.dbar, &q.epsln, &q.oldeps, &q.phibar, &q.cs, &q.sn,
                    &q.gamma, &q.delta, &q.phi, &q.beta1, &q.s, &q.c1, &q.c2, &q.dot, &q.gam, &q.gamn, &q.sv};
    for (int i = 0; i < 21; ++i) *f[i] = s + (size_t)i * 128;
    const int grid = m->sms * 8;
    const dim3 blk(kMRx, kMRy);
    // even B and 16-byte aligned blocks: the two elementwise passes move 16 bytes per access
    const bool vec2 = B % 2 == 0 && (((uintptr_t)X | (uintptr_t)work) & 15) == 0;
    CUDA_TRY(cudaMemsetAsync(q.betasq, 0, 128 * sizeof(double), st));
    k_minres_init<<<grid, blk, 0, st>>>(G, Minv, R1, R2, Y, X, W1, W2, m->N, B, q.betasq);
    k_minres_scalars<<<1, 128, 0, st>>>(q, B, 0, tol);
    CUDA_TRY(cudaMemsetAsync(HY, 0, len * sizeof(double), st));  // later targets are cleared by k_minres_update
    m->launches += 3;
    std::vector<double> phibar(B), beta1(B);
    int it = 0;
    bool done = false;
    // the two blocks the apply alternates between: their tensor maps are encoded once, not every step
    const bool tma = tma_eligible(m, B, Y, HY, eps_dev);
    BlockMaps mapY, mapHY;
    if (tma && ((rc = make_block_maps(&mapY, m, Y, B)) || (rc = make_block_maps(&mapHY, m, HY, B)))) return rc;
    k_minres_scalars<<<1, 128, 0, st>>>(q, B, 1, tol);  // the later steps' s, c1 come from stage 2 of the step before
    m->launches += 1;
    while (it < maxit && !done) {
        // hy = (H~ - eps_j) y,  y = beta v, with dot_j = y_j . hy_j from the operator kernel
        if (tma)
            rc = tma_step(m, mapY, mapHY, nullptr, B, eps_dev, 1.0, 0.0, eps_dev != nullptr, 0.0, true, st, q.dot);
        else
            rc = apply_into_cleared(m, Y, HY, B, eps_dev, q.dot, cuda_stream);
        if (rc) return rc;
        k_minres_scalars<<<1, 128, 0, st>>>(q, B, 3, tol);
        if (vec2 && B <= 64)
            k_minres_lanczos2<1, 2><<<grid, blk, 0, st>>>((double2*)HY, (double2*)R1, (const double2*)R2, Minv, m->N, B, q.s, q.c1,
                                                          q.c2, q.betasq, q.gamn);
        else if (vec2)
            k_minres_lanczos2<2, 1><<<grid, blk, 0, st>>>((double2*)HY, (double2*)R1, (const double2*)R2, Minv, m->N, B, q.s, q.c1,
                                                          q.c2, q.betasq, q.gamn);
        else
            k_minres_lanczos<<<grid, blk, 0, st>>>(HY, R1, R2, Minv, m->N, B, q.s, q.c1, q.c2, q.betasq, q.gamn);
        k_minres_scalars<<<1, 128, 0, st>>>(q, B, 2, tol);
        if (vec2 && B <= 64)
            k_minres_update2<1, 2><<<grid, blk, 0, st>>>((double2*)Y, (double2*)W1, (const double2*)W2, (double2*)X, m->N, B, q.sv,
                                                         q.oldeps, q.delta, q.gamma, q.phi);
        else if (vec2)
            k_minres_update2<2, 1><<<grid, blk, 0, st>>>((double2*)Y, (double2*)W1, (const double2*)W2, (double2*)X, m->N, B, q.sv,
                                                         q.oldeps, q.delta, q.gamma, q.phi);
        else
            k_minres_update<<<grid, blk, 0, st>>>(Y, W1, W2, X, m->N, B, q.sv, q.oldeps, q.delta, q.gamma, q.phi);
        CUDA_TRY(cudaGetLastError());
        m->launches += 4;
        std::swap(Y, HY);  // the preconditioned residual of this step is the next step's y
        std::swap(mapY, mapHY);
        std::swap(R1, R2);
        std::swap(W1, W2);
        ++it;
        if (it % 8 == 0 || it == maxit) {
            CUDA_TRY(cudaMemcpyAsync(phibar.data(), q.phibar, B * sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaMemcpyAsync(beta1.data(), q.beta1, B * sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            done = true;
            for (int j = 0; j < B; ++j)
                if (beta1[j] > 0.0 && phibar[j] > tol * beta1[j]) done = false;
        }
    }
    if (relres_host)
        for (int j = 0; j < B; ++j) relres_host[j] = beta1[j] > 0.0 ? phibar[j] / beta1[j] : 0.0;
    if (iters_host) *iters_host = it;
    return FE_OK;
}

int fe_add_subspace(fe_mesh* m, const double* Psi, const double* D_host, double* P, int B, void* cuda_stream)
{
    if (!m || !Psi || !D_host || !P) return fail(FE_ERR_INVALID, "fe_add_subspace: NULL argument");
    if (B < 1 || B > 128) return fail(FE_ERR_INVALID, "fe_add_subspace: B=%d outside 1..128", B);
    const size_t len = (size_t)m->N * B, bb = (size_t)B * B;
    if (overlap(Psi, len, P, len)) return fail(FE_ERR_INVALID, "fe_add_subspace: Psi and P overlap");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!m->d_small) CUDA_TRY(cudaMalloc((void**)&m->d_small, 2 * 128 * 128 * sizeof(double)));
    CUDA_TRY(cudaMemcpyAsync(m->d_small + bb, D_host, bb * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(launch_rightmul(Psi, m->d_small + bb, P, 1, m->N, B, m->sms, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    m->launches += 1;
    return FE_OK;
}

int fe_gram(fe_mesh* m, const double* A, const double* Bm, int B, double* C_host, void* cuda_stream)
{
    if (!m || !A || !Bm || !C_host) return fail(FE_ERR_INVALID, "fe_gram: NULL argument");
    if (B < 1 || B > 128) return fail(FE_ERR_INVALID, "fe_gram: B=%d outside 1..128", B);
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bb = (size_t)B * B;
    if (!m->d_small) CUDA_TRY(cudaMalloc((void**)&m->d_small, 2 * 128 * 128 * sizeof(double)));
    CUDA_TRY(cudaMemsetAsync(m->d_small, 0, bb * sizeof(double), st));
    CUDA_TRY(launch_gram(A, Bm, m->N, B, m->d_small, m->sms, st));
    CUDA_TRY(cudaMemcpyAsync(C_host, m->d_small, bb * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    m->launches += 1;
    return FE_OK;
}

// ---- fe_gram without any allocation -------------------------------------------------------------------------------------
// The Gram kernels accumulate their B x B result with atomics in device memory; fe_gram keeps that accumulator in a
// cudaMalloc'ed buffer of the mesh.  Callers that must not allocate (code under CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc) get the same product with the accumulator in this file-scope array: 128 x 128 doubles = 128 KB
// that every GPU which loads the library holds until exit.  In host code the NAME of the array is a host-side stand-in, not
// a device address: the address the kernels get comes from cudaGetSymbolAddress, taken once per device with that device
// current.  All calls share the array (it keeps the last call's contents, so every call clears the part it uses); calls
// that overlap on one GPU -- two streams, two threads -- race on it.
constexpr int kGramStaticMaxB = 128;
static __device__ __align__(256) double g_gram_static[kGramStaticMaxB * kGramStaticMaxB];

static int gram_static_address(int device, double** out)
{
    static std::mutex mu;
    static double* addr[64] = {nullptr};  // per device: the symbol has one address on each GPU
    std::lock_guard<std::mutex> lock(mu);
    const bool tracked = device >= 0 && device < 64;
    if (tracked && addr[device]) {
        *out = addr[device];
        return FE_OK;
    }
    double* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_gram_static);  // the current device is `device` (set by the caller)
    if (e != cudaSuccess || !ptr)
        return fail(FE_ERR_CUDA, "fe_gram_static: cudaGetSymbolAddress failed on device %d: %s", device, cudaGetErrorString(e));
    if (tracked) addr[device] = ptr;
    *out = ptr;
    return FE_OK;
}

int fe_gram_static(fe_mesh* m, const double* A, const double* Bm, int B, double* C_host, void* cuda_stream)
{
    if (!m || !A || !Bm || !C_host) return fail(FE_ERR_INVALID, "fe_gram_static: NULL argument");
    if (B < 1 || B > kGramStaticMaxB)
        return fail(FE_ERR_INVALID, "fe_gram_static: B=%d outside 1..%d (the static accumulator holds %d x %d doubles)", B,
                    kGramStaticMaxB, kGramStaticMaxB, kGramStaticMaxB);
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* acc = nullptr;
    int rc = gram_static_address(m->device, &acc);
    if (rc) return rc;
    const size_t bb = (size_t)B * B;
    CUDA_TRY(cudaMemsetAsync(acc, 0, bb * sizeof(double), st));  // the array holds the previous call's product
    CUDA_TRY(launch_gram(A, Bm, m->N, B, acc, m->sms, st));
    CUDA_TRY(cudaMemcpyAsync(C_host, acc, bb * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    m->launches += 1;
    return FE_OK;
}

// ---- density at the quadrature points (NEXT-4; Eq. 4 l.73-77) ------------------------------------------------
int fe_density(fe_mesh* m, const double* X, int B, const double* f_dev, double* rho_dev, void* cuda_stream)
{
    if (!m || !X || !f_dev || !rho_dev) return fail(FE_ERR_INVALID, "fe_density: NULL argument");
    if (m->kind) {  // general mesh: expansion of the hanging values, then gather + interpolation + f psi^2 (fe_general.cuh)
        CUDA_TRY(cudaSetDevice(m->device));
        cudaStream_t gst = (cudaStream_t)cuda_stream;
        int rcg = general_expand(m, X, B, gst);
        if (rcg) return rcg;
        GenDensityParams gp;
        memset(&gp, 0, sizeof(gp));
        gp.X = X; gp.Xh = m->d_Xh ? m->d_Xh : X; gp.f = f_dev; gp.rho = rho_dev; gp.l2g = m->d_gl2g; gp.sc = m->d_gsc;
        gp.N = m->N; gp.B = B; gp.eoN = m->eoN;
        CUDA_TRY(cudaMemsetAsync(rho_dev, 0, (size_t)m->ncells * m->nc * sizeof(double), gst));
        CUDA_TRY(launch_density_gen(gp, m->p, m->ncells, gst));
        m->launches += 1;
        return FE_OK;
    }
    if (B < 1) return fail(FE_ERR_INVALID, "fe_density: B=%d < 1", B);
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DensityParams prm;
    memset(&prm, 0, sizeof(prm));
    prm.X = X; prm.f = f_dev; prm.sm = m->d_sm; prm.rho = rho_dev;
    prm.B = B; prm.cx = m->cx; prm.cy = m->cy; prm.cz = m->cz;
    prm.Nx = m->Nx; prm.NxNy = m->Nx * m->Ny;
    prm.eoN = m->eoN;
    for (int q = 0; q < m->n; ++q) prm.iw[q] = 1.0 / std::sqrt(m->tab.gl_w[q]);
    CUDA_TRY(cudaMemsetAsync(rho_dev, 0, (size_t)m->ncells * m->nc * sizeof(double), st));
    CUDA_TRY(launch_density(prm, m->p, m->ncells, st));
    m->launches += 1;
    return FE_OK;
}

// ---- spectral bounds for the filter: k Lanczos steps on H~ (reading R10; BASELINE config 1 "bounds from 20 Lanczos
//      steps").  Single vector: the applies take the legacy kernel (B = 1), the vector updates are three tiny kernels.
__global__ void k_lz_dot(const double* __restrict__ a, const double* __restrict__ b, long long n, double* out)
{
    double s = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) s = fma(a[i], b[i], s);
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ double red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
        atomicAdd(out, t);
    }
}
// w <- (w - a v - b u) * scale_w ;  optional masked copy-in: v0 -> v with Dirichlet rows zeroed
__global__ void k_lz_update(double* __restrict__ w, const double* __restrict__ v, const double* __restrict__ u, long long n,
                            double a, double b)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        w[i] = w[i] - a * v[i] - b * u[i];
}
__global__ void k_lz_scale(double* __restrict__ dst, const double* __restrict__ src, const double* __restrict__ mask,
                           long long n, double s)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        dst[i] = (mask && mask[i] == 0.0) ? 0.0 : s * src[i];
}

static int lz_dot(fe_mesh* m, const double* a, const double* b, double* out_host, cudaStream_t st)
{
    CUDA_TRY(cudaMemsetAsync(m->d_small, 0, sizeof(double), st));
    k_lz_dot<<<m->sms * 4, 256, 0, st>>>(a, b, m->N, m->d_small);
    CUDA_TRY(cudaMemcpyAsync(out_host, m->d_small, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    m->launches += 1;
    return FE_OK;
}

int fe_lanczos_bounds(fe_mesh* m, const double* v0_dev, int k, double* out3_host, double* work, void* cuda_stream)
{
    if (!m || !v0_dev || !out3_host || !work) return fail(FE_ERR_INVALID, "fe_lanczos_bounds: NULL argument");
    if (k < 1 || k > 128) return fail(FE_ERR_INVALID, "fe_lanczos_bounds: k=%d outside 1..128", k);
    if (!m->have_V) return fail(FE_ERR_STATE, "fe_lanczos_bounds: call fe_set_potential first");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!m->d_small) CUDA_TRY(cudaMalloc((void**)&m->d_small, 2 * 128 * 128 * sizeof(double)));
    const long long N = m->N;
    const int grid = m->sms * 4;
    double *v = work, *u = work + N, *w = work + 2 * N;  // v_j, v_{j-1}, w
    int rc;
    double nrm2 = 0.0;
    k_lz_scale<<<grid, 256, 0, st>>>(v, v0_dev, m->d_sm, N, 1.0);  // Dirichlet rows do not take part (R5)
    if ((rc = lz_dot(m, v, v, &nrm2, st))) return rc;
    if (!(nrm2 > 0.0)) return fail(FE_ERR_INVALID, "fe_lanczos_bounds: start vector is zero on the free rows");
    k_lz_scale<<<grid, 256, 0, st>>>(v, v, nullptr, N, 1.0 / std::sqrt(nrm2));
    CUDA_TRY(cudaMemsetAsync(u, 0, (size_t)N * sizeof(double), st));
    std::vector<double> al, be;
    double beta = 0.0;
    for (int j = 0; j < k; ++j) {
        if ((rc = fe_apply_H(m, v, w, 1, nullptr, cuda_stream))) return rc;
        double alpha = 0.0, b2 = 0.0;
        if ((rc = lz_dot(m, w, v, &alpha, st))) return rc;
        k_lz_update<<<grid, 256, 0, st>>>(w, v, u, N, alpha, beta);
        if ((rc = lz_dot(m, w, w, &b2, st))) return rc;
        beta = std::sqrt(b2);
        al.push_back(alpha);
        be.push_back(beta);
        m->launches += 2;
        if (beta == 0.0) break;
        k_lz_scale<<<grid, 256, 0, st>>>(w, w, nullptr, N, 1.0 / beta);
        double* t = u; u = v; v = w; w = t;  // v_{j-1} <- v_j <- w / beta
    }
    CUDA_TRY(cudaGetLastError());
    const int kk = (int)al.size();
    std::vector<double> T((size_t)kk * kk, 0.0), th, V;
    for (int i = 0; i < kk; ++i) {
        T[(size_t)i * kk + i] = al[i];
        if (i + 1 < kk) T[(size_t)i * kk + i + 1] = T[(size_t)(i + 1) * kk + i] = be[i];
    }
    sym_eigh(T, kk, th, V);
    out3_host[0] = th.front();
    out3_host[1] = th.back();
    out3_host[2] = be.back();
    return FE_OK;
}

// ---- host-buffer entry: the filter end to end (H2D, filter, D2H), column chunks pipelined on two streams -----------------
int cheb_filter_host(fe_mesh* m, double* X_host, int B, int deg, double a, double b, double a0)
{
    if (!m || !X_host) return fail(FE_ERR_INVALID, "cheb_filter_host: NULL argument");
    if (B < 1 || deg < 1) return fail(FE_ERR_INVALID, "cheb_filter_host: need B >= 1 and degree >= 1 (B=%d, m=%d)", B, deg);
    if (!(a0 < a && a < b)) return fail(FE_ERR_INVALID, "cheb_filter_host: need a0 < a < b");
    if (!m->have_V) return fail(FE_ERR_STATE, "cheb_filter_host: call fe_set_potential first");
    CUDA_TRY(cudaSetDevice(m->device));
    // columns are independent in the filter: chunks of 32 columns go through copy-in, filter, copy-out
    // on alternating streams, so the PCIe transfers of one chunk overlap the filter of the other.  What stays exposed is the
    // copy-in of the first chunk and the copy-out of the last: where 16-column tiles run well (p >= 6: the 16-wide launch
    // shape) the first and the last chunk are 16 columns wide, which halves that.
    std::vector<int> width;
    if (B % 32 == 0 && B > 32) {
        const bool edges16 = m->kind == 0 && m->p >= 6;
        if (edges16) width.push_back(16);
        for (int c = 0; c < B / 32 - (edges16 ? 1 : 0); ++c) width.push_back(32);
        if (edges16) width.push_back(16);
    } else {
        width.push_back(B);
    }
    const int nchunks = (int)width.size();
    const int BCmax = *std::max_element(width.begin(), width.end());
    const size_t clen = (size_t)m->N * BCmax;
    const int nbuf = nchunks > 1 ? 2 : 1;
    if (m->host_cap < clen * 3 * nbuf) {
        cudaFree(m->d_host);  // only the staging: d_WU / d_VZU belong to fe_apply_potential and stay valid
        m->d_host = nullptr;
        m->host_cap = 0;
        CUDA_TRY(cudaMalloc((void**)&m->d_host, clen * 3 * nbuf * sizeof(double)));
        m->host_cap = clen * 3 * nbuf;
    }
    for (int i = 0; i < 2; ++i)
        if (!m->hstream[i]) CUDA_TRY(cudaStreamCreateWithFlags(&m->hstream[i], cudaStreamNonBlocking));
    CUDA_TRY(cudaDeviceSynchronize());
    const size_t hp = (size_t)B * sizeof(double);
    int col = 0;
    for (int c = 0; c < nchunks; ++c) {
        const int BC = width[c];
        const size_t dp = (size_t)BC * sizeof(double), cl = (size_t)m->N * BC;
        cudaStream_t st = m->hstream[c % nbuf];
        double* Xd = m->d_host + (size_t)(c % nbuf) * 3 * clen;
        CUDA_TRY(cudaMemcpy2DAsync(Xd, dp, X_host + col, hp, dp, (size_t)m->N, cudaMemcpyHostToDevice, st));
        int rc = cheb_filter(m, Xd, BC, deg, a, b, a0, Xd + cl, (void*)st);
        if (rc) return rc;
        CUDA_TRY(cudaMemcpy2DAsync(X_host + col, hp, Xd, dp, dp, (size_t)m->N, cudaMemcpyDeviceToHost, st));
        col += BC;
    }
    for (int i = 0; i < nbuf; ++i) CUDA_TRY(cudaStreamSynchronize(m->hstream[i]));
    return FE_OK;
}

// ---- potential-only operator (first term of the adjoint right-hand side, Eq. 18 l.174-177) ----------------------------
int fe_apply_potential(fe_mesh* m, const double* Uq_dev, const double* X, double* Y, int B, void* cuda_stream)
{
    if (!m || !Uq_dev || !X || !Y) return fail(FE_ERR_INVALID, "fe_apply_potential: NULL argument");
    if (m->kind) {  // general mesh: the operator step on a scratch record array whose metric fields are 0 and whose WV is w |J| U
        if (!m->have_V) return fail(FE_ERR_STATE, "fe_apply_potential: call fe_set_potential first");
        const size_t lenk = (size_t)m->N * B;
        if (overlap(X, lenk, Y, lenk)) return fail(FE_ERR_INVALID, "fe_apply_potential: X and Y overlap");
        CUDA_TRY(cudaSetDevice(m->device));
        cudaStream_t gst = (cudaStream_t)cuda_stream;
        const int grec = gen_rec_doubles(m->n);
        if (!m->d_grecU) {
            CUDA_TRY(cudaMalloc((void**)&m->d_grecU, (size_t)m->ncells * grec * sizeof(double)));
            CUDA_TRY(cudaMemset(m->d_grecU, 0, (size_t)m->ncells * grec * sizeof(double)));
        }
        k_gen_weight_potential<<<m->sms * 8, 256, 0, gst>>>(m->d_grecU, Uq_dev, m->d_gwdet, m->ncells, m->nc, grec);
        CUDA_TRY(cudaGetLastError());
        m->launches += 1;
        double* keep = m->d_gmetric;
        m->d_gmetric = m->d_grecU;
        m->gbox_off = true;  // the potential-only operator goes through the generic kernel (zero metric)
        const int rcg = general_step(m, X, nullptr, Y, B, nullptr, 1.0, 0.0, 0.0, gst);
        m->gbox_off = false;
        m->d_gmetric = keep;
        return rcg;
    }
    if (B < 1) return fail(FE_ERR_INVALID, "fe_apply_potential: B=%d < 1", B);
    const size_t len = (size_t)m->N * B;
    if (overlap(X, len, Y, len)) return fail(FE_ERR_INVALID, "fe_apply_potential: X and Y overlap");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nq = (size_t)m->ncells * m->nc;
    if (!m->d_WU) {  // J w U of the field handed in, and a scratch record array for the kernel's other output
        CUDA_TRY(cudaMalloc((void**)&m->d_WU, nq * sizeof(double)));
        CUDA_TRY(cudaMalloc((void**)&m->d_VZU, (size_t)m->ncells * small_tile(m->n) * sizeof(double)));
    }
    ApplyParams prm;
    fill_params(m, &prm);
    launch_weight_potential(prm, m->p, Uq_dev, m->d_WU, m->d_VZU, m->ncells, m->sms, st);
    CUDA_TRY(cudaGetLastError());
    prm.X = X; prm.Z = nullptr; prm.Y = Y; prm.eps = nullptr; prm.B = B;
    prm.alpha = 1.0; prm.beta = 0.0; prm.c = 0.0;
    prm.WV = m->d_WU;
    prm.nokin = 1;
    int nl = 0;
    cudaError_t e = launch_apply(prm, m->p, 3, m->N, m->ncells, st, &nl);
    if (e != cudaSuccess) return fail(FE_ERR_CUDA, "fe_apply_potential: launch failed: %s", cudaGetErrorString(e));
    m->launches += 1 + nl;
    return FE_OK;
}

// ---- Ritz residuals and the residual-controlled ChFSI loop (NEXT-4; the eigenproblem residual is driven to
//      t_eig = e_L2^2 / c_eig; l.208-219 for the cycle itself) ------------------------------------------------------------------
__global__ void k_col_sumsq(const double* __restrict__ R, long long N, int B, double* out)
{
    double acc[kMaxColTiles] = {0, 0, 0, 0};
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += (long long)gridDim.x * kMRy)
#pragma unroll
        for (int t = 0; t < kMaxColTiles; ++t) {
            const int j = t * kMRx + threadIdx.x;
            if (j < B) {
                const double v = R[r * B + j];
                acc[t] = fma(v, v, acc[t]);
            }
        }
    block_col_reduce(acc, B, out);
}

int fe_ritz_residuals(fe_mesh* m, const double* X, const double* theta_host, int B, double* res_host, double* work,
                      void* cuda_stream)
{
    if (!m || !X || !theta_host || !res_host || !work) return fail(FE_ERR_INVALID, "fe_ritz_residuals: NULL argument");
    if (B < 1 || B > 128) return fail(FE_ERR_INVALID, "fe_ritz_residuals: B=%d outside 1..128", B);
    if (!m->have_V) return fail(FE_ERR_STATE, "fe_ritz_residuals: call fe_set_potential first");
    CUDA_TRY(cudaSetDevice(m->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!m->d_small) CUDA_TRY(cudaMalloc((void**)&m->d_small, 2 * 128 * 128 * sizeof(double)));
    double* d_theta = m->d_small + 128;  // [0,128): the sums; [128,256): theta
    CUDA_TRY(cudaMemcpyAsync(d_theta, theta_host, B * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemsetAsync(m->d_small, 0, B * sizeof(double), st));
    int rc = fe_apply_H(m, X, work, B, d_theta, cuda_stream);  // R_j = (H~ - theta_j I) x_j, Dirichlet rows 0 (Eq. 20)
    if (rc) return rc;
    k_col_sumsq<<<m->sms * 8, dim3(kMRx, kMRy), 0, st>>>(work, m->N, B, m->d_small);
    CUDA_TRY(cudaGetLastError());
    m->launches += 1;
    CUDA_TRY(cudaMemcpyAsync(res_host, m->d_small, B * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    for (int j = 0; j < B; ++j) res_host[j] = std::sqrt(std::max(res_host[j], 0.0));
    return FE_OK;
}

int fe_chfsi(fe_mesh* m, double* X, int B, int deg, double a, double b, double a0, double t_eig, int n_gate,
             int max_cycles, double* theta_host, double* res_host, int* cycles_host, double* work, void* cuda_stream)
{
    if (!m || !X || !theta_host || !res_host || !work) return fail(FE_ERR_INVALID, "fe_chfsi: NULL argument");
    if (B < 1 || B > 128) return fail(FE_ERR_INVALID, "fe_chfsi: B=%d outside 1..128", B);
    if (n_gate < 1 || n_gate > B) return fail(FE_ERR_INVALID, "fe_chfsi: n_gate=%d outside 1..B", n_gate);
    if (max_cycles < 1 || !(t_eig >= 0.0)) return fail(FE_ERR_INVALID, "fe_chfsi: need max_cycles >= 1 and t_eig >= 0");
    int cycles = 0, rc = FE_OK;
    for (;;) {
        if ((rc = cheb_filter(m, X, B, deg, a, b, a0, work, cuda_stream))) return rc;       // l.208-210
        if ((rc = fe_rayleigh_ritz(m, X, B, theta_host, work, cuda_stream))) return rc;     // Eq. 23-24
        if ((rc = fe_ritz_residuals(m, X, theta_host, B, res_host, work, cuda_stream))) return rc;
        ++cycles;
        double worst = 0.0;
        for (int j = 0; j < n_gate; ++j) worst = std::max(worst, res_host[j]);
        if (worst <= t_eig || cycles >= max_cycles) break;
        // next window (survey 8(c) step 8): the unwanted part starts at the largest Ritz value of the block, the
        // normalisation point moves to the smallest; b stays the upper bound of the spectrum
        a = theta_host[B - 1];
        a0 = theta_host[0];
        if (!(a0 < a && a < b)) return fail(FE_ERR_STATE, "fe_chfsi: Ritz values left the window (theta_min=%g theta_max=%g b=%g)", a0, a, b);
    }
    if (cycles_host) *cycles_host = cycles;
    return FE_OK;
}

// ---- step-0 ceilings (fe_diag.cuh): not on the product path; bench.py prints them beside the roofline ---------------------
int fe_diag_peak(int cuda_device, int kind, double min_seconds, double* value_host)
{
    if (!value_host) return fail(FE_ERR_INVALID, "fe_diag_peak: NULL result");
    if (kind < 0 || kind > 4) return fail(FE_ERR_INVALID, "fe_diag_peak: kind %d outside 0..4", kind);
    if (!(min_seconds > 0.0) || min_seconds > 30.0) return fail(FE_ERR_INVALID, "fe_diag_peak: min_seconds outside (0, 30]");
    CUDA_TRY(cudaSetDevice(cuda_device));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, cuda_device));
    const int sms = prop.multiProcessorCount;
    const long long n = 1ll << 27;  // doubles per array of the memory kinds: 1 GiB, far beyond the 126 MB L2
    double *a = nullptr, *b = nullptr, *c = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = FE_OK;
    double work = 0.0;  // flops or bytes per launch
    auto launch = [&]() {
        switch (kind) {
            case 0: k_diag_dfma<8><<<sms * 4, 256>>>(a, 4096, -1e-9, 0.0); break;
            case 1: k_diag_dmma<<<sms * 4, 256>>>(a, 4096, 0.25, 1e-3); break;
            case 2: k_diag_stream<<<sms * 16, 256>>>((const double2*)a, (const double2*)b, (double2*)c, n / 2, 0.5); break;
            case 3: k_diag_bulk_red<16384><<<sms * 4, 128, 16384>>>(a, n * 8 / 16384); break;
            default: k_diag_red<<<sms * 16, 256>>>(a, n, 1.0); break;
        }
    };
    do {
        const size_t small = (size_t)sms * 4 * 256 * sizeof(double);
        cudaError_t ce = cudaMalloc((void**)&a, kind <= 1 ? small : (size_t)n * sizeof(double));
        if (ce == cudaSuccess && kind == 2) ce = cudaMalloc((void**)&b, (size_t)n * sizeof(double));
        if (ce == cudaSuccess && kind == 2) ce = cudaMalloc((void**)&c, (size_t)n * sizeof(double));
        if (ce == cudaSuccess && kind >= 2) ce = cudaMemset(a, 0, (size_t)n * sizeof(double));
        if (ce == cudaSuccess && kind == 2) ce = cudaMemset(b, 0, (size_t)n * sizeof(double));
        if (ce == cudaSuccess) ce = cudaEventCreate(&e0);
        if (ce == cudaSuccess) ce = cudaEventCreate(&e1);
        if (ce != cudaSuccess) { rc = fail(FE_ERR_NOMEM, "fe_diag_peak: setup failed: %s", cudaGetErrorString(ce)); break; }
        const double threads = (double)sms * 4 * 256;
        if (kind == 0) work = threads * 4096.0 * 16 * 8 * 2;            // iters x unroll x chains x (mul + add)
        else if (kind == 1) work = threads / 32 * 4096.0 * 8 * 4 * 512;  // warps x iters x unroll x chains x 8*8*4*2
        else if (kind == 2) work = 3.0 * n * 8;
        else work = 1.0 * n * 8;                                          // payload bytes added into global memory
        if (kind == 3) cudaFuncSetAttribute(k_diag_bulk_red<16384>, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384);
        launch();  // warm-up
        ce = cudaDeviceSynchronize();
        if (ce != cudaSuccess) { rc = fail(FE_ERR_CUDA, "fe_diag_peak: kernel failed: %s", cudaGetErrorString(ce)); break; }
        double best = 0.0, total = 0.0;
        while (total < min_seconds) {
            cudaEventRecord(e0);
            launch();
            cudaEventRecord(e1);
            ce = cudaEventSynchronize(e1);
            float ms = 0.f;
            if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
            if (ce != cudaSuccess || !(ms > 0.f)) { rc = fail(FE_ERR_CUDA, "fe_diag_peak: timing failed: %s", cudaGetErrorString(ce)); break; }
            total += ms * 1e-3;
            best = std::max(best, work / (ms * 1e-3));
        }
        *value_host = best * (kind <= 1 ? 1e-12 : 1e-9);  // TFLOP/s or GB/s, best launch
    } while (false);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(a); cudaFree(b); cudaFree(c);
    return rc;
}
