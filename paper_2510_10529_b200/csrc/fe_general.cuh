// fe_general.cuh -- the fused operator step on GENERAL hexahedral cells with hanging nodes (PAPER.md
// l.151, l.273, Fig. 6; Eq. 17 l.171 on a trilinearly mapped cell)
//
//   Y[g,j] = mu_g ( alpha ( s_g [C^T sum_e P_e^T y_e]_g - (c + eps_j) X[g,j] ) + beta Z[g,j] ),   x_all = C (s . X)
//
// with C = [I; C_hanging] the constraint matrix of the hanging nodes and y_e the cell contraction in its generic form: the
// metric of a mapped cell is a full symmetric 3 x 3 matrix per quadrature point, so the kinetic term no longer separates
// and the contraction takes 12 one-dimensional sweeps instead of the 10 of the box-cell kernel (fe_apply_tma.cuh):
//
//   U  = (Nz Ny Nx) x_e                                         interpolate to the Gauss points            3 sweeps
//   (gx, gy, gz) = (Dx U, Dy U, Dz U)                           reference gradient, collocation derivative  3 sweeps
//   (fx, fy, fz) = G_q (gx, gy, gz),  t = WV_q U                pointwise: G_q = 1/2 w_q |J| J^-1 J^-T, WV_q = w_q |J| V_q
//   T  = t + Dx^T fx + Dy^T fy + Dz^T fz                                                                    3 sweeps
//   y_e = (Nx^T Ny^T Nz^T) T                                                                                3 sweeps
//
// Threads: lane = vector j (BT per cell tile), threadIdx.y = a plane index.  A thread owns a nodal z-plane (phases A, E),
// the yz-plane qx = pl (phases B, D: everything along z) or the xy-plane qz = pl (phase C: everything along x and y), so
// every 1-D matrix entry is a warp-uniform constant-bank operand; the cell tile crosses shared memory between phases
// (three fields of n^3 x BT doubles: x/A/U/t/R, gy/fy, gz/fz).  Gather and scatter go through the explicit l2g; hanging
// nodes read the expanded values X_h = C_h (s . X) (k_gen_expand) and scatter into Y_h, which k_gen_collapse distributes
// to the unconstrained nodes with C_h^T.  The shift and recurrence terms are written by k_gen_init, which replaces the
// zero-fill of Y.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "fe_apply_tma.cuh"
#include "fe_kernels.cuh"

namespace fecheb {

struct GenParams {
    const double* X;     // N * B
    const double* Xh;    // (N_all - N) * B: expanded hanging values
    double* Y;           // N * B
    double* Yh;          // (N_all - N) * B
    const int32_t* l2g;  // ncells * n^3
    const double* sc;    // ncells * n^3: s_g = mu_g M_c,gg^{-1/2} at the cell's unconstrained nodes, 1 at its hanging nodes
    const double* rec;   // ncells * GREC: per-cell record, 6 metric fields (fe_general.h) then WV = w_q |J| V_q, n^3 each
    long long N;
    int B;
    double alpha;
    // even-odd halves (fe_kernels.cuh): N and N^T are centro-symmetric, the collocation derivative D and D^T are
    // centro-ANTIsymmetric (D[n-1-s][n-1-q] = -D[s][q]); for those the row i = h of S holds the middle row D[h][k], k < h
    EOTab eoN, eoNT, eoD, eoDT;
};

// Y = mu (kappa_j X + beta Z), kappa_j = -alpha (c + eps_j): the part of the step that is diagonal in the nodes
__global__ void k_gen_init(double* __restrict__ Y, const double* __restrict__ X, const double* __restrict__ Z,
                           const double* __restrict__ s, const double* __restrict__ eps, double alpha, double beta,
                           double c, long long N, int B)
{
    const long long total = N * B;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long g = i / B;
        const int j = (int)(i - g * B);
        double v = 0.0;
        if (s[g] != 0.0) {
            const double kappa = -alpha * (c + (eps ? eps[j] : 0.0));
            if (kappa != 0.0) v = kappa * X[i];
            if (Z) v = fma(beta, Z[i], v);
        }
        Y[i] = v;
    }
}

// X_h[r, j] = sum_k cval (s . X)[ccol, j]: values of the hanging nodes (rows r of the constraint matrix)
__global__ void k_gen_expand(double* __restrict__ Xh, const double* __restrict__ X, const double* __restrict__ s,
                             const long long* __restrict__ crow, const int32_t* __restrict__ ccol,
                             const double* __restrict__ cval, long long nh, int B)
{
    const long long total = nh * B;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long r = i / B;
        const int j = (int)(i - r * B);
        double v = 0.0;
        for (long long k = crow[r]; k < crow[r + 1]; ++k) {
            const int32_t g = ccol[k];
            const double sg = s[g];
            if (sg != 0.0) v = fma(cval[k] * sg, X[(long long)g * B + j], v);  // Dirichlet rows of caller data are ignored
        }
        Xh[i] = v;
    }
}

// Y[ccol, j] += alpha s_ccol cval Y_h[r, j]: the transpose of the expansion
__global__ void k_gen_collapse(double* __restrict__ Y, const double* __restrict__ Yh, const double* __restrict__ s,
                               const long long* __restrict__ crow, const int32_t* __restrict__ ccol,
                               const double* __restrict__ cval, long long nh, int B, double alpha)
{
    const long long total = nh * B;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long r = i / B;
        const int j = (int)(i - r * B);
        const double y = alpha * Yh[i];
        for (long long k = crow[r]; k < crow[r + 1]; ++k) {
            const int32_t g = ccol[k];
            const double sg = s[g];
            if (sg != 0.0) atomicAdd(Y + (long long)g * B + j, cval[k] * sg * y);
        }
    }
}

// per-cell record of the general kernel: 7 fields of n^3 doubles (6 metric entries, WV), padded to a multiple of 16 bytes
inline int gen_rec_doubles(int n) { const int r = 7 * n * n * n; return r + (r & 1); }

// field 6 of every record: WV[e][q] = w_q |J| V[e][q]
__global__ void k_gen_weight_potential(double* __restrict__ rec, const double* __restrict__ V,
                                       const double* __restrict__ wdet, long long ncells, int n3, int grec)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ncells * n3; i += (long long)gridDim.x * blockDim.x) {
        const long long e = i / n3;
        rec[e * grec + 6 * n3 + (i - e * n3)] = wdet[i] * V[i];
    }
}

// even-odd product with a centro-ANTIsymmetric matrix: out[i] = E + O, out[n-1-i] = O - E (mat1d_eo has E - O there)
template <int n>
__device__ __forceinline__ void mat1d_eoa(const EOTab& T, const double (&in)[n], double (&out)[n])
{
    constexpr int h = n / 2;
    double e[h > 0 ? h : 1], o[h > 0 ? h : 1];
#pragma unroll
    for (int k = 0; k < h; ++k) {
        e[k] = in[k] + in[n - 1 - k];
        o[k] = in[k] - in[n - 1 - k];
    }
#pragma unroll
    for (int i = 0; i < h; ++i) {
        double se;
        if (n % 2 == 1) {
            se = T.Mid[i] * in[h];
#pragma unroll
            for (int k = 0; k < h; ++k) se = fma(T.S[i * h + k], e[k], se);
        } else {
            se = T.S[i * h] * e[0];
#pragma unroll
            for (int k = 1; k < h; ++k) se = fma(T.S[i * h + k], e[k], se);
        }
        double so = T.A[i * h] * o[0];
#pragma unroll
        for (int k = 1; k < h; ++k) so = fma(T.A[i * h + k], o[k], so);
        out[i] = se + so;
        out[n - 1 - i] = so - se;
    }
    if (n % 2 == 1) {
        double sm = 0.0;
        if (h > 0) {
            sm = T.S[h * h] * o[0];
#pragma unroll
            for (int k = 1; k < h; ++k) sm = fma(T.S[h * h + k], o[k], sm);
        }
        out[h] = sm;
    }
}

template <int P, int BT>
constexpr size_t gen_smem_bytes()
{
    constexpr int n3 = (P + 1) * (P + 1) * (P + 1);
    return (size_t)3 * n3 * BT * sizeof(double) + (size_t)(7 * n3 + 1) * sizeof(double) +
           (size_t)n3 * (sizeof(double) + sizeof(int32_t)) + 32;
}

template <int P, int BT, int MINB>
__global__ void __launch_bounds__((P + 1) * BT, MINB) k_apply_gen(const __grid_constant__ GenParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n;
    extern __shared__ __align__(128) double smem[];
    double* F0 = smem;                  // x -> A -> U -> t -> R
    double* F1 = F0 + (size_t)n3 * BT;  // gy -> fy
    double* F2 = F1 + (size_t)n3 * BT;  // gz -> fz
    double* sRec = F2 + (size_t)n3 * BT;  // the cell's record (6 metric fields, WV), one bulk copy in flight during A and B
    constexpr int GREC = 7 * n3 + ((7 * n3) & 1);
    double* sSc = sRec + GREC;            // [n^3] gather / scatter scale of the cell's nodes
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(sSc + n3 + (n3 & 1));
    int32_t* sId = reinterpret_cast<int32_t*>(bar + 1);  // [n^3] global ids
    const int lane = threadIdx.x, pl = threadIdx.y, tid = pl * BT + lane;
    const long long cell = blockIdx.x;
    const int j = blockIdx.y * BT + lane;
    const bool act = j < prm.B;
    const long long B = prm.B;
    double t[n], o[n];

    // ---- gather: ids and scales of the cell, then every thread fetches ITS nodal plane with independent 8-byte cp.async ------
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, (unsigned)(GREC * sizeof(double)));
        bulk_load(sRec, prm.rec + cell * GREC, (unsigned)(GREC * sizeof(double)), bar);
    }
    for (int a = tid; a < n3; a += n * BT) {
        sId[a] = prm.l2g[cell * n3 + a];
        sSc[a] = prm.sc[cell * n3 + a];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < n2; ++k) {
        const int a = pl * n2 + k;
        const long long g = sId[a];
        const double* src = g < prm.N ? prm.X + g * B + j : prm.Xh + (g - prm.N) * B + j;
        cp_async8(F0 + (size_t)a * BT + lane, act ? src : prm.X, act);
    }
    cp_async_commit();
    cp_async_wait_all();
    // ---- phase A: the nodal plane az = pl: scale, interpolate in x and y (table N) ---------------------------------------------
    {
        double v[n][n];
#pragma unroll
        for (int ay = 0; ay < n; ++ay)
#pragma unroll
            for (int ax = 0; ax < n; ++ax) {
                const int a = pl * n2 + ay * n + ax;
                const double sg = sSc[a];
                const double x = F0[(size_t)a * BT + lane];
                v[ay][ax] = sg != 0.0 ? sg * x : 0.0;  // Dirichlet rows of caller data are ignored (R5)
            }
#pragma unroll
        for (int ay = 0; ay < n; ++ay) {
            mat1d_eo<n>(prm.eoN, v[ay], o);
#pragma unroll
            for (int q = 0; q < n; ++q) v[ay][q] = o[q];
        }
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int a = 0; a < n; ++a) t[a] = v[a][qx];
            mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) F0[((size_t)(pl * n + qy) * n + qx) * BT + lane] = o[qy];
        }
    }
    __syncthreads();
    // ---- phase B: the yz-plane qx = pl: U = Nz A (table N), then gz = Dz U along z and gy = Dy U along y (table D) ---------------
    {
        double u[n][n];  // [qy][qz]
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int az = 0; az < n; ++az) t[az] = F0[((size_t)(az * n + qy) * n + pl) * BT + lane];
            mat1d_eo<n>(prm.eoN, t, u[qy]);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) F0[((size_t)(qz * n + qy) * n + pl) * BT + lane] = u[qy][qz];
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eoa<n>(prm.eoD, u[qy], o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) F2[((size_t)(qz * n + qy) * n + pl) * BT + lane] = o[qz];
        }
#pragma unroll
        for (int qz = 0; qz < n; ++qz) {
#pragma unroll
            for (int qy = 0; qy < n; ++qy) t[qy] = u[qy][qz];
            mat1d_eoa<n>(prm.eoD, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) F1[((size_t)(qz * n + qy) * n + pl) * BT + lane] = o[qy];
        }
    }
    __syncthreads();
    // ---- phase C: the xy-plane qz = pl, row by row: gx = Dx U (table D), the metric at the points, t = WV U + Dx^T fx (D^T) ------
    {
        const size_t base = (size_t)pl * n2;
        double gx[n][n];
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int qx = 0; qx < n; ++qx) t[qx] = F0[(base + qy * n + qx) * BT + lane];
            mat1d_eoa<n>(prm.eoD, t, gx[qy]);
        }
        mbar_wait(bar, 0);
        const double* Mq = sRec + pl * n2;  // + c * n3 + qy * n + qx
        const double* WVq = sRec + 6 * n3 + pl * n2;
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) {
                const int q = qy * n + qx;
                const size_t idx = (base + q) * BT + lane;
                const double gyv = F1[idx], gzv = F2[idx], gxv = gx[qy][qx];
                const double g0 = Mq[q], g1 = Mq[n3 + q], g2 = Mq[2 * n3 + q], g3 = Mq[3 * n3 + q], g4 = Mq[4 * n3 + q],
                             g5 = Mq[5 * n3 + q];
                gx[qy][qx] = fma(g0, gxv, fma(g1, gyv, g2 * gzv));
                F1[idx] = fma(g1, gxv, fma(g3, gyv, g4 * gzv));
                F2[idx] = fma(g2, gxv, fma(g4, gyv, g5 * gzv));
                F0[idx] *= WVq[q];
            }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eoa<n>(prm.eoDT, gx[qy], o);
#pragma unroll
            for (int qx = 0; qx < n; ++qx) F0[(base + qy * n + qx) * BT + lane] += o[qx];
        }
    }
    __syncthreads();
    // ---- phase D: the yz-plane qx = pl: T = t + Dz^T fz + Dy^T fy (table D^T), R = Nz^T T (table N^T) -----------------------------
    {
        double T[n][n];  // [qy][qz]
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int qz = 0; qz < n; ++qz) t[qz] = F2[((size_t)(qz * n + qy) * n + pl) * BT + lane];
            mat1d_eoa<n>(prm.eoDT, t, o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) T[qy][qz] = F0[((size_t)(qz * n + qy) * n + pl) * BT + lane] + o[qz];
        }
#pragma unroll
        for (int qz = 0; qz < n; ++qz) {
#pragma unroll
            for (int qy = 0; qy < n; ++qy) t[qy] = F1[((size_t)(qz * n + qy) * n + pl) * BT + lane];
            mat1d_eoa<n>(prm.eoDT, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) T[qy][qz] += o[qy];
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoNT, T[qy], o);
#pragma unroll
            for (int az = 0; az < n; ++az) F0[((size_t)(az * n + qy) * n + pl) * BT + lane] = o[az];
        }
    }
    __syncthreads();
    // ---- phase E: back-interpolate the nodal plane az = pl in y and x (table N^T), scatter through the l2g ---------------------------
    {
        double v[n][n];
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) v[qy][qx] = F0[((size_t)(pl * n + qy) * n + qx) * BT + lane];
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int q = 0; q < n; ++q) t[q] = v[q][qx];
            mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
            for (int a = 0; a < n; ++a) v[a][qx] = o[a];
        }
#pragma unroll
        for (int ay = 0; ay < n; ++ay) {
            mat1d_eo<n>(prm.eoNT, v[ay], o);
            if (act) {
#pragma unroll
                for (int ax = 0; ax < n; ++ax) {
                    const int a = pl * n2 + ay * n + ax;
                    const long long g = sId[a];
                    const double sg = sSc[a];
                    const bool master = g < prm.N;
                    double* dst = master ? prm.Y + g * B + j : prm.Yh + (g - prm.N) * B + j;
                    if (sg != 0.0) atomicAdd(dst, master ? prm.alpha * sg * o[ax] : o[ax]);
                }
            }
        }
    }
}

template <int P, int BT, int MINB>
cudaError_t launch_gen(const GenParams& prm, long long ncells, cudaStream_t st)
{
    constexpr int n = P + 1;
    constexpr size_t smem = gen_smem_bytes<P, BT>();
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_apply_gen<P, BT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    dim3 grid((unsigned)ncells, (unsigned)((prm.B + BT - 1) / BT)), block(BT, n);
    k_apply_gen<P, BT, MINB><<<grid, block, smem, st>>>(prm);
    return cudaGetLastError();
}

// vector-tile width per order: three fields of n^3 x BT doubles per CTA, several CTAs per SM where they fit
inline cudaError_t launch_apply_gen(const GenParams& prm, int p, long long ncells, cudaStream_t st)
{
    switch (p) {
        case 1: return launch_gen<1, 32, 8>(prm, ncells, st);
        case 2: return launch_gen<2, 32, 6>(prm, ncells, st);
        case 3: return launch_gen<3, 32, 4>(prm, ncells, st);
        case 4: return launch_gen<4, 32, 2>(prm, ncells, st);
        case 5: return launch_gen<5, 16, 2>(prm, ncells, st);
        case 6: return launch_gen<6, 16, 1>(prm, ncells, st);
        case 7: return launch_gen<7, 8, 2>(prm, ncells, st);
        case 8: return launch_gen<8, 8, 1>(prm, ncells, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace fecheb
