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
// (four fields of n^3 x BT doubles: U/t/T/R, gz/fz, fx, fy).  Gather and scatter go through the explicit l2g; hanging
// nodes read the expanded values X_h = C_h (s . X) (k_gen_expand) and scatter into Y_h, which k_gen_collapse distributes
// to the unconstrained nodes with C_h^T.  The shift and recurrence terms are written by k_gen_init, which replaces the
// zero-fill of Y.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "fe_kernels.cuh"

namespace fecheb {

struct GenParams {
    const double* X;     // N * B
    const double* Xh;    // (N_all - N) * B: expanded hanging values
    double* Y;           // N * B
    double* Yh;          // (N_all - N) * B
    const double* s;     // N: mu_g M_c,gg^{-1/2}
    const int32_t* l2g;  // ncells * n^3
    const double* metric;  // ncells * 6 * n^3 (fe_general.h)
    const double* WV;      // ncells * n^3: w_q |J| V_q
    long long N;
    int B;
    double alpha;
    double Nt[81];  // N[q*n + a] = l_a(gl_x[q])
    double Dt[81];  // D[s*n + q] = l^_q'(gl_x[s])
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

// WV[e][q] = w_q |J| V[e][q] from the weight field of the metric (component 6)
__global__ void k_gen_weight_potential(double* __restrict__ WV, const double* __restrict__ V,
                                       const double* __restrict__ wdet, long long total)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
        WV[i] = wdet[i] * V[i];
}

template <int n>
__device__ __forceinline__ void mat1d(const double* __restrict__ M, const double (&in)[n], double (&out)[n])
{
#pragma unroll
    for (int i = 0; i < n; ++i) {
        double s = M[i * n] * in[0];
#pragma unroll
        for (int k = 1; k < n; ++k) s = fma(M[i * n + k], in[k], s);
        out[i] = s;
    }
}
template <int n>
__device__ __forceinline__ void mat1d_t(const double* __restrict__ M, const double (&in)[n], double (&out)[n])  // M^T in
{
#pragma unroll
    for (int i = 0; i < n; ++i) {
        double s = M[i] * in[0];
#pragma unroll
        for (int k = 1; k < n; ++k) s = fma(M[k * n + i], in[k], s);
        out[i] = s;
    }
}

template <int P, int BT>
constexpr size_t gen_smem_bytes() { return (size_t)4 * (P + 1) * (P + 1) * (P + 1) * BT * sizeof(double); }

template <int P, int BT, int MINB>
__global__ void __launch_bounds__((P + 1) * BT, MINB) k_apply_gen(const __grid_constant__ GenParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n;
    extern __shared__ double smem[];
    double* F0 = smem;                 // A -> U -> t / T -> R
    double* F1 = F0 + (size_t)n3 * BT;  // gz -> fz
    double* F2 = F1 + (size_t)n3 * BT;  // fx
    double* F3 = F2 + (size_t)n3 * BT;  // fy
    const int lane = threadIdx.x, pl = threadIdx.y;
    const long long cell = blockIdx.x;
    const int j = blockIdx.y * BT + lane;
    const bool act = j < prm.B;
    const long long B = prm.B;
    const int32_t* l2g = prm.l2g + cell * n3;
    const double* Nt = prm.Nt;
    const double* Dt = prm.Dt;
    double t[n], o[n];

    // ---- phase A: gather the nodal plane az = pl, interpolate in x and y ------------------------------------------------
    {
        double v[n][n];
#pragma unroll
        for (int ay = 0; ay < n; ++ay)
#pragma unroll
            for (int ax = 0; ax < n; ++ax) {
                const long long g = l2g[(pl * n + ay) * n + ax];
                double x = 0.0;
                if (act) {
                    if (g < prm.N) {
                        const double sg = prm.s[g];
                        x = sg != 0.0 ? sg * prm.X[g * B + j] : 0.0;  // Dirichlet rows of caller data are ignored (R5)
                    } else
                        x = prm.Xh[(g - prm.N) * B + j];
                }
                v[ay][ax] = x;
            }
#pragma unroll
        for (int ay = 0; ay < n; ++ay) {
            mat1d<n>(Nt, v[ay], o);
#pragma unroll
            for (int q = 0; q < n; ++q) v[ay][q] = o[q];
        }
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int a = 0; a < n; ++a) t[a] = v[a][qx];
            mat1d<n>(Nt, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) F0[((pl * n + qy) * n + qx) * BT + lane] = o[qy];
        }
    }
    __syncthreads();
    // ---- phase B: the yz-plane qx = pl: U = Nz A, gz = Dz U (lines along z) ------------------------------------------------
#pragma unroll
    for (int qy = 0; qy < n; ++qy) {
#pragma unroll
        for (int az = 0; az < n; ++az) t[az] = F0[((az * n + qy) * n + pl) * BT + lane];
        mat1d<n>(Nt, t, o);
        mat1d<n>(Dt, o, t);
#pragma unroll
        for (int qz = 0; qz < n; ++qz) {
            F0[((qz * n + qy) * n + pl) * BT + lane] = o[qz];
            F1[((qz * n + qy) * n + pl) * BT + lane] = t[qz];
        }
    }
    __syncthreads();
    // ---- phase C: the xy-plane qz = pl: gx, gy, the pointwise metric, Dx^T and Dy^T ----------------------------------------
    {
        double u[n][n];
        const size_t base = (size_t)pl * n2;
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) u[qy][qx] = F0[(base + qy * n + qx) * BT + lane];
        const double* Mq = prm.metric + cell * 6 * n3 + pl * n2;  // + c * n3 + qy * n + qx
        const double* WVq = prm.WV + cell * n3 + pl * n2;
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            double gx[n], gy[n];
            mat1d<n>(Dt, u[qy], gx);
#pragma unroll
            for (int qx = 0; qx < n; ++qx) {
                double s = Dt[qy * n] * u[0][qx];
#pragma unroll
                for (int r = 1; r < n; ++r) s = fma(Dt[qy * n + r], u[r][qx], s);
                gy[qx] = s;
            }
#pragma unroll
            for (int qx = 0; qx < n; ++qx) {
                const int q = qy * n + qx;
                const double gz = F1[(base + q) * BT + lane];
                const double g0 = Mq[q], g1 = Mq[n3 + q], g2 = Mq[2 * n3 + q], g3 = Mq[3 * n3 + q], g4 = Mq[4 * n3 + q],
                             g5 = Mq[5 * n3 + q];
                F2[(base + q) * BT + lane] = fma(g0, gx[qx], fma(g1, gy[qx], g2 * gz));
                F3[(base + q) * BT + lane] = fma(g1, gx[qx], fma(g3, gy[qx], g4 * gz));
                F1[(base + q) * BT + lane] = fma(g2, gx[qx], fma(g4, gy[qx], g5 * gz));
            }
        }
        // t = WV U + Dx^T fx (rows) + Dy^T fy (columns), into F0; the thread re-reads only what it wrote itself
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int qx = 0; qx < n; ++qx) t[qx] = F2[(base + qy * n + qx) * BT + lane];
            mat1d_t<n>(Dt, t, o);
#pragma unroll
            for (int qx = 0; qx < n; ++qx) u[qy][qx] = fma(WVq[qy * n + qx], u[qy][qx], o[qx]);
        }
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int qy = 0; qy < n; ++qy) t[qy] = F3[(base + qy * n + qx) * BT + lane];
            mat1d_t<n>(Dt, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) F0[(base + qy * n + qx) * BT + lane] = u[qy][qx] + o[qy];
        }
    }
    __syncthreads();
    // ---- phase D: the yz-plane qx = pl again: T += Dz^T fz, R = Nz^T T --------------------------------------------------------
#pragma unroll
    for (int qy = 0; qy < n; ++qy) {
        double tz[n];
#pragma unroll
        for (int qz = 0; qz < n; ++qz) {
            t[qz] = F1[((qz * n + qy) * n + pl) * BT + lane];
            tz[qz] = F0[((qz * n + qy) * n + pl) * BT + lane];
        }
        mat1d_t<n>(Dt, t, o);
#pragma unroll
        for (int qz = 0; qz < n; ++qz) tz[qz] += o[qz];
        mat1d_t<n>(Nt, tz, o);
#pragma unroll
        for (int az = 0; az < n; ++az) F0[((az * n + qy) * n + pl) * BT + lane] = o[az];
    }
    __syncthreads();
    // ---- phase E: back-interpolate the nodal plane az = pl in y and x, scatter through the l2g -------------------------------
    {
        double v[n][n];
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) v[qy][qx] = F0[((pl * n + qy) * n + qx) * BT + lane];
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int q = 0; q < n; ++q) t[q] = v[q][qx];
            mat1d_t<n>(Nt, t, o);
#pragma unroll
            for (int a = 0; a < n; ++a) v[a][qx] = o[a];
        }
#pragma unroll
        for (int ay = 0; ay < n; ++ay) {
            mat1d_t<n>(Nt, v[ay], o);
            if (act) {
#pragma unroll
                for (int ax = 0; ax < n; ++ax) {
                    const long long g = l2g[(pl * n + ay) * n + ax];
                    if (g < prm.N) {
                        const double sg = prm.s[g];
                        if (sg != 0.0) atomicAdd(prm.Y + g * B + j, prm.alpha * sg * o[ax]);
                    } else
                        atomicAdd(prm.Yh + (g - prm.N) * B + j, o[ax]);
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

// vector-tile width per order: four fields of n^3 x BT doubles must fit the 227 KB of shared memory
inline cudaError_t launch_apply_gen(const GenParams& prm, int p, long long ncells, cudaStream_t st)
{
    switch (p) {
        case 1: return launch_gen<1, 32, 8>(prm, ncells, st);
        case 2: return launch_gen<2, 32, 4>(prm, ncells, st);
        case 3: return launch_gen<3, 32, 3>(prm, ncells, st);
        case 4: return launch_gen<4, 16, 3>(prm, ncells, st);
        case 5: return launch_gen<5, 16, 2>(prm, ncells, st);
        case 6: return launch_gen<6, 16, 1>(prm, ncells, st);
        case 7: return launch_gen<7, 8, 1>(prm, ncells, st);
        case 8: return launch_gen<8, 8, 1>(prm, ncells, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace fecheb
