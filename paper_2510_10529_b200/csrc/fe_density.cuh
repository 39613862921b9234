// fe_density.cuh -- electron density at the quadrature points (NEXT-4; Eq. 4 l.73-77)
//
//   rho[e][q] = sum_j f_j psi_j(x_q)^2 ,   psi_j = M^{-1/2} psi~_j  (Eq. 19: the API vectors are psi~ = M^{1/2} psi)
//
// evaluated where V is given (cells x n_q^3, q = qx + n(qy + n qz)): the interpolation half of the operator kernel
// (gather, x/y interpolation per nodal plane, z interpolation per line) followed by a square, the occupancy weight
// and a sum over the vectors, which are the lanes of a warp (shuffle reduction).  Unit = (cell, 32 vectors); the
// tiles of a cell accumulate with atomicAdd into a zero-filled rho.
#pragma once
#include <cuda_runtime.h>

#include "fe_kernels.cuh"

namespace fecheb {

struct DensityParams {
    const double* X;   // N x B, psi~
    const double* f;   // B occupancies
    const double* sm;  // N: mu M^{-1/2}
    double* rho;       // cells x n^3
    int B, cx, cy, cz;
    long long Nx, NxNy;
    EOTab eoN;         // even-odd halves of N' = diag(sqrt w) N
    double iw[9];      // 1 / sqrt(w_q): undoes the weight folded into N'
};

template <int P>
__global__ void __launch_bounds__((P + 1) * 32) k_density(const __grid_constant__ DensityParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n2 * n, BT = 32;
    extern __shared__ double sA[];  // [n^3][BT]
    const int lane = threadIdx.x, pl = threadIdx.y;
    const int cell = blockIdx.x;
    const int ex = cell % prm.cx, ey = (cell / prm.cx) % prm.cy, ez = cell / (prm.cx * prm.cy);
    const int j = blockIdx.y * BT + lane;
    const bool act = j < prm.B;
    const long long g0 = (long long)ex * P + prm.Nx * ((long long)ey * P) + prm.NxNy * ((long long)ez * P + pl);
    double v[n][n], t[n], o[n];
    // plane phase: gather with the mu M^{-1/2} scale, interpolate in x and y
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) {
            const long long g = g0 + ax + prm.Nx * ay;
            const double sg = prm.sm[g];
            v[ay][ax] = (act && sg != 0.0) ? prm.X[g * prm.B + j] * sg : 0.0;  // Dirichlet rows may hold anything (R5)
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
        for (int q = 0; q < n; ++q) sA[((pl * n + q) * n + qx) * BT + lane] = o[q];
    }
    __syncthreads();
    // line phase: the thread owns the yz-plane qx = pl; interpolate in z, square, weight, reduce over the lanes
    const double fj = act ? prm.f[j] : 0.0;
    double* rho = prm.rho + (long long)cell * n3;
#pragma unroll 1
    for (int qy = 0; qy < n; ++qy) {
#pragma unroll
        for (int az = 0; az < n; ++az) t[az] = sA[((az * n + qy) * n + pl) * BT + lane];
        mat1d_eo<n>(prm.eoN, t, o);
        const double wxy = prm.iw[pl] * prm.iw[qy];
#pragma unroll
        for (int qz = 0; qz < n; ++qz) {
            const double psi = o[qz] * (wxy * prm.iw[qz]);
            double r = fj * psi * psi;
#pragma unroll
            for (int sft = 16; sft > 0; sft >>= 1) r += __shfl_xor_sync(0xffffffffu, r, sft);
            if (lane == 0) atomicAdd(rho + (qz * n + qy) * n + pl, r);
        }
    }
}

template <int P>
cudaError_t launch_density_p(const DensityParams& prm, long long ncells, cudaStream_t st)
{
    constexpr int n = P + 1;
    const size_t smem = (size_t)n * n * n * 32 * sizeof(double);
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_density<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    dim3 grid((unsigned)ncells, (unsigned)((prm.B + 31) / 32)), block(32, n);
    k_density<P><<<grid, block, smem, st>>>(prm);
    return cudaGetLastError();
}

inline cudaError_t launch_density(const DensityParams& prm, int p, long long ncells, cudaStream_t st)
{
    switch (p) {
        case 1: return launch_density_p<1>(prm, ncells, st);
        case 2: return launch_density_p<2>(prm, ncells, st);
        case 3: return launch_density_p<3>(prm, ncells, st);
        case 4: return launch_density_p<4>(prm, ncells, st);
        case 5: return launch_density_p<5>(prm, ncells, st);
        case 6: return launch_density_p<6>(prm, ncells, st);
        case 7: return launch_density_p<7>(prm, ncells, st);
        case 8: return launch_density_p<8>(prm, ncells, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace fecheb
