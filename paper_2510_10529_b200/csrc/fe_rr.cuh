// fe_rr.cuh -- tall-skinny FP64 kernels of the Rayleigh-Ritz step of ChFSI (Eq. 23-24, l.210-219; R8, R9)
//
//   k_gram     : C = A^T B          (B x B, from two N x B node-major blocks)     S_Y = Y^T Y,  H~_Y = Q^T (H~ Q)
//   k_rightmul : Y <- Y R           (N x B times a small B x B matrix, in place)   Q = Y L^{-T},  X = Q V
//
// Both stream the block once (16 bytes of traffic per 2B flops per element): with B = 64..128 they sit at the FP64
// ridge, so they are register-tiled DFMA kernels with the operands staged in shared memory; the B x B result of
// k_gram is accumulated in registers over a persistent row loop and added to global memory once per CTA.
#pragma once
#include <cuda_runtime.h>

namespace fecheb {

constexpr int kRRThreads = 256;  // 16 x 16 threads, each owning a T x T block of the B x B matrix
constexpr int kRRRows = 32;      // rows of the block staged per iteration

// C[i*B + j] += sum_r A[r*B + i] * Bm[r*B + j];  C must be zero on entry.  T*16 >= B.
template <int T>
__global__ void __launch_bounds__(kRRThreads) k_gram(const double* __restrict__ A, const double* __restrict__ Bm,
                                                     long long N, int B, double* __restrict__ C)
{
    extern __shared__ double sm[];
    double* sA = sm;                      // [kRRRows][B]
    double* sB = sm + kRRRows * B;        // [kRRRows][B]
    const int ti = threadIdx.x / 16, tj = threadIdx.x % 16;
    double acc[T][T];
#pragma unroll
    for (int a = 0; a < T; ++a)
#pragma unroll
        for (int b = 0; b < T; ++b) acc[a][b] = 0.0;
    const long long ntiles = (N + kRRRows - 1) / kRRRows;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const long long r0 = tile * kRRRows;
        const int rows = (int)((N - r0 < kRRRows) ? (N - r0) : kRRRows);
        __syncthreads();
        for (int i = threadIdx.x; i < kRRRows * B; i += kRRThreads) {
            const bool in = i < rows * B;
            sA[i] = in ? A[r0 * B + i] : 0.0;
            sB[i] = in ? Bm[r0 * B + i] : 0.0;
        }
        __syncthreads();
#pragma unroll 4
        for (int r = 0; r < kRRRows; ++r) {
            double a[T], b[T];
#pragma unroll
            for (int k = 0; k < T; ++k) {
                const int i = ti + 16 * k, j = tj + 16 * k;  // strided ownership: conflict-free shared-memory reads
                a[k] = i < B ? sA[r * B + i] : 0.0;
                b[k] = j < B ? sB[r * B + j] : 0.0;
            }
#pragma unroll
            for (int x = 0; x < T; ++x)
#pragma unroll
                for (int y = 0; y < T; ++y) acc[x][y] = fma(a[x], b[y], acc[x][y]);
        }
    }
#pragma unroll
    for (int x = 0; x < T; ++x)
#pragma unroll
        for (int y = 0; y < T; ++y) {
            const int i = ti + 16 * x, j = tj + 16 * y;
            if (i < B && j < B) atomicAdd(C + (size_t)i * B + j, acc[x][y]);
        }
}

// Out[r*B + j] (+)= sum_i Y[r*B + i] * R[i*B + j];  Out may be Y (each CTA stages its rows before overwriting them)
template <int T>
__global__ void __launch_bounds__(kRRThreads) k_rightmul(const double* Y, const double* __restrict__ R, double* Out,
                                                         int accumulate, long long N, int B)
{
    extern __shared__ double sm[];
    double* sR = sm;              // [B][B]
    double* sY = sm + B * B;      // [kRRRows][B + 1]   (+1: rows are read down a column)
    const int ti = threadIdx.x / 16, tj = threadIdx.x % 16;  // ti: rows ti, ti+16; tj: columns tj + 16 k
    for (int i = threadIdx.x; i < B * B; i += kRRThreads) sR[i] = R[i];
    const long long ntiles = (N + kRRRows - 1) / kRRRows;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const long long r0 = tile * kRRRows;
        const int rows = (int)((N - r0 < kRRRows) ? (N - r0) : kRRRows);
        __syncthreads();
        for (int i = threadIdx.x; i < kRRRows * B; i += kRRThreads) {
            const int r = i / B, c = i - r * B;
            sY[r * (B + 1) + c] = r < rows ? Y[r0 * B + i] : 0.0;
        }
        __syncthreads();
        double acc[2][T];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < T; ++b) acc[a][b] = 0.0;
        for (int i = 0; i < B; ++i) {
            const double y0 = sY[ti * (B + 1) + i], y1 = sY[(ti + 16) * (B + 1) + i];
#pragma unroll
            for (int k = 0; k < T; ++k) {
                const int j = tj + 16 * k;
                const double rv = j < B ? sR[i * B + j] : 0.0;
                acc[0][k] = fma(y0, rv, acc[0][k]);
                acc[1][k] = fma(y1, rv, acc[1][k]);
            }
        }
#pragma unroll
        for (int k = 0; k < T; ++k) {
            const int j = tj + 16 * k;
            if (j < B) {
                if (ti < rows) Out[(r0 + ti) * B + j] = acc[0][k] + (accumulate ? Out[(r0 + ti) * B + j] : 0.0);
                if (ti + 16 < rows) Out[(r0 + ti + 16) * B + j] = acc[1][k] + (accumulate ? Out[(r0 + ti + 16) * B + j] : 0.0);
            }
        }
    }
}

inline cudaError_t launch_gram(const double* A, const double* Bm, long long N, int B, double* C, int sms, cudaStream_t st)
{
    const size_t smem = (size_t)2 * kRRRows * B * sizeof(double);
    const int T = (B + 15) / 16;
    if (T > 8) return cudaErrorInvalidValue;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_gram<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * kRRRows * 128 * 8);
        configured = true;
    }
    const int grid = sms * 2;
    if (T <= 1) k_gram<1><<<grid, kRRThreads, smem, st>>>(A, Bm, N, B, C);
    else if (T <= 2) k_gram<2><<<grid, kRRThreads, smem, st>>>(A, Bm, N, B, C);
    else if (T <= 4) k_gram<4><<<grid, kRRThreads, smem, st>>>(A, Bm, N, B, C);
    else k_gram<8><<<grid, kRRThreads, smem, st>>>(A, Bm, N, B, C);
    return cudaGetLastError();
}

inline cudaError_t launch_rightmul(const double* Y, const double* R, double* Out, int accumulate, long long N, int B,
                                   int sms, cudaStream_t st)
{
    const size_t smem = ((size_t)B * B + (size_t)kRRRows * (B + 1)) * sizeof(double);
    const int T = (B + 15) / 16;
    if (T > 8) return cudaErrorInvalidValue;
    static bool configured = false;
    if (!configured) {
        const int mx = (128 * 128 + kRRRows * 129) * 8;
        cudaFuncSetAttribute(k_rightmul<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        cudaFuncSetAttribute(k_rightmul<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        cudaFuncSetAttribute(k_rightmul<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        cudaFuncSetAttribute(k_rightmul<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        configured = true;
    }
    const int grid = sms * (B > 64 ? 1 : 2);
    if (T <= 1) k_rightmul<1><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    else if (T <= 2) k_rightmul<2><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    else if (T <= 4) k_rightmul<4><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    else k_rightmul<8><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    return cudaGetLastError();
}

}  // namespace fecheb
