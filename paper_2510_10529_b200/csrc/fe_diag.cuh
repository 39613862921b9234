// fe_diag.cuh -- step-0 ceilings of the device, measured by fe_diag_peak (include/fe_cheb.h) so that the roofline
// denominators and the "matrix-free on DFMA vs per-cell GEMM on DMMA" decision rest on
// numbers bench.py prints in the same run:
//   0  register-resident DFMA chains                      TFLOP/s   (the FP64 ALU pipe the operator kernel is bound by)
//   1  mma.sync.m8n8k4.f64 (DMMA) chains                  TFLOP/s   (the only FP64 tensor path: tcgen05 has no .kind::f64)
//   2  y = a x + z, two reads and one write per element    GB/s      (the byte pattern of a filter step: 24 B per node-vector)
//   3  cp.reduce.async.bulk .add.f64, shared -> global      GB/s      (the scatter of the TMA kernel, bytes of payload)
//   4  red.global.add.f64, one per thread, coalesced        GB/s      (the scatter of the legacy kernel)
// Nothing here is on the product path.
#pragma once
#include <cuda_runtime.h>

namespace fecheb {

template <int CHAINS>
__global__ void __launch_bounds__(256) k_diag_dfma(double* out, int iters, double a, double b)
{
    (void)b;
    double x[CHAINS];
#pragma unroll
    for (int k = 0; k < CHAINS; ++k) x[k] = 1e-3 * (threadIdx.x + 1) + k;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u)
#pragma unroll
            for (int k = 0; k < CHAINS; ++k) x[k] = fma(x[k], a, x[k]);  // two distinct register operands: with three
                                                                         // (x, a, b) the register file caps DFMA at 34.1 TFLOP/s
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < CHAINS; ++k) s += x[k];
    out[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_diag_dmma(double* out, int iters, double a, double b)
{
    constexpr int CH = 4;
    double c0[CH], c1[CH];
#pragma unroll
    for (int k = 0; k < CH; ++k) { c0[k] = 1e-3 * threadIdx.x + k; c1[k] = 0.5 * k; }
    const double fa = a * (1 + (threadIdx.x & 3)), fb = b;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int k = 0; k < CH; ++k)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c0[k]), "+d"(c1[k]) : "d"(fa), "d"(fb));
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += c0[k] + c1[k];
    out[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_diag_stream(const double2* __restrict__ x, const double2* __restrict__ z,
                                                     double2* __restrict__ y, long long n2, double a)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n2; i += (long long)gridDim.x * blockDim.x) {
        const double2 xv = x[i], zv = z[i];
        y[i] = make_double2(fma(a, xv.x, zv.x), fma(a, xv.y, zv.y));
    }
}

// every CTA adds its shared-memory tile (TILE bytes) into successive TILE-sized pieces of Y with the bulk engine
template <int TILE>
__global__ void __launch_bounds__(128) k_diag_bulk_red(double* Y, long long tiles_total)
{
    extern __shared__ __align__(128) double tile[];
    for (int i = threadIdx.x; i < TILE / 8; i += blockDim.x) tile[i] = 1.0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned src = (unsigned)__cvta_generic_to_shared(tile);
        for (long long t = blockIdx.x; t < tiles_total; t += gridDim.x) {
            double* dst = Y + t * (TILE / 8);
            asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;"
                         ::"l"(dst), "r"(src), "r"(TILE) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 8;" ::: "memory");  // a bounded queue, like the operator kernel's
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
}

__global__ void __launch_bounds__(256) k_diag_red(double* Y, long long n, double v)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        atomicAdd(Y + i, v);
}

}  // namespace fecheb
