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

#include <cstdint>

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

// ---- fast paths for even B: 16-byte cp.async staging into a two-stage ring, 128-bit shared-memory reads ------------------
__device__ __forceinline__ void rr_cp16(void* dst, const void* src, bool valid)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst);
    const int sz = valid ? 16 : 0;  // src-size 0 zero-fills the 16 destination bytes
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void rr_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int K>
__device__ __forceinline__ void rr_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(K) : "memory"); }

// thread t of 16 owns the index pairs {2t + 32m, 2t + 32m + 1 : m < T/2}: 16-byte reads, conflict-free across the 16
__device__ __forceinline__ int rr_own(int t, int k) { return 2 * t + 32 * (k >> 1) + (k & 1); }

// stage `rows` rows of a node-major block (pitch B) into smem rows of pitch BP; rows beyond N are zero-filled
__device__ __forceinline__ void rr_stage(double* dst, const double* src, long long r0, int rows_tile, long long N, int B, int BP)
{
    const int chunks = B / 2;
    for (int i = threadIdx.x; i < rows_tile * chunks; i += kRRThreads) {
        const int r = i / chunks, c = i - r * chunks;
        const bool ok = r0 + r < N;
        rr_cp16(dst + r * BP + 2 * c, src + (ok ? (r0 + r) * B + 2 * c : 0), ok);
    }
}

template <int T>
__global__ void __launch_bounds__(kRRThreads) k_gram2(const double* __restrict__ A, const double* __restrict__ Bm,
                                                      long long N, int B, double* __restrict__ C)
{
    constexpr int BP = 16 * T, R = kRRRows;
    extern __shared__ __align__(16) double sm[];
    const bool same = (A == Bm);
    double* sA = sm;                               // [2][R][BP]
    double* sB = same ? sm : sm + 2 * R * BP;      // [2][R][BP]
    const int ti = threadIdx.x / 16, tj = threadIdx.x % 16;
    for (int i = threadIdx.x; i < (same ? 2 : 4) * R * BP; i += kRRThreads) sm[i] = 0.0;  // the pad columns stay 0
    __syncthreads();
    double acc[T][T];
#pragma unroll
    for (int a = 0; a < T; ++a)
#pragma unroll
        for (int b = 0; b < T; ++b) acc[a][b] = 0.0;
    const long long ntiles = (N + R - 1) / R;
    long long tile = blockIdx.x;
    if (tile < ntiles) {
        rr_stage(sA, A, tile * R, R, N, B, BP);
        if (!same) rr_stage(sB, Bm, tile * R, R, N, B, BP);
    }
    rr_commit();
    int st = 0;
    for (; tile < ntiles; tile += gridDim.x, st ^= 1) {
        const long long nxt = tile + gridDim.x;
        if (nxt < ntiles) {
            rr_stage(sA + (st ^ 1) * R * BP, A, nxt * R, R, N, B, BP);
            if (!same) rr_stage(sB + (st ^ 1) * R * BP, Bm, nxt * R, R, N, B, BP);
        }
        rr_commit();
        rr_wait<1>();
        __syncthreads();
        const double* pa = sA + st * R * BP;
        const double* pb = sB + st * R * BP;
#pragma unroll 4
        for (int r = 0; r < R; ++r) {
            double a[T], b[T];
#pragma unroll
            for (int k = 0; k < T; k += 2) {
                const double2 va = *reinterpret_cast<const double2*>(pa + r * BP + rr_own(ti, k));
                const double2 vb = *reinterpret_cast<const double2*>(pb + r * BP + rr_own(tj, k));
                a[k] = va.x; a[k + 1] = va.y; b[k] = vb.x; b[k + 1] = vb.y;
            }
#pragma unroll
            for (int x = 0; x < T; ++x)
#pragma unroll
                for (int y = 0; y < T; ++y) acc[x][y] = fma(a[x], b[y], acc[x][y]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int x = 0; x < T; ++x)
#pragma unroll
        for (int y = 0; y < T; ++y) {
            const int i = rr_own(ti, x), j = rr_own(tj, y);
            if (i < B && j < B) atomicAdd(C + (size_t)i * B + j, acc[x][y]);
        }
}

// RT rows per thread (tile of 16*RT rows), T columns per thread; the B x B factor stays in shared memory
template <int T, int RT>
__global__ void __launch_bounds__(kRRThreads) k_rightmul2(const double* Y, const double* __restrict__ Rm, double* Out,
                                                          int accumulate, long long N, int B)
{
    constexpr int BP = 16 * T, R = 16 * RT;
    extern __shared__ __align__(16) double sm[];
    double* sR = sm;                 // [B][BP]
    double* sY = sm + (size_t)B * BP;  // [2][R][BP]
    const int ti = threadIdx.x / 16, tj = threadIdx.x % 16;
    for (int i = threadIdx.x; i < B * BP + 2 * R * BP; i += kRRThreads) sm[i] = 0.0;
    __syncthreads();
    for (int i = threadIdx.x; i < B * B; i += kRRThreads) sR[(i / B) * BP + (i % B)] = Rm[i];
    const long long ntiles = (N + R - 1) / R;
    long long tile = blockIdx.x;
    if (tile < ntiles) rr_stage(sY, Y, tile * R, R, N, B, BP);
    rr_commit();
    int st = 0;
    for (; tile < ntiles; tile += gridDim.x, st ^= 1) {
        const long long nxt = tile + gridDim.x;
        if (nxt < ntiles) rr_stage(sY + (st ^ 1) * R * BP, Y, nxt * R, R, N, B, BP);
        rr_commit();
        rr_wait<1>();
        __syncthreads();
        const double* py = sY + st * R * BP;
        double acc[RT][T];
#pragma unroll
        for (int a = 0; a < RT; ++a)
#pragma unroll
            for (int b = 0; b < T; ++b) acc[a][b] = 0.0;
#pragma unroll 2
        for (int i = 0; i < B; i += 2) {  // B is even
            double2 y[RT];
#pragma unroll
            for (int m = 0; m < RT; ++m) y[m] = *reinterpret_cast<const double2*>(py + (ti + 16 * m) * BP + i);
#pragma unroll
            for (int k = 0; k < T; k += 2) {
                const double2 r0 = *reinterpret_cast<const double2*>(sR + i * BP + rr_own(tj, k));
                const double2 r1 = *reinterpret_cast<const double2*>(sR + (i + 1) * BP + rr_own(tj, k));
#pragma unroll
                for (int m = 0; m < RT; ++m) {
                    acc[m][k] = fma(y[m].x, r0.x, acc[m][k]);
                    acc[m][k + 1] = fma(y[m].x, r0.y, acc[m][k + 1]);
                    acc[m][k] = fma(y[m].y, r1.x, acc[m][k]);
                    acc[m][k + 1] = fma(y[m].y, r1.y, acc[m][k + 1]);
                }
            }
        }
        const long long r0g = tile * R;
#pragma unroll
        for (int m = 0; m < RT; ++m) {
            const long long r = r0g + ti + 16 * m;
            if (r < N) {
#pragma unroll
                for (int k = 0; k < T; k += 2) {
                    const int j = rr_own(tj, k);
                    if (j < B) {  // j even and B even: the pair is inside
                        double2 o = make_double2(acc[m][k], acc[m][k + 1]);
                        double2* dst = reinterpret_cast<double2*>(Out + r * B + j);
                        if (accumulate) { const double2 old = *dst; o.x += old.x; o.y += old.y; }
                        *dst = o;
                    }
                }
            }
        }
        __syncthreads();
    }
}

// ---- Gram product on the FP64 tensor path: mma.sync.m8n8k4.f64 (DMMA) ------------------------------------------------------
// C = A^T Bm is a pure contraction over the N rows, so it belongs on DMMA (same peak as DFMA on sm_100a, fe_diag.cuh, but
// 1/8 of the issue slots and no shared-memory read per FMA): every warp owns 32 x (32 NJ/4) of the BB x BB result, i.e.
// 4 x NJ accumulator tiles of 8 x 8, and per step of 4 rows loads 4 + NJ fragments for 4 NJ MMAs.  Fragment of the row
// block [r0, r0+4) and the column block [c0, c0+8): lane t holds M[r0 + t%4][c0 + t/4] for the A and the B operand alike
// (A^T is the .row operand, Bm the .col operand).  Row pitch BB + 4 doubles makes those reads conflict-free.  BB = 32, 64
// or 128; 8 warps per CTA split the result tiles and, where there are fewer than 8 tiles, the k steps among them.
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int BB>
__global__ void __launch_bounds__(256) k_gram_mma(const double* __restrict__ A, const double* __restrict__ Bm,
                                                  long long N, double* __restrict__ C)
{
    constexpr int S = BB + 4, R = BB == 32 ? 64 : 32;  // smem row pitch, rows per stage
    constexpr int TI = BB / 32;                        // 32-wide blocks of the result per dimension
    constexpr int NJ = BB == 128 ? 8 : 4;              // 8-wide column tiles per warp (128: two 32-blocks side by side)
    constexpr int NT = BB == 128 ? 8 : TI * TI;        // warp tiles of the result
    constexpr int KS = 8 / NT;                         // warps that share a tile split the k steps
    extern __shared__ __align__(16) double sm[];
    const bool same = (A == Bm);
    double* sA = sm;                                // [2][R][S]
    double* sB = same ? sm : sm + 2 * R * S;        // [2][R][S]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = warp % NT, kpart = warp / NT;
    const int i0 = (BB == 128 ? tile / 2 : tile / TI) * 32, j0 = (BB == 128 ? (tile % 2) * 64 : (tile % TI) * 32);
    const int fr = lane & 3, fc = lane >> 2;
    double acc[4][NJ][2];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < NJ; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
    auto stage = [&](double* dst, const double* src, long long r0) {
        constexpr int chunks = BB / 2;
        for (int i = threadIdx.x; i < R * chunks; i += 256) {
            const int r = i / chunks, c = i - r * chunks;
            const bool ok = r0 + r < N;
            rr_cp16(dst + r * S + 2 * c, src + (ok ? (r0 + r) * BB + 2 * c : 0), ok);
        }
    };
    const long long ntiles = (N + R - 1) / R;
    long long t = blockIdx.x;
    if (t < ntiles) {
        stage(sA, A, t * R);
        if (!same) stage(sB, Bm, t * R);
    }
    rr_commit();
    int st = 0;
    for (; t < ntiles; t += gridDim.x, st ^= 1) {
        const long long nxt = t + gridDim.x;
        if (nxt < ntiles) {
            stage(sA + (st ^ 1) * R * S, A, nxt * R);
            if (!same) stage(sB + (st ^ 1) * R * S, Bm, nxt * R);
        }
        rr_commit();
        rr_wait<1>();
        __syncthreads();
        const double* pa = sA + st * R * S + fr * S + i0 + fc;
        const double* pb = sB + st * R * S + fr * S + j0 + fc;
#pragma unroll
        for (int kk = kpart; kk < R / 4; kk += KS) {
            double a[4], b[NJ];
#pragma unroll
            for (int m = 0; m < 4; ++m) a[m] = pa[kk * 4 * S + 8 * m];
#pragma unroll
            for (int q = 0; q < NJ; ++q) b[q] = pb[kk * 4 * S + 8 * q];
#pragma unroll
            for (int m = 0; m < 4; ++m)
#pragma unroll
                for (int q = 0; q < NJ; ++q) dmma884(acc[m][q][0], acc[m][q][1], a[m], b[q]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int q = 0; q < NJ; ++q) {
            double* c = C + (size_t)(i0 + 8 * m + fc) * BB + j0 + 8 * q + 2 * fr;
            atomicAdd(c, acc[m][q][0]);
            atomicAdd(c + 1, acc[m][q][1]);
        }
}

template <int BB>
cudaError_t launch_gram_mma(const double* A, const double* Bm, long long N, double* C, int sms, cudaStream_t st)
{
    const size_t full = (size_t)4 * (BB == 32 ? 64 : 32) * (BB + 4) * sizeof(double);
    const size_t smem = A == Bm ? full / 2 : full;
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_gram_mma<BB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)full);
    });
    if (e0 != cudaSuccess) return e0;
    k_gram_mma<BB><<<sms * (BB == 128 ? 1 : 2), 256, smem, st>>>(A, Bm, N, C);
    return cudaGetLastError();
}

// Out = Y Rm (+ Out) on DMMA: a CTA stages ROWS rows of Y (two-stage ring) and keeps the BB x BB factor in shared memory;
// the .row operand is the Y tile (lane t holds Y[r0 + t/4][k0 + t%4]), the .col operand the factor (Rm[k0 + t%4][j0 + t/4]),
// both conflict-free at pitch BB + 4.  Warp tiles: BB = 64: 16 rows x 32 columns (64-row tiles); BB = 128: 8 rows x 64
// columns (32-row tiles); BB = 32: 8 rows x 32 columns (64-row tiles).  In place is fine: a tile is staged before it is written.
template <int BB>
__global__ void __launch_bounds__(256) k_rightmul_mma(const double* Y, const double* __restrict__ Rm, double* Out,
                                                      int accumulate, long long N)
{
    constexpr int S = BB + 4;
    constexpr int ROWS = BB == 128 ? 32 : 64;
    constexpr int MI = BB == 64 ? 2 : 1, NJ = BB == 128 ? 8 : 4;       // warp tile = 8 MI rows x 8 NJ columns
    constexpr int WR = ROWS / (8 * MI);                                 // warps along the rows
    extern __shared__ __align__(16) double sm[];
    double* sR = sm;                     // [BB][S]
    double* sY = sm + (size_t)BB * S;    // [2][ROWS][S]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int fr = lane & 3, fc = lane >> 2;
    const int r0w = (warp % WR) * 8 * MI, j0 = (warp / WR) * 8 * NJ;
    for (int i = threadIdx.x; i < BB * BB; i += 256) sR[(i / BB) * S + (i % BB)] = Rm[i];
    auto stage = [&](double* dst, long long r0) {
        constexpr int chunks = BB / 2;
        for (int i = threadIdx.x; i < ROWS * chunks; i += 256) {
            const int r = i / chunks, c = i - r * chunks;
            const bool ok = r0 + r < N;
            rr_cp16(dst + r * S + 2 * c, Y + (ok ? (r0 + r) * BB + 2 * c : 0), ok);
        }
    };
    const long long ntiles = (N + ROWS - 1) / ROWS;
    long long t = blockIdx.x;
    if (t < ntiles) stage(sY, t * ROWS);
    rr_commit();
    int st = 0;
    for (; t < ntiles; t += gridDim.x, st ^= 1) {
        const long long nxt = t + gridDim.x;
        if (nxt < ntiles) stage(sY + (st ^ 1) * ROWS * S, nxt * ROWS);
        rr_commit();
        rr_wait<1>();
        __syncthreads();
        double acc[MI][NJ][2];
#pragma unroll
        for (int m = 0; m < MI; ++m)
#pragma unroll
            for (int q = 0; q < NJ; ++q) acc[m][q][0] = acc[m][q][1] = 0.0;
        const double* py = sY + st * ROWS * S + (r0w + fc) * S + fr;
        const double* pr = sR + fr * S + j0 + fc;
#pragma unroll 4
        for (int k = 0; k < BB; k += 4) {
            double a[MI], b[NJ];
#pragma unroll
            for (int m = 0; m < MI; ++m) a[m] = py[8 * m * S + k];
#pragma unroll
            for (int q = 0; q < NJ; ++q) b[q] = pr[k * S + 8 * q];
#pragma unroll
            for (int m = 0; m < MI; ++m)
#pragma unroll
                for (int q = 0; q < NJ; ++q) dmma884(acc[m][q][0], acc[m][q][1], a[m], b[q]);
        }
        const long long rg = t * ROWS + r0w + fc;
#pragma unroll
        for (int m = 0; m < MI; ++m) {
            const long long r = rg + 8 * m;
            if (r < N) {
#pragma unroll
                for (int q = 0; q < NJ; ++q) {
                    double2 o = make_double2(acc[m][q][0], acc[m][q][1]);
                    double2* dst = reinterpret_cast<double2*>(Out + r * BB + j0 + 8 * q + 2 * fr);
                    if (accumulate) { const double2 old = *dst; o.x += old.x; o.y += old.y; }
                    *dst = o;
                }
            }
        }
        __syncthreads();
    }
}

template <int BB>
cudaError_t launch_rightmul_mma(const double* Y, const double* R, double* Out, int accumulate, long long N, int sms,
                                cudaStream_t st)
{
    constexpr int ROWS = BB == 128 ? 32 : 64;
    const size_t smem = ((size_t)BB + 2 * ROWS) * (BB + 4) * sizeof(double);
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_rightmul_mma<BB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    k_rightmul_mma<BB><<<sms * (BB == 128 ? 1 : 2), 256, smem, st>>>(Y, R, Out, accumulate, N);
    return cudaGetLastError();
}

template <int T>
cudaError_t launch_gram2(const double* A, const double* Bm, long long N, int B, double* C, int sms, cudaStream_t st)
{
    const size_t smem = (size_t)(A == Bm ? 2 : 4) * kRRRows * 16 * T * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(k_gram2<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * kRRRows * 16 * T * 8);
    if (e != cudaSuccess) return e;
    k_gram2<T><<<sms * 2, kRRThreads, smem, st>>>(A, Bm, N, B, C);
    return cudaGetLastError();
}

template <int T, int RT>
cudaError_t launch_rightmul2(const double* Y, const double* R, double* Out, int accumulate, long long N, int B, int sms,
                             cudaStream_t st)
{
    const size_t smem = ((size_t)B * 16 * T + (size_t)2 * 16 * RT * 16 * T) * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(k_rightmul2<T, RT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_rightmul2<T, RT><<<sms * (smem > 100 * 1024 ? 1 : 2), kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    return cudaGetLastError();
}

inline cudaError_t launch_gram(const double* A, const double* Bm, long long N, int B, double* C, int sms, cudaStream_t st)
{
    const size_t smem = (size_t)2 * kRRRows * B * sizeof(double);
    const int T = (B + 15) / 16;
    if (T > 8) return cudaErrorInvalidValue;
    if ((((uintptr_t)A | (uintptr_t)Bm) & 15) == 0) {  // 16-byte aligned rows, B = 32 / 64 / 128: the DMMA kernel
        if (B == 32) return launch_gram_mma<32>(A, Bm, N, C, sms, st);
        if (B == 64) return launch_gram_mma<64>(A, Bm, N, C, sms, st);
        if (B == 128) return launch_gram_mma<128>(A, Bm, N, C, sms, st);
    }
    if (B % 2 == 0 && (((uintptr_t)A | (uintptr_t)Bm) & 15) == 0) {  // even B, 16-byte aligned rows: the fast DFMA path
        if (T <= 2) return launch_gram2<2>(A, Bm, N, B, C, sms, st);
        if (T <= 4) return launch_gram2<4>(A, Bm, N, B, C, sms, st);
        if (T <= 6) return launch_gram2<6>(A, Bm, N, B, C, sms, st);
        return launch_gram2<8>(A, Bm, N, B, C, sms, st);
    }
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_gram<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * kRRRows * 128 * 8);
    });
    if (e0 != cudaSuccess) return e0;
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
    if ((((uintptr_t)Y | (uintptr_t)Out) & 15) == 0) {  // B = 32 / 64 / 128: the DMMA kernel
        if (B == 32) return launch_rightmul_mma<32>(Y, R, Out, accumulate, N, sms, st);
        if (B == 64) return launch_rightmul_mma<64>(Y, R, Out, accumulate, N, sms, st);
        if (B == 128) return launch_rightmul_mma<128>(Y, R, Out, accumulate, N, sms, st);
    }
    if (B % 2 == 0 && (((uintptr_t)Y | (uintptr_t)Out) & 15) == 0) {
        if (T <= 2) return launch_rightmul2<2, 4>(Y, R, Out, accumulate, N, B, sms, st);
        if (T <= 4) return launch_rightmul2<4, 4>(Y, R, Out, accumulate, N, B, sms, st);
        if (T <= 6) return launch_rightmul2<6, 2>(Y, R, Out, accumulate, N, B, sms, st);
        return launch_rightmul2<8, 2>(Y, R, Out, accumulate, N, B, sms, st);
    }
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        const int mx = (128 * 128 + kRRRows * 129) * 8;
        cudaError_t e = cudaFuncSetAttribute(k_rightmul<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rightmul<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rightmul<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_rightmul<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
        return e;
    });
    if (e0 != cudaSuccess) return e0;
    const int grid = sms * (B > 64 ? 1 : 2);
    if (T <= 1) k_rightmul<1><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    else if (T <= 2) k_rightmul<2><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    else if (T <= 4) k_rightmul<4><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    else k_rightmul<8><<<grid, kRRThreads, smem, st>>>(Y, R, Out, accumulate, N, B);
    return cudaGetLastError();
}

}  // namespace fecheb
