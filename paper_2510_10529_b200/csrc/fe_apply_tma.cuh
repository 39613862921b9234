// fe_apply_tma.cuh -- the TMA generation of the fused operator step (sm_100a)
//
//   Y[g,j] (+)= s_g sum_{e∋g} yhat_e[a,j]  +  kappa_j X[g,j]          (reduce-add into a pre-initialised Y)
//   W[g,j]   = beta' X[g,j]                                            (pre-initialises the NEXT step's target)
//
// One CTA = one cell x BT vectors.  a1 (gather) is ONE cp.async.bulk.tensor load of the cell's n x n x n x BT box of
// X (the layout of PAPER.md l.233-235 makes the block a 4-D tensor (j, gx, gy, gz)); a3 (scatter) is one
// cp.reduce.async.bulk.tensor .add per nodal plane, so no thread computes a global address or issues an atomic.
// The recurrence terms of the Chebyshev step (l.208-210; R7) need no read of Y_{k-1} at all: step k-1 stores
// beta_k Y_{k-1} into the buffer that becomes Y_{k+1} (the "pre-initialisation"), and step k adds
// kappa_j Y_k = -alpha (c + eps_j) Y_k from the owner cell of each node plus alpha s_g sum_e yhat_e.
//
// Cell contraction (a2; Eq. 17 l.171 on an axis-aligned box cell), with the Gauss weights folded into the tables,
// N' = diag(sqrt w) N, G' = diag(w^-1/2) (D~^T W D~) diag(w^-1/2), and everything divided by kz = 2J/hz^2:
//   A  = (N'y N'x) xhat                 A2 = G'x A + (ky/kx) G'y A                     per nodal z-plane
//   U  = N'z A ;  T = VZ.U + G'z U + (kx/kz) N'z A2 ;  R = N'z^T T                      per (qx,qy) line
//   yhat/kz = N'x^T N'y^T R                                                            per nodal z-plane
// VZ = V_q hz^2/2 (= J V_q / kz); the output scale tile carries alpha kz s_g.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "fe_kernels.cuh"

namespace fecheb {

struct TmaParams {
    CUtensorMap mXn;   // X : box (BT,n,n,n), load
    CUtensorMap mYn1;  // Y : box (BT,n,n,1), reduce-add
    CUtensorMap mYp1;  // Y : box (BT,p,p,1), reduce-add of the owner term kappa_j X
    CUtensorMap mWp1;  // W : box (BT,p,p,1), store of beta' X
    const double* eps;
    const double* VZ;  // cells * n*n*NP: V_q hz^2/2, [qx][qy][qz padded to NP]
    const double *sx, *sy, *sz;  // per-axis mu M^{-1/2}
    const double *gx, *gy, *gz;  // per-axis cell geometry, 4 doubles per cell: h, h^2, 1/h^2, 1/h
    int B, cx, cy, cz;
    int owner, preinit;
    double alpha, c, beta_next;
    EOTab eoN, eoNT, eoG;  // even-odd halves of N', N'^T, G'
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    unsigned ok = 0;
    while (!ok)
        asm volatile("{.reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0,1,0,p;}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load4(void* dst, const CUtensorMap* m, int c0, int c1, int c2, int c3,
                                          unsigned long long* bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2,%3,%4,%5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(m), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_reduce_add4(const CUtensorMap* m, const void* src, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group [%0, {%2,%3,%4,%5}], [%1];"
                 ::"l"(m), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_store4(const CUtensorMap* m, const void* src, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%2,%3,%4,%5}], [%1];"
                 ::"l"(m), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int n>
struct TmaShape {
    static constexpr int NP = n + (n & 1);  // rows of the small tiles padded to an even length (16-byte LDS.128)
    static constexpr int SMALL = n * n * NP;
};

template <int P, int BT>
constexpr size_t tma_smem_bytes()
{
    constexpr int n = P + 1;
    return ((size_t)2 * n * n * n * BT + 3 * TmaShape<n>::SMALL) * sizeof(double) + 16;
}

// FIRST: X is caller data whose Dirichlet rows may hold anything (R5) -> mask them in the owner / pre-init terms.
template <int P, int BT, int MINB, bool FIRST, bool PERSIST>
__global__ void __launch_bounds__((P + 1) * BT, MINB) k_apply_tma(const __grid_constant__ TmaParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n, NP = TmaShape<n>::NP, SMALL = TmaShape<n>::SMALL;
    extern __shared__ __align__(128) double smem[];
    double* buf0 = smem;                // [n^3][BT]  the two tile buffers swap roles every unit:
    double* buf1 = smem + n3 * BT;      // [n^3][BT]    bufX: X -> A -> R -> scaled output;  bufO: owner term -> A2 -> next X
    double* sVZ = buf1 + n3 * BT;       // [qx][qy][NP]
    double* sIn = sVZ + SMALL;          // [az][ay][NP]  s_g
    double* sOut = sIn + SMALL;         // [az][ay][NP]  alpha kz s_g
    unsigned long long* bar = (unsigned long long*)(sOut + SMALL);
    const int lane = threadIdx.x, pl = threadIdx.y, tid = pl * BT + lane;
    const int nbt = (prm.B + BT - 1) / BT;
    const long long nunits = (long long)prm.cx * prm.cy * prm.cz * nbt;  // unit = (cell, tile of BT vectors), tile fastest
    const bool issuer = (lane == 0) && (pl < P);
    const bool early = prm.owner || prm.preinit;

    if (tid == 0) {
        mbar_init(bar, 1);
        const long long u = blockIdx.x;
        const int cell = (int)(u / nbt), ex = cell % prm.cx, ey = (cell / prm.cx) % prm.cy, ez = cell / (prm.cx * prm.cy);
        mbar_expect_tx(bar, (unsigned)((n3 * BT + SMALL) * sizeof(double)));
        tma_load4(buf0, &prm.mXn, (int)(u % nbt) * BT, ex * P, ey * P, ez * P, bar);
        bulk_load(sVZ, prm.VZ + (size_t)cell * SMALL, (unsigned)(SMALL * sizeof(double)), bar);
    }
    __syncthreads();
    unsigned parity = 0;
    double* bufA = buf0;
    double* bufB = buf1;
    // persistent over units: the next unit's X tile lands in bufB while plane phase 2 of this unit runs out of bufA
    for (long long u = blockIdx.x; u < nunits; u += gridDim.x) {
    const int cell = (int)(u / nbt);
    const int ex = cell % prm.cx, ey = (cell / prm.cx) % prm.cy, ez = cell / (prm.cx * prm.cy);
    const int j0 = (int)(u % nbt) * BT;
    const int gx0 = ex * P, gy0 = ey * P, gz0 = ez * P;
    const double4 qx = *reinterpret_cast<const double4*>(prm.gx + 4 * ex);
    const double4 qy = *reinterpret_cast<const double4*>(prm.gy + 4 * ey);
    const double4 qz = *reinterpret_cast<const double4*>(prm.gz + 4 * ez);
    {   // scale tiles of this thread's own nodal plane (read back only by the lanes of this plane)
        const double akz = prm.alpha * 0.25 * qx.x * qy.x * qz.w;  // alpha * 2J/hz^2, J = hx hy hz / 8
        const double szv = prm.sz[gz0 + pl];
        for (int i = lane; i < n * NP; i += BT) {
            const int ax = i % NP, ay = i / NP;
            const double s = ax < n ? prm.sx[gx0 + ax] * prm.sy[gy0 + ay] * szv : 0.0;
            sIn[pl * n * NP + i] = s;
            sOut[pl * n * NP + i] = akz * s;
        }
    }
    const double ry = qx.y * qy.z;   // ky/kx = hx^2/hy^2
    const double rxz = qz.y * qx.z;  // kx/kz = hz^2/hx^2
    double kappa = 0.0;
    if (prm.owner) {
        const int j = j0 + lane;
        kappa = -prm.alpha * (prm.c + ((prm.eps && j < prm.B) ? prm.eps[j] : 0.0));
    }
    if (lane == 0) bulk_wait_read0();  // the previous unit's reduce-add has read its source (now bufB)
    __syncwarp();
    mbar_wait(bar, parity);
    parity ^= 1;

    double v[n][n], t[n], o[n];
    double* pA = bufA + (size_t)pl * n2 * BT + lane;
    double* pB = bufB + (size_t)pl * n2 * BT + lane;
    const double* sin_pl = sIn + pl * n * NP;
    // ---- plane phase 1 -------------------------------------------------------------------------------------------
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) v[ay][ax] = pA[(ay * n + ax) * BT];
    if (early) {
        if (pl < P) {
            // compact p x p sub-planes: beta' X -> own plane of bufA (store to W), kappa X -> own plane of bufB (add to Y)
#pragma unroll
            for (int ay = 0; ay < P; ++ay)
#pragma unroll
                for (int ax = 0; ax < P; ++ax) {
                    double x = v[ay][ax];
                    if (FIRST) x = (__double2hiint(sin_pl[ay * NP + ax]) != 0) ? x : 0.0;
                    if (prm.preinit) pA[(ay * P + ax) * BT] = prm.beta_next * x;
                    if (prm.owner) pB[(ay * P + ax) * BT] = kappa * x;
                }
            fence_async_smem();
        }
        __syncwarp();
        if (issuer) {
            if (prm.preinit) tma_store4(&prm.mWp1, pA, j0, gx0, gy0, gz0 + pl);
            if (prm.owner) tma_reduce_add4(&prm.mYp1, pB, j0, gx0, gy0, gz0 + pl);
            bulk_commit();
        }
    }
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) v[ay][ax] *= sin_pl[ay * NP + ax];
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
        for (int q = 0; q < n; ++q) v[q][qx] = o[q];
    }
    if (early) {  // the bulk operations must have read their shared-memory sources before A / A2 overwrite them
        if (issuer) bulk_wait_read0();
        __syncwarp();
    }
    if constexpr (n >= 7) {
        // large planes: park A in shared memory first and re-read its columns for the y stiffness, so that only one
        // plane (plus a line) is live in registers instead of two
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) pA[(qy * n + qx) * BT] = v[qy][qx];
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoG, v[qy], o);
#pragma unroll
            for (int qx = 0; qx < n; ++qx) v[qy][qx] = o[qx];
        }
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int a = 0; a < n; ++a) t[a] = pA[(a * n + qx) * BT];
            mat1d_eo<n>(prm.eoG, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) pB[(qy * n + qx) * BT] = fma(ry, o[qy], v[qy][qx]);
        }
    } else {
        double v2[n][n];
#pragma unroll
        for (int qy = 0; qy < n; ++qy) mat1d_eo<n>(prm.eoG, v[qy], v2[qy]);
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int a = 0; a < n; ++a) t[a] = v[a][qx];
            mat1d_eo<n>(prm.eoG, t, o);
#pragma unroll
            for (int qy = 0; qy < n; ++qy) v2[qy][qx] = fma(ry, o[qy], v2[qy][qx]);
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) {
                pA[(qy * n + qx) * BT] = v[qy][qx];
                pB[(qy * n + qx) * BT] = v2[qy][qx];
            }
    }
    __syncthreads();
    // ---- line phase as four plane passes: the thread owns the yz-plane qx = pl; one 1-D table per pass ----------------
    {
        double* la = bufA + (size_t)pl * BT + lane;  // + ((az*n + qy)*n)*BT
        double* lb = bufB + (size_t)pl * BT + lane;
        const double* lv = sVZ + pl * n * NP;        // + qy*NP + qz
        // pass 1: U = N'z A
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int az = 0; az < n; ++az) t[az] = la[((az * n + qy) * n) * BT];
            mat1d_eo<n>(prm.eoN, t, v[qy]);
        }
        // pass 2: T = VZ . U + G'z U
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoG, v[qy], o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) v[qy][qz] = fma(lv[qy * NP + qz], v[qy][qz], o[qz]);
        }
        // pass 3: T += (kx/kz) N'z A2
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int az = 0; az < n; ++az) t[az] = lb[((az * n + qy) * n) * BT];
            mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) v[qy][qz] = fma(rxz, o[qz], v[qy][qz]);
        }
        // pass 4: R = N'z^T T, back into the A field
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoNT, v[qy], o);
#pragma unroll
            for (int az = 0; az < n; ++az) la[((az * n + qy) * n) * BT] = o[az];
        }
    }
    __syncthreads();
    if (PERSIST && tid == 0 && u + gridDim.x < nunits) {  // bufB (A2) and sVZ are dead: bring in the next unit
        const long long un = u + gridDim.x;
        const int cn = (int)(un / nbt), nx = cn % prm.cx, ny = (cn / prm.cx) % prm.cy, nz = cn / (prm.cx * prm.cy);
        mbar_expect_tx(bar, (unsigned)((n3 * BT + SMALL) * sizeof(double)));
        tma_load4(bufB, &prm.mXn, (int)(un % nbt) * BT, nx * P, ny * P, nz * P, bar);
        bulk_load(sVZ, prm.VZ + (size_t)cn * SMALL, (unsigned)(SMALL * sizeof(double)), bar);
    }
    // ---- plane phase 2: back-interpolate in y and x, scale by alpha kz s_g, one bulk reduce-add per nodal plane ---------
#pragma unroll
    for (int qy = 0; qy < n; ++qy)
#pragma unroll
        for (int qx = 0; qx < n; ++qx) v[qy][qx] = pA[(qy * n + qx) * BT];
#pragma unroll
    for (int qx = 0; qx < n; ++qx) {
#pragma unroll
        for (int q = 0; q < n; ++q) t[q] = v[q][qx];
        mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
        for (int a = 0; a < n; ++a) v[a][qx] = o[a];
    }
    const double* sout_pl = sOut + pl * n * NP;
#pragma unroll
    for (int ay = 0; ay < n; ++ay) {
        mat1d_eo<n>(prm.eoNT, v[ay], o);
#pragma unroll
        for (int ax = 0; ax < n; ++ax) pA[(ay * n + ax) * BT] = sout_pl[ay * NP + ax] * o[ax];
    }
    fence_async_smem();
    __syncwarp();
    if (lane == 0) {
        tma_reduce_add4(&prm.mYn1, pA, j0, gx0, gy0, gz0 + pl);
        bulk_commit();
    }
    if (!PERSIST) break;
    double* tmp = bufA; bufA = bufB; bufB = tmp;
    }  // units
    if (lane == 0) bulk_wait_read0();  // shared memory must stay valid until the bulk engine has read it
}

// ctas > 0: persistent launch with that many CTAs (each walks units blockIdx.x, +ctas, ...); 0: one CTA per unit
template <int P, int BT, int MINB>
cudaError_t launch_tma(const TmaParams& prm, long long ncells, bool first, cudaStream_t st, int ctas)
{
    constexpr int n = P + 1;
    constexpr size_t smem = tma_smem_bytes<P, BT>();
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const long long nunits = ncells * ((prm.B + BT - 1) / BT);
    const bool persist = ctas > 0 && (long long)ctas * MINB < nunits;
    dim3 grid((unsigned)(persist ? (long long)ctas * MINB : nunits)), block(BT, n);
    if (persist) {
        if (first)
            k_apply_tma<P, BT, MINB, true, true><<<grid, block, smem, st>>>(prm);
        else
            k_apply_tma<P, BT, MINB, false, true><<<grid, block, smem, st>>>(prm);
    } else {
        if (first)
            k_apply_tma<P, BT, MINB, true, false><<<grid, block, smem, st>>>(prm);
        else
            k_apply_tma<P, BT, MINB, false, false><<<grid, block, smem, st>>>(prm);
    }
    return cudaGetLastError();
}

// Launch shape of the TMA kernel.  Variants: 0 = default, 5 = one CTA per unit everywhere, 6 = 32-wide box at p = 6 with
// one CTA per unit, 7 = persistent everywhere, 8 = 32-wide persistent at p = 6 (= the default when B > 16).
// p = 6 default: ONE persistent 7-warp CTA per SM walking (cell, 32 vectors) units.  Its warps run the same 74 KB of
// straight-line code nearly in lockstep and share instruction-cache lines; two independent 16-wide CTAs per SM
// each stream the code through the 32 KB L1.5 on their own (ncu: no_instruction stall 0.9 -> 0.08 per issue).
inline bool tma_wide6(int p, int variant, int B)
{
    return p == 6 && (variant == 6 || variant == 8 || (variant == 0 && B > 16));
}
inline int tma_bt(int p, int variant, int B) { return (p >= 6 && !tma_wide6(p, variant, B)) ? 16 : 32; }

inline cudaError_t launch_apply_tma(const TmaParams& prm, int p, long long ncells, bool first, cudaStream_t st,
                                    int variant, int sms)
{
    const bool wide6 = tma_wide6(p, variant, prm.B);
    if (!(variant == 7 || variant == 8 || (variant == 0 && wide6))) sms = 0;
    if (wide6) return launch_tma<6, 32, 1>(prm, ncells, first, st, sms);
    switch (p) {
        case 1: return launch_tma<1, 32, 8>(prm, ncells, first, st, sms);
        case 2: return launch_tma<2, 32, 6>(prm, ncells, first, st, sms);
        case 3: return launch_tma<3, 32, 4>(prm, ncells, first, st, sms);
        case 4: return launch_tma<4, 32, 3>(prm, ncells, first, st, sms);
        case 5: return launch_tma<5, 32, 1>(prm, ncells, first, st, sms);
        case 6: return launch_tma<6, 16, 2>(prm, ncells, first, st, sms);
        case 7: return launch_tma<7, 16, 1>(prm, ncells, first, st, sms);
        case 8: return launch_tma<8, 16, 1>(prm, ncells, first, st, sms);
    }
    return cudaErrorInvalidValue;
}

// zero the six boundary faces of a node-major block (rows of B doubles)
__global__ void k_zero_faces(double* __restrict__ Y, long long Nx, long long Ny, long long Nz, int B)
{
    const long long nf = 2 * (Nx * Ny + Ny * Nz + Nx * Nz);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < nf * B; i += (long long)gridDim.x * blockDim.x) {
        long long f = i / B;
        const int j = (int)(i - f * B);
        long long gx, gy, gz;
        if (f < 2 * Nx * Ny) {
            gz = (f >= Nx * Ny) ? Nz - 1 : 0; f %= Nx * Ny; gx = f % Nx; gy = f / Nx;
        } else if ((f -= 2 * Nx * Ny) < 2 * Ny * Nz) {
            gx = (f >= Ny * Nz) ? Nx - 1 : 0; f %= Ny * Nz; gy = f % Ny; gz = f / Ny;
        } else {
            f -= 2 * Ny * Nz;
            gy = (f >= Nx * Nz) ? Ny - 1 : 0; f %= Nx * Nz; gx = f % Nx; gz = f / Nx;
        }
        Y[(gx + Nx * (gy + Ny * gz)) * B + j] = 0.0;
    }
}

}  // namespace fecheb
