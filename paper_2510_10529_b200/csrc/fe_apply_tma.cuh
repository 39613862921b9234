// fe_apply_tma.cuh -- the TMA generation of the fused operator step (sm_100a)
//
//   Y[g,j] (+)= s_g sum_{e∋g} yhat_e[a,j]  +  kappa_j X[g,j]          (reduce-add into a pre-initialised Y)
//   W[g,j]   = beta' X[g,j]                                            (pre-initialises the NEXT step's target)
//
// Unit of work = one cell x BT vectors (one CTA per unit, or a persistent CTA walking units).  a1 (gather) is ONE
// cp.async.bulk.tensor load of the cell's n x n x n x BT box of X (the layout of PAPER.md l.233-235 makes the block a
// 4-D tensor (j, gx, gy, gz)); a3 (scatter) is one cp.reduce.async.bulk.tensor .add per nodal plane, so no thread
// computes a global address or issues an atomic.
// The recurrence terms of the Chebyshev step (l.208-210; R7) need no read of Y_{k-1} at all: step k-1 stores
// beta_k Y_{k-1} into the buffer that becomes Y_{k+1} (the "pre-initialisation"), and step k adds
// kappa_j Y_k = -alpha (c + eps_j) Y_k from the owner cell of each node plus alpha s_g sum_e yhat_e.
//
// Cell contraction (a2; Eq. 17 l.171 on an axis-aligned box cell), with the Gauss weights folded into the tables,
// N' = diag(sqrt w) N, G' = diag(w^-1/2) (D~^T W D~) diag(w^-1/2), and everything divided by kz = 2J/hz^2:
//   A  = (N'y N'x) xhat                 A2 = G'x A + (ky/kx) G'y A                     per nodal z-plane
//   U  = N'z A ;  T = VZ.U + G'z U + (kx/kz) N'z A2 ;  R = N'z^T T                      per (qx,qy) line
//   yhat/kz = N'x^T N'y^T R                                                            per nodal z-plane
// VZ = V_q hz^2/2 (= J V_q / kz); the output scale tile carries kz s_g and the last back-interpolation table alpha.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "fe_kernels.cuh"

namespace fecheb {

struct TmaParams {
    CUtensorMap mXn;   // X : box (BT,n,n,n), load
    CUtensorMap mYh1;  // Y : box (BT,n,ceil(n/2),1), reduce-add of the first rows of an output plane
    CUtensorMap mYh2;  // Y : box (BT,n,floor(n/2),1), reduce-add of the remaining rows
    CUtensorMap mYp1;  // Y : box (BT,p,p,1), reduce-add of the owner term kappa_j X
    CUtensorMap mWp1;  // W : box (BT,p,p,1), store of beta' X
    const double* eps;
    double* dots;       // DOTS kernels: dots[j] += sum_g X[g,j] Y_contribution[g,j], the column-wise x . (H~ - eps_j) x of a plain apply
    const double* rec;  // cells * REC: per-cell record  VZ = V_q hz^2/2 [qx][qy][NP] | s_g [az][ay][NP] | ky/kx, kx/kz, kz | kz s_g
    int B, cx, cy, cz;
    int owner, preinit;
    int blk;   // block edge T of the walk order (walk_cell), a divisor of cy and cz
    double alpha, c, beta_next;
    EOTab eoN, eoNT, eoG;  // even-odd halves of N', N'^T, G'
    EOTab eoNTa;           // alpha N'^T (the last back-interpolation carries the step's alpha)
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
__device__ __forceinline__ void bulk_wait_read1() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Walk order of the cells: x fastest inside T x T blocks of (y, z) columns (T divides cy and cz; T = 1 is the plain
// x-y-z order), so that the z-neighbour of a cell is at most T cx cells away in the walk and the shared face is still in
// L2 when it is gathered / reduced into.  `k` is the position in the walk; the record of cell (ex,ey,ez) is at
// ex + cx (ey + cy ez).
__device__ __forceinline__ void walk_cell(int k, int cx, int cy, int T, int& ex, int& ey, int& ez)
{
    const int per = cx * T * T, b = k / per, r = k - b * per, nby = cy / T;
    ex = r % cx;
    const int q = r / cx, ly = q % T, lz = q / T;
    ey = T * (b % nby) + ly;
    ez = T * (b / nby) + lz;
}

template <int n>
struct TmaShape {
    static constexpr int NP = n + (n & 1);  // rows of the small tiles padded to an even length (16-byte LDS.128)
    static constexpr int SMALL = n * n * NP;
    // per-cell record in global memory, brought in by ONE bulk copy per unit: VZ | s_g | ry, rxz, kz, pad | kz s_g
    static constexpr int REC = 3 * SMALL + 8;
    static constexpr int TAIL = 2 * SMALL, SOUT = 2 * SMALL + 8;
    static constexpr int REC_SLIM = 2 * SMALL + 8;  // SLIM kernels leave the kz s_g tile out and multiply by kz instead
};

// STAGED shape (p = 6 at 32 vectors; p = 7 measured no gain): the last rows of every output plane leave from a staging tile of their own instead
// of bufB, so the next unit can write bufB while the bulk engine still reads them (k_apply_tma, plane phase 2)
template <int P, int BT, bool SLIM, bool DOTS>
__host__ __device__ constexpr bool tma_staged() { return !SLIM && !DOTS && P == 6 && BT == 32; }

template <int P, int BT, bool SLIM = false, bool DOTS = false>
constexpr size_t tma_smem_bytes()
{
    constexpr int n = P + 1;
    if (SLIM) return ((size_t)2 * n * n * n * BT + TmaShape<n>::REC_SLIM) * sizeof(double) + 16;
    return ((size_t)2 * n * n * n * BT + 2 * TmaShape<n>::REC + (DOTS ? n * BT : 0) +
            (tma_staged<P, BT, SLIM, DOTS>() ? n * (n / 2) * n * BT : 0)) * sizeof(double) + 16;
}

// FIRST: X is caller data whose Dirichlet rows may hold anything (R5) -> mask them in the owner / pre-init terms.
// DOTS: also accumulate the column-wise inner products x_j . y_j of input and result (MINRES alpha, l.221-225) from
// cell-local terms: x^T y_e = kz U^T T at the Gauss points of the line phase, plus the owner term kappa_j x^2.
// SLIM (one CTA per unit only): one record buffer without the kz s_g tile and no DOTS scratch, so that two 6-warp CTAs of
// p = 5 fit one SM (12 warps, three per sub-partition, instead of one persistent CTA whose 6 warps sit 2,2,1,1).
template <int P, int BT, int MINB, bool FIRST, bool PERSIST, bool DOTS = false, bool SLIM = false>
__global__ void __launch_bounds__((P + 1) * BT, MINB) k_apply_tma(const __grid_constant__ TmaParams prm)
{
    static_assert(!SLIM || (!PERSIST && !DOTS), "SLIM kernels run one unit and deliver no dots");
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n, NP = TmaShape<n>::NP, SMALL = TmaShape<n>::SMALL,
                  REC = SLIM ? TmaShape<n>::REC_SLIM : TmaShape<n>::REC, RECG = TmaShape<n>::REC,
                  TAIL = TmaShape<n>::TAIL, SOUT = TmaShape<n>::SOUT;
    extern __shared__ __align__(128) double smem[];
    double* buf0 = smem;                // [n^3][BT]  bufA: X -> A (dead after pass 1 of the line phase) -> next unit's X
    double* buf1 = smem + n3 * BT;      // [n^3][BT]  bufB: owner term -> A2 -> R -> scaled output (source of the reduce-add)
    double* rec0 = buf1 + n3 * BT;      // two cell records (double-buffered like the tiles): VZ [qx][qy][NP],
    double* rec1 = SLIM ? rec0 : rec0 + REC;  //   s_g [az][ay][NP], {ky/kx, kx/kz, kz}, kz s_g [az][ay][NP]
    constexpr bool STG = tma_staged<P, BT, SLIM, DOTS>();
    constexpr int H2 = n / 2, CPL = H2 * n * BT;  // staging tile: the last H2 rows of each output plane
    double* bufC = rec1 + REC;
    unsigned long long* bar = (unsigned long long*)(bufC + (STG ? n * CPL : 0));  // bar[0]: tile + record landed; bar[1]: A consumed
    double* red = (double*)(bar + 2);   // [n][BT] DOTS: per-plane partial sums of the unit
    const int lane = threadIdx.x, pl = threadIdx.y, tid = pl * BT + lane;
    const int nbt = (prm.B + BT - 1) / BT;
    const long long nunits = (long long)prm.cx * prm.cy * prm.cz * nbt;  // unit = (cell, tile of BT vectors), tile fastest
    const bool issuer = (lane == 0) && (pl < P);
    const bool early = prm.owner || prm.preinit;

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 1, (n * BT + 31) / 32);
        const long long u = blockIdx.x;
        int ex, ey, ez;
        walk_cell((int)(u / nbt), prm.cx, prm.cy, prm.blk, ex, ey, ez);
        const int cell = ex + prm.cx * (ey + prm.cy * ez);
        mbar_expect_tx(bar, (unsigned)((n3 * BT + REC) * sizeof(double)));
        tma_load4(buf0, &prm.mXn, (int)(u % nbt) * BT, ex * P, ey * P, ez * P, bar);
        bulk_load(rec0, prm.rec + (size_t)cell * RECG, (unsigned)(REC * sizeof(double)), bar);
    }
    __syncthreads();
    unsigned parity = 0;
    double* const bufA = buf0;
    double* const bufB = buf1;
    double* rec = rec0;
    double* recN = rec1;
    // persistent over units: the next unit's X tile is requested during the line phase, once every warp is past pass 1
    for (long long u = blockIdx.x; u < nunits; u += gridDim.x) {
    int ex, ey, ez;
    walk_cell((int)(u / nbt), prm.cx, prm.cy, prm.blk, ex, ey, ez);
    const int j0 = (int)(u % nbt) * BT;
    const int gx0 = ex * P, gy0 = ey * P, gz0 = ez * P;
    double kappa = 0.0;
    if (prm.owner) {
        const int j = j0 + lane;
        kappa = -prm.alpha * (prm.c + ((prm.eps && j < prm.B) ? prm.eps[j] : 0.0));
    }
    if (lane == 0) {  // the previous unit's reduce-adds have read their sources in bufB (the staged last one may still be reading)
        if (STG) bulk_wait_read1(); else bulk_wait_read0();
    }
    __syncwarp();
    mbar_wait(bar, parity);
    parity ^= 1;
    const double* sVZ = rec;
    const double* sIn = rec + SMALL;
    const double* sOut = SLIM ? sIn : rec + SOUT;
    const double ry = rec[TAIL], rxz = rec[TAIL + 1];  // ky/kx = hx^2/hy^2, kx/kz = hz^2/hx^2
    const double kzs = SLIM ? rec[TAIL + 2] : 1.0;     // SLIM: the output scale is kz times the gather scale

    double v[n][n], t[n], o[n];
    double dacc = 0.0;  // DOTS: this thread's share of x . y for vector j0 + lane
    double* pA = bufA + (size_t)pl * n2 * BT + lane;
    double* pB = bufB + (size_t)pl * n2 * BT + lane;
    const double* sin_pl = sIn + pl * n * NP;
    // ---- plane phase 1 -------------------------------------------------------------------------------------------
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) v[ay][ax] = pA[(ay * n + ax) * BT];
    if (FIRST) {
        // Caller data may hold NaN / Inf in the Dirichlet rows (R5: "ignored"): those values are selected to 0 here, once,
        // and only in the cells that touch the box surface (s_g = 0 nowhere else; the branch is uniform over the CTA), so
        // the interior cells run exactly the arithmetic of the later steps.  (Selecting at every use cost 5 % of a FIRST
        // launch: 3 instructions per value against one DMUL.)
        if (ex == 0 || ey == 0 || ez == 0 || ex == prm.cx - 1 || ey == prm.cy - 1 || ez == prm.cz - 1) {
#pragma unroll
            for (int ay = 0; ay < n; ++ay)
#pragma unroll
                for (int ax = 0; ax < n; ++ax)
                    v[ay][ax] = (__double2hiint(sin_pl[ay * NP + ax]) != 0) ? v[ay][ax] : 0.0;
        }
    }
    if (early) {
        if (pl < P) {
            // compact p x p sub-planes: beta' X -> own plane of bufA (store to W), kappa X -> own plane of bufB (add to Y)
#pragma unroll
            for (int ay = 0; ay < P; ++ay)
#pragma unroll
                for (int ax = 0; ax < P; ++ax) {
                    const double x = v[ay][ax];
                    if (prm.preinit) pA[(ay * P + ax) * BT] = prm.beta_next * x;
                    if (prm.owner) pB[(ay * P + ax) * BT] = kappa * x;
                    if (DOTS) dacc = fma(kappa * x, x, dacc);
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
    // a1: xhat = mu_g s_g x (the Dirichlet rows of caller data are already 0)
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
        if (PERSIST) {  // this warp no longer needs A: when all warps say so, bufA can take the next unit's X
            __syncwarp();
            if ((tid & 31) == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar + 1)) : "memory");
        }
        if constexpr (!DOTS) {
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
        } else {
        // DOTS: U must still be in v when each part of T meets it, so N'z A2 comes first and is parked in the lines of the A2
        // field it was read from (this thread's own lines), then T = VZ . U + G'z U + (kx/kz) N'z A2 with U^T T on the way
        double dq = 0.0, ds = 0.0;
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int az = 0; az < n; ++az) t[az] = lb[((az * n + qy) * n) * BT];
            mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) {
                dq = fma(v[qy][qz], o[qz], dq);
                lb[((qz * n + qy) * n) * BT] = o[qz];
            }
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoG, v[qy], o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) {
                const double tn = fma(lv[qy * NP + qz], v[qy][qz], o[qz]);
                ds = fma(v[qy][qz], tn, ds);
                v[qy][qz] = fma(rxz, lb[((qz * n + qy) * n) * BT], tn);
            }
        }
        dacc = fma(rec[TAIL + 2], fma(rxz, dq, ds), dacc);  // x^T y_e = kz U^T T
        }
        // next-tile request, between passes 3 and 4 (measured: after pass 2 -0.7 %, after pass 4 -8 %: the tile must be
        // in flight for about a third of the unit).  The producer duty sits on warp 3: with 32-wide tiles warps map
        // 0,4 / 1,5 / 2,6 / 3 onto the four sub-partitions, so warp 3 is the one with issue slots to spare (measured
        // +1.2 % over thread 0)
        if (PERSIST && tid == (n > 3 ? 3 * BT : 0) && u + gridDim.x < nunits) {
            const long long un = u + gridDim.x;
            int nx, ny, nz;
            walk_cell((int)(un / nbt), prm.cx, prm.cy, prm.blk, nx, ny, nz);
            const int cn = nx + prm.cx * (ny + prm.cy * nz);
            mbar_wait(bar + 1, parity ^ 1);  // parity was flipped after this unit's tile wait
            mbar_expect_tx(bar, (unsigned)((n3 * BT + REC) * sizeof(double)));
            tma_load4(bufA, &prm.mXn, (int)(un % nbt) * BT, nx * P, ny * P, nz * P, bar);
            bulk_load(recN, prm.rec + (size_t)cn * RECG, (unsigned)(REC * sizeof(double)), bar);
        }
        // pass 4: R = N'z^T T, into the lines of the A2 field this thread has just consumed
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoNT, v[qy], o);
#pragma unroll
            for (int az = 0; az < n; ++az) lb[((az * n + qy) * n) * BT] = o[az];
        }
    }
    __syncthreads();
    // ---- plane phase 2: back-interpolate in y and x, scale by alpha kz s_g, two bulk reduce-adds per nodal plane --------
#pragma unroll
    for (int qy = 0; qy < n; ++qy)
#pragma unroll
        for (int qx = 0; qx < n; ++qx) v[qy][qx] = pB[(qy * n + qx) * BT];
#pragma unroll
    for (int qx = 0; qx < n; ++qx) {
#pragma unroll
        for (int q = 0; q < n; ++q) t[q] = v[q][qx];
        mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
        for (int a = 0; a < n; ++a) v[a][qx] = o[a];
    }
    const double* sout_pl = sOut + pl * n * NP;
    constexpr int H1 = (n + 1) / 2;  // the plane leaves in two bulk reduce-adds: the first overlaps the remaining rows
    double* pC = STG ? bufC + (size_t)pl * CPL + lane - (size_t)H1 * n * BT : pB;  // rows ay >= H1 (staged: a tile of their own)
    if (STG) {  // the previous unit's last reduce-add (a whole unit ago) has read the staging tile
        if (lane == 0) bulk_wait_read0();
        __syncwarp();
    }
#pragma unroll
    for (int ay = 0; ay < n; ++ay) {
        mat1d_eo<n>(prm.eoNTa, v[ay], o);
        double* dst = ay < H1 ? pB : pC;
#pragma unroll
        for (int ax = 0; ax < n; ++ax)
            dst[(ay * n + ax) * BT] = (SLIM ? kzs * sout_pl[ay * NP + ax] : sout_pl[ay * NP + ax]) * o[ax];
        if (ay == H1 - 1 && H1 < n) {
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                tma_reduce_add4(&prm.mYh1, pB, j0, gx0, gy0, gz0 + pl);
                bulk_commit();
            }
        }
    }
    fence_async_smem();
    __syncwarp();
    if (lane == 0) {
        if (H1 < n)
            tma_reduce_add4(&prm.mYh2, pC + (size_t)H1 * n * BT, j0, gx0, gy0 + H1, gz0 + pl);
        else
            tma_reduce_add4(&prm.mYh1, pB, j0, gx0, gy0, gz0 + pl);
        bulk_commit();
    }
    if constexpr (DOTS) {
        red[pl * BT + lane] = dacc;
        __syncthreads();
        if (pl == 0 && j0 + lane < prm.B) {
            double sum = red[lane];
#pragma unroll
            for (int k = 1; k < n; ++k) sum += red[k * BT + lane];
            atomicAdd(prm.dots + j0 + lane, sum);
        }
    }
    if (!PERSIST) break;
    double* tmp = rec; rec = recN; recN = tmp;
    }  // units
    if (lane == 0) bulk_wait_read0();  // shared memory must stay valid until the bulk engine has read it
}

// ctas > 0: persistent launch with that many CTAs (each walks units blockIdx.x, +ctas, ...); 0: one CTA per unit
template <int P, int BT, int MINB>
cudaError_t launch_tma(const TmaParams& prm, long long ncells, bool first, cudaStream_t st, int ctas)
{
    constexpr int n = P + 1;
    constexpr size_t smem = tma_smem_bytes<P, BT>(), smem_d = tma_smem_bytes<P, BT, false, true>();
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        cudaError_t e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return e;
    });
    if (e0 != cudaSuccess) return e0;
    const long long nunits = ncells * ((prm.B + BT - 1) / BT);
    const bool persist = ctas > 0 && (long long)ctas * MINB < nunits;
    dim3 grid((unsigned)(persist ? (long long)ctas * MINB : nunits)), block(BT, n);
    if (prm.dots) {  // plain apply on caller data with the column-wise dots: FIRST kernels only
        if (!first) return cudaErrorInvalidValue;
        static PerDeviceOnce once_d;
        cudaError_t ed = once_per_device(once_d, [&] {
            cudaError_t e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_d);
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_d);
            return e;
        });
        if (ed != cudaSuccess) return ed;
        if (persist)
            k_apply_tma<P, BT, MINB, true, true, true><<<grid, block, smem_d, st>>>(prm);
        else
            k_apply_tma<P, BT, MINB, true, false, true><<<grid, block, smem_d, st>>>(prm);
        return cudaGetLastError();
    }
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

// one SLIM CTA per unit (p = 5)
template <int P, int BT, int MINB>
cudaError_t launch_tma_slim(const TmaParams& prm, long long ncells, bool first, cudaStream_t st)
{
    constexpr int n = P + 1;
    constexpr size_t smem = tma_smem_bytes<P, BT, true>();
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        cudaError_t e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, true, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k_apply_tma<P, BT, MINB, false, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        return e;
    });
    if (e0 != cudaSuccess) return e0;
    dim3 grid((unsigned)(ncells * ((prm.B + BT - 1) / BT))), block(BT, n);
    if (first)
        k_apply_tma<P, BT, MINB, true, false, false, true><<<grid, block, smem, st>>>(prm);
    else
        k_apply_tma<P, BT, MINB, false, false, false, true><<<grid, block, smem, st>>>(prm);
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
    // default: persistent wherever only one CTA fits an SM (p = 5, 7, 8 and the 32-wide p = 6 shape): nothing else
    // would hide the tile latency there; with several CTAs per SM one CTA per unit measured faster (p <= 4)
    const bool one_cta = wide6 || p == 5 || p >= 7;
    if (!(variant == 7 || variant == 8 || (variant == 0 && one_cta))) sms = 0;
    if (wide6) return launch_tma<6, 32, 1>(prm, ncells, first, st, sms);
    // p = 5 default: two one-unit SLIM CTAs per SM (variant 7 keeps the persistent CTA; the dots need the full kernel)
    if (p == 5 && variant == 0 && !prm.dots) return launch_tma_slim<5, 32, 2>(prm, ncells, first, st);
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

// the mesh-dependent part of the cell records: s_g and kz s_g at the cell's nodes, ky/kx and kx/kz (VZ is written by
// k_weight_potential); sx, sy, sz = per-axis mu M^{-1/2}, hx, hy, hz = per-axis cell sizes
__global__ void k_build_records(double* __restrict__ rec, int n, int cx, int cy, long long ncells,
                                const double* __restrict__ sx, const double* __restrict__ sy,
                                const double* __restrict__ sz, const double* __restrict__ hx,
                                const double* __restrict__ hy, const double* __restrict__ hz)
{
    const int NP = n + (n & 1), SMALL = n * n * NP, REC = 3 * SMALL + 8, p = n - 1;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ncells * SMALL; i += (long long)gridDim.x * blockDim.x) {
        const long long e = i / SMALL;
        const int k = (int)(i - e * SMALL), ax = k % NP, ay = (k / NP) % n, az = k / (NP * n);
        const int ex = (int)(e % cx), ey = (int)((e / cx) % cy), ez = (int)(e / ((long long)cx * cy));
        const double s = ax < n ? sx[ex * p + ax] * sy[ey * p + ay] * sz[ez * p + az] : 0.0;
        const double kz = 0.25 * hx[ex] * hy[ey] / hz[ez];  // 2J/hz^2, J = hx hy hz / 8
        double* r = rec + e * REC;
        r[SMALL + k] = s;
        r[2 * SMALL + 8 + k] = kz * s;
        if (k < 8) r[2 * SMALL + k] = k == 0 ? (hx[ex] * hx[ex]) / (hy[ey] * hy[ey]) : k == 1 ? (hz[ez] * hz[ez]) / (hx[ex] * hx[ex]) : k == 2 ? kz : 0.0;
    }
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
