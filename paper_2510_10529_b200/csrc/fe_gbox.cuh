// fe_gbox.cuh -- the fused operator step on a general mesh (explicit l2g, hanging nodes) whose cells are all AXIS-ALIGNED
// BOXES: the leaves of an octree refinement of a box, the shape of the paper's adaptive meshes (Fig. 6).
//
// On such a cell the metric of Eq. 17 (l.171) is diagonal and constant, so the kinetic term separates and the cell
// contraction is the 10-sweep, plane-in-registers form of the box-mesh kernel (fe_apply_tma.cuh: A = N'y N'x xhat,
// A2 = G'x A + (ky/kx) G'y A per nodal plane; U = N'z A, T = VZ.U + G'z U + (kx/kz) N'z A2, R = N'z^T T per line;
// yhat / kz = N'x^T N'y^T R per nodal plane) instead of the generic 12 sweeps over shared-memory lines of k_apply_gen
// (fe_general.cuh).  What differs from the box-mesh kernel is the data movement: a refined mesh is no tensor, so
//   gather  : every thread copies the n x n rows of ITS nodal plane through the explicit l2g (8-byte cp.async into the field
//             it will read itself; unconstrained nodes from X, hanging nodes from the expanded values X_h = C_h (s . X));
//             the copies of the next unit are issued when the line phase has released the field, and run under plane phase 2;
//   scatter : red.global.add.f64 per value into Y (unconstrained) or Y_h (hanging; k_gen_collapse distributes it);
//   record  : one bulk copy per unit brings V_q hz^2/2, the gather and scatter scales, the cell's ratios and its n^3 ids.
// The diagonal terms of the step (shift, recurrence) come from the owner cell of each node as in the box-mesh kernel (store of
// beta' X into the next target, kappa_j X added to Y), so a filter step reads no Y_{k-1} and needs no k_gen_init pass; callers
// that pass a Z block, and the colour-ordered mode, keep k_gen_init.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "fe_apply_tma.cuh"
#include "fe_kernels.cuh"

namespace fecheb {

// per-cell record: VZ [qx][qy][NP] | s [az][ay][NP] (gather scale: s_g, 1 at hanging nodes) | tail (8) | kz s [az][ay][NP]
// | ids (n^3 int32, padded to a multiple of 4; bit 31 set where this cell is the OWNER of the node: the first cell that lists
// it).  tail = { ky/kx, kx/kz, kz, hz^2/2, 1 if a node of the cell is a Dirichlet
// node, 0, 0, 0 }
template <int n>
struct GBoxShape {
    static constexpr int NP = n + (n & 1), SMALL = n * n * NP, N3P = (n * n * n + 3) & ~3;
    static constexpr int TAIL = 2 * SMALL, SOUT = 2 * SMALL + 8, IDS = 3 * SMALL + 8;
    static constexpr int REC = IDS + N3P / 2;  // doubles (even: every piece is)
};
__host__ __device__ inline int gbox_rec_doubles(int n) { const int NP = n + (n & 1); return 3 * n * n * NP + 8 + (((n * n * n + 3) & ~3) / 2); }

struct GBoxParams {
    const double* X;     // N * B
    const double* Xh;    // (N_all - N) * B: expanded hanging values
    double* Y;           // N * B, holds the diagonal terms (k_gen_init)
    double* Yh;          // (N_all - N) * B, zero on entry
    const double* rec;   // ncells * REC
    const int32_t* cell_list;  // NULL: all cells; else the cells of one colour (colour-ordered scatter)
    long long N, ncells;
    int B;
    EOTab eoN, eoNT, eoG;  // even-odd halves of N' = diag(sqrt w) N, N'^T, G' = diag(w^-1/2) G diag(w^-1/2)
    EOTab eoNTa;           // alpha N'^T: unconstrained AND hanging targets receive alpha yhat (the collapse then runs with 1)
    // diagonal terms from the OWNER cell of every unconstrained node (the first cell that lists it; bit 31 of its id in that
    // cell's record), as in the box-mesh kernel: Y += kappa_j X with kappa_j = -alpha (c + eps_j) when `owner`, and the
    // pre-initialisation W = beta_next X of the NEXT filter step's target when W != NULL (no k_gen_init pass, no read of Y_{k-1})
    double* W;
    const double* eps;
    double alpha, c, beta_next;
    int owner;
};

// VZ tile of every record from the caller's V[e][q], q = qx + n (qy + n qz)
__global__ void k_gbox_weight_potential(double* __restrict__ rec, const double* __restrict__ V, long long ncells, int n)
{
    const int NP = n + (n & 1), n3 = n * n * n, REC = gbox_rec_doubles(n), TAIL = 2 * n * n * NP;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ncells * n3; i += (long long)gridDim.x * blockDim.x) {
        const long long e = i / n3;
        const int q = (int)(i - e * n3), qx = q % n, qy = (q / n) % n, qz = q / (n * n);
        rec[e * REC + (qx * n + qy) * NP + qz] = rec[e * REC + TAIL + 3] * V[i];
    }
}

// SLIM (p = 5): ONE record buffer without the kz s tile (the output scale is kz times the gather scale), one unit per CTA, so that
// two 6-warp CTAs fit an SM (12 warps, three per sub-partition) instead of one persistent CTA whose warps sit 2,2,1,1
template <int P, int BT, bool SLIM = false>
constexpr size_t gbox_smem_bytes()
{
    constexpr int n = P + 1;
    constexpr int recs = SLIM ? GBoxShape<n>::SOUT + GBoxShape<n>::N3P / 2 : 2 * GBoxShape<n>::REC;
    return ((size_t)2 * n * n * n * BT + recs) * sizeof(double) + 16;
}

// Block (BT lanes = vectors, n nodal planes).  A CTA walks units (cell, tile of BT vectors) u = blockIdx.x, + gridDim.x, ...
template <int P, int BT, int MINB, bool SLIM = false>
__global__ void __launch_bounds__((P + 1) * BT, MINB) k_apply_gbox(const __grid_constant__ GBoxParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n, NP = GBoxShape<n>::NP, SMALL = GBoxShape<n>::SMALL,
                  RECG = GBoxShape<n>::REC, TAIL = GBoxShape<n>::TAIL, IDSG = GBoxShape<n>::IDS, NID = GBoxShape<n>::N3P / 2,
                  // shared-memory record: SLIM keeps VZ | s | tail | ids (the ids move up into the place of the kz s tile)
                  REC = SLIM ? GBoxShape<n>::SOUT + NID : RECG, SOUT = SLIM ? SMALL : GBoxShape<n>::SOUT,
                  IDS = SLIM ? GBoxShape<n>::SOUT : IDSG;
    extern __shared__ __align__(128) double smem[];
    double* bufA = smem;               // [n^3][BT]  gathered X -> A (free once the line phase is over) -> next unit's X
    double* bufB = smem + n3 * BT;     // [n^3][BT]  A2 -> R
    double* recs = bufB + n3 * BT;     // [2][REC] (SLIM: one)
    unsigned long long* bar = (unsigned long long*)(recs + (SLIM ? 1 : 2) * REC);  // bar[b]: record b landed
    const int lane = threadIdx.x, pl = threadIdx.y, tid = pl * BT + lane;
    const int nbt = (prm.B + BT - 1) / BT;
    const long long nunits = prm.ncells * nbt;

    auto request_rec = [&](long long u, int b) {  // one thread
        const long long cu = u / nbt, c = prm.cell_list ? (long long)prm.cell_list[cu] : cu;
        mbar_expect_tx(bar + b, (unsigned)(REC * sizeof(double)));
        if constexpr (SLIM) {  // two pieces of the global record: VZ | s | tail, and the ids
            bulk_load(recs, prm.rec + c * RECG, (unsigned)(IDS * sizeof(double)), bar + b);
            bulk_load(recs + IDS, prm.rec + c * RECG + IDSG, (unsigned)(NID * sizeof(double)), bar + b);
        } else {
            bulk_load(recs + b * REC, prm.rec + c * RECG, (unsigned)(REC * sizeof(double)), bar + b);
        }
    };
    // Addresses in 32-bit pieces: ids and N fit 32 bits (int32 l2g), so the row of node g starts at base + g * (8 B) bytes with
    // ONE wide multiply-add, base = X (unconstrained) or X_h - N * 8 B (hanging: g - N is its row of X_h).  (The plain 64-bit
    // form g * B + j with a two-way pointer select cost ~25 integer instructions per node and direction: ncu, 56 % of the
    // kernel's instructions were not FP64.)
    const unsigned N32 = (unsigned)prm.N, B8 = (unsigned)prm.B * 8u;
    const unsigned long long hoff = (unsigned long long)N32 * B8;
    // the rows of this thread's nodal plane, straight into the plane of bufA it reads itself (no CTA barrier in between)
    auto request_rows = [&](long long u, int b) {
        const int32_t* ids = reinterpret_cast<const int32_t*>(recs + b * REC + IDS) + pl * n2;
        const int j = (int)(u % nbt) * BT + lane;
        const bool act = j < prm.B;
        const char* bX = reinterpret_cast<const char*>(prm.X + (act ? j : 0));
        const char* bH = reinterpret_cast<const char*>(prm.Xh + (act ? j : 0)) - hoff;
        const unsigned d0 = smem_u32(bufA + (size_t)pl * n2 * BT + lane);
        const int sz = act ? 8 : 0;  // src-size 0 zero-fills the 8 destination bytes
#pragma unroll
        for (int a = 0; a < n2; ++a) {
            const unsigned g = (unsigned)ids[a] & 0x7fffffffu;
            const char* src = (g < N32 ? bX : bH) + (unsigned long long)g * B8;
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d0 + (unsigned)(a * BT * 8)), "l"(src), "r"(sz) : "memory");
        }
        cp_async_commit();
    };

    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 1, 1);
    }
    __syncthreads();
    unsigned ph0 = 0, ph1 = 0;
    if ((long long)blockIdx.x < nunits) {
        if (tid == 0) request_rec(blockIdx.x, 0);
        mbar_wait(bar, ph0);
        ph0 ^= 1;
        request_rows(blockIdx.x, 0);
    }
    int buf = 0;
    for (long long u = blockIdx.x; u < nunits; u += gridDim.x, buf ^= 1) {
    const long long un = u + gridDim.x;
    const bool more = !SLIM && un < nunits;  // SLIM: one unit per CTA (the launch gives every unit its own)
    const int j = (int)(u % nbt) * BT + lane;
    const bool act = j < prm.B;
    const double* rec = recs + buf * REC;
    const double* sVZ = rec;
    const double ry = rec[TAIL], rxz = rec[TAIL + 1];
    const bool surface = rec[TAIL + 4] != 0.0;
    const double kzs = SLIM ? rec[TAIL + 2] : 1.0;  // SLIM: output scale = kz times the gather scale

    double v[n][n], t[n], o[n];
    double* pA = bufA + (size_t)pl * n2 * BT + lane;
    double* pB = bufB + (size_t)pl * n2 * BT + lane;
    const double* sin_pl = rec + SMALL + pl * n * NP;
    cp_async_wait_all();  // this thread's own copies: the plane it reads now
    // ---- plane phase 1 -----------------------------------------------------------------------------------------------
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) v[ay][ax] = pA[(ay * n + ax) * BT];
    if (surface) {  // Dirichlet rows of caller data are ignored (R5), whatever they hold; uniform over the CTA
#pragma unroll
        for (int ay = 0; ay < n; ++ay)
#pragma unroll
            for (int ax = 0; ax < n; ++ax)
                v[ay][ax] = (__double2hiint(sin_pl[ay * NP + ax]) != 0) ? v[ay][ax] : 0.0;
    }
    if (prm.W != nullptr || prm.owner) {  // uniform over the grid
        // The store is predicated (owner cells only); the add is UNCONDITIONAL with the value selected to 0 elsewhere: ptxas
        // turns a predicated red.global into a branch with uniform-register spills around it (11 instructions per node).
        const int32_t* idp = reinterpret_cast<const int32_t*>(rec + IDS) + pl * n2;
        const int jj = act ? j : 0;
        char* wX = reinterpret_cast<char*>(prm.W + jj);
        char* aX = reinterpret_cast<char*>(prm.Y + jj);
        char* aH = reinterpret_cast<char*>(prm.Yh + jj) - hoff;
        const double kappa = (prm.owner && act) ? -prm.alpha * (prm.c + (prm.eps ? prm.eps[j] : 0.0)) : 0.0;
        const double bnext = prm.beta_next;
        const bool has_w = prm.W != nullptr;
#pragma unroll
        for (int ay = 0; ay < n; ++ay)
#pragma unroll
            for (int ax = 0; ax < n; ++ax) {
                const int enc = idp[ay * n + ax];
                const unsigned g = (unsigned)enc & 0x7fffffffu;
                const bool own = act && enc < 0;
                const double x = v[ay][ax];
                if (own && has_w) *reinterpret_cast<double*>(wX + (unsigned long long)g * B8) = bnext * x;
                // nodes this cell does not own receive +0.0 at their own address (hanging nodes, never owned, in Y_h): spread
                // over the block like the real adds, no hot spot
                atomicAdd(reinterpret_cast<double*>((g < N32 ? aX : aH) + (unsigned long long)g * B8), own ? kappa * x : 0.0);
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
    if constexpr (n >= 7) {
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
    // every thread is past the previous unit: its record buffer can take the next unit's record (needed at plane phase 2)
    if (more && tid == 0) request_rec(un, buf ^ 1);
    // ---- line phase: the thread owns the yz-plane qx = pl ----------------------------------------------------------------
    {
        double* la = bufA + (size_t)pl * BT + lane;
        double* lb = bufB + (size_t)pl * BT + lane;
        const double* lv = sVZ + pl * n * NP;
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int az = 0; az < n; ++az) t[az] = la[((az * n + qy) * n) * BT];
            mat1d_eo<n>(prm.eoN, t, v[qy]);
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoG, v[qy], o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) v[qy][qz] = fma(lv[qy * NP + qz], v[qy][qz], o[qz]);
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
#pragma unroll
            for (int az = 0; az < n; ++az) t[az] = lb[((az * n + qy) * n) * BT];
            mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
            for (int qz = 0; qz < n; ++qz) v[qy][qz] = fma(rxz, o[qz], v[qy][qz]);
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoNT, v[qy], o);
#pragma unroll
            for (int az = 0; az < n; ++az) lb[((az * n + qy) * n) * BT] = o[az];
        }
    }
    __syncthreads();
    // bufA is free: the next unit's rows travel while this unit is back-interpolated and scattered
    if (more) {
        if (buf == 0) { mbar_wait(bar + 1, ph1); ph1 ^= 1; } else { mbar_wait(bar, ph0); ph0 ^= 1; }
        request_rows(un, buf ^ 1);
    }
    // ---- plane phase 2: back-interpolate in y and x, scale by alpha kz s, scatter through the l2g -------------------------------
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
    const double* sout_pl = rec + SOUT + pl * n * NP;
    const int32_t* ids = reinterpret_cast<const int32_t*>(rec + IDS) + pl * n2;
    char* yX = reinterpret_cast<char*>(prm.Y + (act ? j : 0));
    char* yH = reinterpret_cast<char*>(prm.Yh + (act ? j : 0)) - hoff;
#pragma unroll
    for (int ay = 0; ay < n; ++ay) {
        mat1d_eo<n>(prm.eoNTa, v[ay], o);
#pragma unroll
        for (int ax = 0; ax < n; ++ax) {
            const double sc = sout_pl[ay * NP + ax];
            const unsigned g = (unsigned)ids[ay * n + ax] & 0x7fffffffu;
            char* dst = (g < N32 ? yX : yH) + (unsigned long long)g * B8;
            // unconditional add (a predicated red.global becomes a branch): Dirichlet nodes (scale 0) and idle lanes (column 0
            // of their node) add +0.0, which changes nothing
            atomicAdd(reinterpret_cast<double*>(dst), (act && __double2hiint(sc) != 0) ? (SLIM ? kzs * sc : sc) * o[ax] : 0.0);
        }
    }
    }  // units
}

template <int P, int BT, int MINB, bool SLIM = false>
cudaError_t launch_gbox_t(const GBoxParams& prm, long long ncells, int sms, cudaStream_t st)
{
    constexpr size_t smem = gbox_smem_bytes<P, BT, SLIM>();
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_apply_gbox<P, BT, MINB, SLIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    const long long nunits = ncells * ((prm.B + BT - 1) / BT);
    if (nunits <= 0) return cudaSuccess;
    dim3 grid((unsigned)(SLIM ? nunits : std::min<long long>(nunits, (long long)sms * MINB))), block(BT, P + 1);
    k_apply_gbox<P, BT, MINB, SLIM><<<grid, block, smem, st>>>(prm);
    return cudaGetLastError();
}

inline bool gbox_supported(int p) { return p >= 1 && p <= 7; }

inline cudaError_t launch_apply_gbox(const GBoxParams& prm, int p, long long ncells, int sms, cudaStream_t st)
{
    switch (p) {
        case 1: return launch_gbox_t<1, 32, 8>(prm, ncells, sms, st);
        case 2: return launch_gbox_t<2, 32, 6>(prm, ncells, sms, st);
        case 3: return launch_gbox_t<3, 32, 4>(prm, ncells, sms, st);
        case 4: return launch_gbox_t<4, 32, 3>(prm, ncells, sms, st);
        case 5: return launch_gbox_t<5, 32, 2, true>(prm, ncells, sms, st);  // two one-unit SLIM CTAs per SM: 48.8 -> 56.4 GDoF-vec/s
        case 6: return launch_gbox_t<6, 32, 1>(prm, ncells, sms, st);
        case 7: return launch_gbox_t<7, 24, 1>(prm, ncells, sms, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace fecheb
