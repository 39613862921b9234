// fe_minres.cuh -- block preconditioned MINRES around the shifted apply (NEXT-2; Eq. 20 l.183)
//
// Every column j solves its own system (H~ - eps_j I) p_j = g_j with its own Paige-Saunders recurrences; the
// columns advance in lock-step so that each Krylov step is ONE fused fe_apply_H launch for the whole block.  The
// normalised Lanczos vector v = y / beta is never stored: the apply runs on y and the scale is folded into what follows.
// The operator kernel itself delivers the column-wise dots y_j . (H~ - eps_j) y_j from cell-local terms (fe_apply_tma.cuh,
// DOTS), so alfa_j is known right after the apply and the two Lanczos vector updates are ONE elementwise pass
// (k_minres_lanczos: also beta_j^2 = r_j . M^{-1} r_j and the y . r1 of the next step); a second pass updates w and x and
// clears the next apply target.  The Givens / Lanczos scalars live in device arrays of length B and are advanced by a
// one-block kernel, so an iteration needs no host synchronisation.
// Preconditioner (l.225): inverse diagonal of the mass-scaled negative Laplacian, positive on free rows.
#pragma once
#include <cuda_runtime.h>

namespace fecheb {

struct MinresScalars {  // B doubles each, device
    double *beta, *oldb, *alfa, *betasq, *dbar, *epsln, *oldeps, *phibar, *cs, *sn, *gamma, *delta, *phi, *beta1;
    double *s, *c1, *c2;  // 1/beta, beta/oldb, alfa/beta of the running step
    double *dot, *gam, *gamn;  // y.(H~-eps)y from the operator kernel; y.r1 of this step and of the next
    double* sv;                // s of the step whose w / x update is still to run (stage 2 moves on to the next step's s)
};

constexpr int kMRx = 32, kMRy = 8, kMaxColTiles = 4;  // B <= 128

// column-wise partial sums of a thread block -> atomicAdd into out[j]
__device__ __forceinline__ void block_col_reduce(double (&acc)[kMaxColTiles], int B, double* out)
{
    __shared__ double red[kMRy][kMRx];
#pragma unroll
    for (int t = 0; t < kMaxColTiles; ++t) {
        const int j = t * kMRx + threadIdx.x;
        if (t * kMRx >= B) break;
        red[threadIdx.y][threadIdx.x] = acc[t];
        __syncthreads();
        if (threadIdx.y == 0 && j < B) {
            double sum = 0.0;
#pragma unroll
            for (int y = 0; y < kMRy; ++y) sum += red[y][threadIdx.x];
            atomicAdd(out + j, sum);
        }
        __syncthreads();
    }
}

// phase 0 (start):  r1 = r2 = g (masked); y = Minv r; betasq = r.y; x = w = w2 = 0
__global__ void k_minres_init(const double* __restrict__ G, const double* __restrict__ Minv, double* __restrict__ R1,
                              double* __restrict__ R2, double* __restrict__ Y, double* __restrict__ X,
                              double* __restrict__ W, double* __restrict__ W2, long long N, int B, double* betasq)
{
    double acc[kMaxColTiles] = {0, 0, 0, 0};
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += (long long)gridDim.x * kMRy) {
        const double mi = Minv[r];
#pragma unroll
        for (int t = 0; t < kMaxColTiles; ++t) {
            const int j = t * kMRx + threadIdx.x;
            if (j < B) {
                const long long i = r * B + j;
                const double g = mi != 0.0 ? G[i] : 0.0;  // Dirichlet rows do not take part (R5)
                const double y = mi * g;
                R1[i] = g; R2[i] = g; Y[i] = y; X[i] = 0.0; W[i] = 0.0; W2[i] = 0.0;
                acc[t] = fma(g, y, acc[t]);
            }
        }
    }
    block_col_reduce(acc, B, betasq);
}

// column-wise x . y of two blocks (the fallback when the operator kernel cannot deliver the dots itself)
__global__ void k_col_dot(const double* __restrict__ X, const double* __restrict__ Y, long long N, int B, double* out)
{
    double acc[kMaxColTiles] = {0, 0, 0, 0};
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += (long long)gridDim.x * kMRy)
#pragma unroll
        for (int t = 0; t < kMaxColTiles; ++t) {
            const int j = t * kMRx + threadIdx.x;
            if (j < B) acc[t] = fma(X[r * B + j], Y[r * B + j], acc[t]);
        }
    block_col_reduce(acc, B, out);
}

// phases B + C in one pass.  The apply ran on the un-normalised y (= beta v): hy = (H~ - eps) y, and alfa_j = v_j . y'_j with
// y' = s_j hy - c1_j r1 is already known from the dots of the operator kernel (k_minres_scalars stage 3), so
//   t = s_j hy - c1_j r1 - c2_j r2 ;  r1 <- t (the host swaps r1 / r2 afterwards) ;  y_next = Minv t (into hy's block) ;
//   betasq_j = t_j . y_next,j ;  gamn_j = y_next,j . r2_j  (the y . r1 of the NEXT step, whose r1 is this r2)
__global__ void k_minres_lanczos(double* __restrict__ HY, double* __restrict__ R1, const double* __restrict__ R2,
                                 const double* __restrict__ Minv, long long N, int B, const double* __restrict__ s,
                                 const double* __restrict__ c1, const double* __restrict__ c2, double* betasq, double* gamn)
{
    double acc[kMaxColTiles] = {0, 0, 0, 0}, acg[kMaxColTiles] = {0, 0, 0, 0};
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += (long long)gridDim.x * kMRy) {
        const double mi = Minv[r];
#pragma unroll
        for (int t = 0; t < kMaxColTiles; ++t) {
            const int j = t * kMRx + threadIdx.x;
            if (j < B) {
                const long long i = r * B + j;
                const double r2 = R2[i];
                const double yp = fma(s[j], HY[i], -c1[j] * R1[i]);
                const double tt = fma(-c2[j], r2, yp);
                const double y = mi * tt;
                R1[i] = tt;
                HY[i] = y;
                acc[t] = fma(tt, y, acc[t]);
                acg[t] = fma(y, r2, acg[t]);
            }
        }
    }
    block_col_reduce(acc, B, betasq);
    block_col_reduce(acg, B, gamn);
}

// phase D:  w_new = (v - oldeps_j w1 - delta_j w2) / gamma_j  (into w1's storage), v = s_j y_old ;  x += phi_j w_new.
// y_old is read here for the last time and its block is the NEXT step's apply target: it is cleared on the way out, which
// replaces the zero-fill pass of fe_apply_H.
__global__ void k_minres_update(double* __restrict__ Yold, double* __restrict__ W1, const double* __restrict__ W2,
                                double* __restrict__ X, long long N, int B, const double* __restrict__ s,
                                const double* __restrict__ oldeps, const double* __restrict__ delta,
                                const double* __restrict__ gamma, const double* __restrict__ phi)
{
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += (long long)gridDim.x * kMRy)
#pragma unroll
        for (int t = 0; t < kMaxColTiles; ++t) {
            const int j = t * kMRx + threadIdx.x;
            if (j < B) {
                const long long i = r * B + j;
                const double w = (s[j] * Yold[i] - oldeps[j] * W1[i] - delta[j] * W2[i]) / gamma[j];
                Yold[i] = 0.0;
                W1[i] = w;
                X[i] = fma(phi[j], w, X[i]);
            }
        }
}

// ---- 16-byte variants of the two passes (even B, 16-byte aligned blocks): a lane owns the adjacent columns 2(32t + lane) + {0, 1}
// and a thread moves two rows per trip, so every pass keeps 2 x 3..4 independent 16-byte loads per thread in flight (the 8-byte
// kernels above reach 4.0 - 4.7 TB/s of the 6.5 TB/s stream rate, ncu).  Same arithmetic, same order within a column.
// VT = tiles of 64 columns (1 for B <= 64, 2 for B <= 128), ROWS = rows per trip; 64 registers per thread keep four blocks per SM

template <int VT>
__device__ __forceinline__ void block_col_reduce2(const double2 (&acc)[VT], int B, double* out)
{
    __shared__ double red2[kMRy][2 * kMRx];
    const int tid = threadIdx.y * kMRx + threadIdx.x;
#pragma unroll
    for (int t = 0; t < VT; ++t) {
        if (t * 2 * kMRx >= B) break;
        red2[threadIdx.y][2 * threadIdx.x] = acc[t].x;
        red2[threadIdx.y][2 * threadIdx.x + 1] = acc[t].y;
        __syncthreads();
        if (tid < 2 * kMRx && t * 2 * kMRx + tid < B) {
            double sum = 0.0;
#pragma unroll
            for (int y = 0; y < kMRy; ++y) sum += red2[y][tid];
            atomicAdd(out + t * 2 * kMRx + tid, sum);
        }
        __syncthreads();
    }
}

__device__ __forceinline__ double2 ld2(const double* p, int jv, bool on)
{
    return on ? reinterpret_cast<const double2*>(p)[jv] : make_double2(0.0, 0.0);
}

template <int VT, int ROWS>
__global__ void __launch_bounds__(kMRx * kMRy, 3)
k_minres_lanczos2(double2* __restrict__ HY, double2* __restrict__ R1, const double2* __restrict__ R2,
                  const double* __restrict__ Minv, long long N, int B, const double* __restrict__ s,
                  const double* __restrict__ c1, const double* __restrict__ c2, double* betasq, double* gamn)
{
    const int Bh = B >> 1;
    bool on[VT];
    double2 sj[VT], c1j[VT], c2j[VT], acc[VT], acg[VT];
#pragma unroll
    for (int t = 0; t < VT; ++t) {
        const int jv = t * kMRx + threadIdx.x;
        on[t] = jv < Bh;
        sj[t] = ld2(s, jv, on[t]); c1j[t] = ld2(c1, jv, on[t]); c2j[t] = ld2(c2, jv, on[t]);
        acc[t] = make_double2(0.0, 0.0); acg[t] = make_double2(0.0, 0.0);
    }
    const long long step = (long long)gridDim.x * kMRy;
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += ROWS * step) {
        double2 hy[ROWS][VT], r1[ROWS][VT], r2[ROWS][VT];
        double mi[ROWS];
#pragma unroll
        for (int u = 0; u < ROWS; ++u) {
            const long long rr = r + u * step;
            if (rr < N) {
                mi[u] = Minv[rr];
#pragma unroll
                for (int t = 0; t < VT; ++t)
                    if (on[t]) {
                        const long long i = rr * Bh + t * kMRx + threadIdx.x;
                        hy[u][t] = HY[i]; r1[u][t] = R1[i]; r2[u][t] = R2[i];
                    }
            }
        }
#pragma unroll
        for (int u = 0; u < ROWS; ++u) {
            const long long rr = r + u * step;
            if (rr < N) {
#pragma unroll
                for (int t = 0; t < VT; ++t)
                    if (on[t]) {
                        const long long i = rr * Bh + t * kMRx + threadIdx.x;
                        double2 tt, y;
                        tt.x = fma(-c2j[t].x, r2[u][t].x, fma(sj[t].x, hy[u][t].x, -c1j[t].x * r1[u][t].x));
                        tt.y = fma(-c2j[t].y, r2[u][t].y, fma(sj[t].y, hy[u][t].y, -c1j[t].y * r1[u][t].y));
                        y.x = mi[u] * tt.x; y.y = mi[u] * tt.y;
                        R1[i] = tt; HY[i] = y;
                        acc[t].x = fma(tt.x, y.x, acc[t].x); acc[t].y = fma(tt.y, y.y, acc[t].y);
                        acg[t].x = fma(y.x, r2[u][t].x, acg[t].x); acg[t].y = fma(y.y, r2[u][t].y, acg[t].y);
                    }
            }
        }
    }
    block_col_reduce2<VT>(acc, B, betasq);
    block_col_reduce2<VT>(acg, B, gamn);
}

template <int VT, int ROWS>
__global__ void __launch_bounds__(kMRx * kMRy, 3)
k_minres_update2(double2* __restrict__ Yold, double2* __restrict__ W1, const double2* __restrict__ W2,
                 double2* __restrict__ X, long long N, int B, const double* __restrict__ s,
                 const double* __restrict__ oldeps, const double* __restrict__ delta,
                 const double* __restrict__ gamma, const double* __restrict__ phi)
{
    const int Bh = B >> 1;
    bool on[VT];
    double2 sj[VT], oe[VT], de[VT], ga[VT], ph[VT];
#pragma unroll
    for (int t = 0; t < VT; ++t) {
        const int jv = t * kMRx + threadIdx.x;
        on[t] = jv < Bh;
        sj[t] = ld2(s, jv, on[t]); oe[t] = ld2(oldeps, jv, on[t]); de[t] = ld2(delta, jv, on[t]);
        ga[t] = on[t] ? reinterpret_cast<const double2*>(gamma)[jv] : make_double2(1.0, 1.0);
        ga[t].x = 1.0 / ga[t].x; ga[t].y = 1.0 / ga[t].y;  // one division per column and thread, not one per element
        ph[t] = ld2(phi, jv, on[t]);
    }
    const long long step = (long long)gridDim.x * kMRy;
    for (long long r = blockIdx.x * (long long)kMRy + threadIdx.y; r < N; r += ROWS * step) {
        double2 yo[ROWS][VT], w1[ROWS][VT], w2[ROWS][VT], x[ROWS][VT];
#pragma unroll
        for (int u = 0; u < ROWS; ++u) {
            const long long rr = r + u * step;
            if (rr < N) {
#pragma unroll
                for (int t = 0; t < VT; ++t)
                    if (on[t]) {
                        const long long i = rr * Bh + t * kMRx + threadIdx.x;
                        yo[u][t] = Yold[i]; w1[u][t] = W1[i]; w2[u][t] = W2[i]; x[u][t] = X[i];
                    }
            }
        }
#pragma unroll
        for (int u = 0; u < ROWS; ++u) {
            const long long rr = r + u * step;
            if (rr < N) {
#pragma unroll
                for (int t = 0; t < VT; ++t)
                    if (on[t]) {
                        const long long i = rr * Bh + t * kMRx + threadIdx.x;
                        double2 w, xn;
                        w.x = (sj[t].x * yo[u][t].x - oe[t].x * w1[u][t].x - de[t].x * w2[u][t].x) * ga[t].x;
                        w.y = (sj[t].y * yo[u][t].y - oe[t].y * w1[u][t].y - de[t].y * w2[u][t].y) * ga[t].y;
                        xn.x = fma(ph[t].x, w.x, x[u][t].x); xn.y = fma(ph[t].y, w.y, x[u][t].y);
                        Yold[i] = make_double2(0.0, 0.0);
                        W1[i] = w;
                        X[i] = xn;
                    }
            }
        }
    }
}

// scalar recurrences, one thread per column.  stage 0: after init (beta1); stage 1: before the first step (s, c1); stage 3:
// after the apply (alfa, c2 from the operator kernel's dots); stage 2: after the Lanczos pass (beta, Givens rotation, phi), and
// straight on to the NEXT step's s, c1 (what stage 1 does), the finished step's s staying in sv for its w / x update
__global__ void k_minres_scalars(MinresScalars q, int B, int stage, double tol)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= B) return;
    if (stage == 0) {
        const double b1 = sqrt(fmax(q.betasq[j], 0.0));
        q.beta1[j] = b1; q.beta[j] = b1; q.oldb[j] = 0.0; q.dbar[j] = 0.0; q.epsln[j] = 0.0; q.phibar[j] = b1;
        q.cs[j] = -1.0; q.sn[j] = 0.0; q.betasq[j] = 0.0; q.alfa[j] = 0.0; q.gam[j] = 0.0; q.gamn[j] = 0.0; q.dot[j] = 0.0;
        q.gamma[j] = 1.0; q.delta[j] = 0.0; q.oldeps[j] = 0.0; q.phi[j] = 0.0; q.sv[j] = 0.0;
        return;
    }
    if (stage == 3) {  // after the apply: alfa = v . (s hy - c1 r1) = s^2 (y . hy) - c1 s (y . r1);  c2 = alfa / beta
        const double sj = q.s[j];
        const double alfa = sj * sj * q.dot[j] - q.c1[j] * sj * q.gam[j];
        q.alfa[j] = alfa;
        q.c2[j] = q.beta[j] > 0.0 ? alfa / q.beta[j] : 0.0;
        return;
    }
    if (stage == 2) {
        const bool live = q.s[j] != 0.0;
        q.sv[j] = q.s[j];
        q.gam[j] = q.gamn[j];
        const double alfa = q.alfa[j], oldb = q.beta[j];
        const double beta = sqrt(fmax(q.betasq[j], 0.0));
        if (!live) {
            q.phi[j] = 0.0; q.gamma[j] = 1.0; q.delta[j] = 0.0; q.oldeps[j] = 0.0;
        } else {
            const double cs = q.cs[j], sn = q.sn[j], dbar = q.dbar[j];
            const double oldeps = q.epsln[j];
            const double delta = cs * dbar + sn * alfa;
            const double gbar = sn * dbar - cs * alfa;
            const double epsln = sn * beta;
            const double dbar2 = -cs * beta;
            const double gamma = fmax(sqrt(gbar * gbar + beta * beta), 2.220446049250313e-16);
            const double cs2 = gbar / gamma, sn2 = beta / gamma;
            q.phi[j] = cs2 * q.phibar[j];
            q.phibar[j] = sn2 * q.phibar[j];
            q.oldeps[j] = oldeps; q.delta[j] = delta; q.gamma[j] = gamma; q.epsln[j] = epsln; q.dbar[j] = dbar2;
            q.cs[j] = cs2; q.sn[j] = sn2; q.oldb[j] = oldb; q.beta[j] = beta;
        }
    }
    // stage 1, and the tail of stage 2: the scalars of the step that starts now
    {
        const double beta = q.beta[j], oldb = q.oldb[j];
        const bool live = beta > 0.0 && q.phibar[j] > tol * q.beta1[j];  // a converged column stops moving
        q.s[j] = live ? 1.0 / beta : 0.0;
        q.c1[j] = (live && oldb > 0.0) ? beta / oldb : 0.0;
        q.alfa[j] = 0.0;
        q.betasq[j] = 0.0;
        q.dot[j] = 0.0;
        q.gamn[j] = 0.0;
    }
}

// Minv[g] = s_g^2 / diag(1/2 K)_g on free rows (0 on Dirichlet rows): inverse diagonal of the mass-scaled negative
// Laplacian, from per-axis diagonals: diag(1/2 K) = 1/2 (kx my mz + mx ky mz + mx my kz) with the Gauss-quadrature
// 1-D stiffness / mass diagonals k?, m?;  s? = per-axis mu M^{-1/2}
__global__ void k_build_precond(double* __restrict__ Minv, long long Nx, long long Ny, long long Nz,
                                const double* __restrict__ kx, const double* __restrict__ ky, const double* __restrict__ kz,
                                const double* __restrict__ mx, const double* __restrict__ my, const double* __restrict__ mz,
                                const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz)
{
    const long long total = Nx * Ny * Nz;
    for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < total; g += (long long)gridDim.x * blockDim.x) {
        const long long ix = g % Nx, iy = (g / Nx) % Ny, iz = g / (Nx * Ny);
        const double s = sx[ix] * sy[iy] * sz[iz];
        const double d = 0.5 * (kx[ix] * my[iy] * mz[iz] + mx[ix] * ky[iy] * mz[iz] + mx[ix] * my[iy] * kz[iz]);
        Minv[g] = s != 0.0 ? 1.0 / (s * s * d) : 0.0;
    }
}

}  // namespace fecheb
