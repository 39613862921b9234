// fe_kernels.cuh -- sm_100a kernels of the fused operator step
//
//   Y[g,j] = mu_g ( alpha ( s_g sum_{e∋g} y_e[a,j] - (c + eps_j) X[g,j] ) + beta Z[g,j] )
//
// with y_e = (1/2 K_e + M_{V,e}) (mu s X)_e evaluated matrix-free by sum factorisation (Eq. 17 l.171 on an
// axis-aligned cell; l.237 "cell-level dense-dense products", here never formed as matrices):
//
//   A  = (Ny Nx) x_e                                      per nodal z-plane        (interpolate to Gauss points in x,y)
//   A2 = kx wy (Gx A) + ky wx (Gy A)                      per nodal z-plane        (x,y stiffness in Gauss space)
//   U = Nz A, U2 = Nz A2                                  per (qx,qy) line
//   T = WV.U + wz.U2 + kz wx wy (Gz U),  R = Nz^T T       per (qx,qy) line
//   y_e = Nx^T Ny^T R                                     per nodal z-plane
//
// N[q][a] = l_a(xi_q) (Eq. 12), G = D~^T W D~ the 1-D stiffness on the Gauss points, WV = J w_q V_q,
// kd = 1/2 J (2/h_d)^2.  Lanes of a warp are consecutive VECTORS j (the layout of l.233-235 makes every global and
// shared access of a warp one contiguous 8*BT-byte row); a thread owns one z-plane (n x n values in registers) in
// the plane phases and n z-lines in the line phase, so 1-D matrix entries are warp-uniform constant-bank operands.
#pragma once
#include <cuda_runtime.h>

#include <atomic>

namespace fecheb {

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute and fe_mesh_create takes any cuda_device: every
// launcher keeps one bit per device (thread-safe) and sets the attribute on the first launch on each device.
struct PerDeviceOnce {
    std::atomic<unsigned long long> bits{0};
};
template <class F>
inline cudaError_t once_per_device(PerDeviceOnce& o, F&& set)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && ((o.bits.load(std::memory_order_acquire) >> dev) & 1ull)) return cudaSuccess;
    e = set();
    if (e == cudaSuccess && tracked) o.bits.fetch_or(1ull << dev, std::memory_order_release);
    return e;
}

// Even-odd form of a centro-symmetric n x n matrix M (M[i][k] = M[n-1-i][n-1-k]), h = n/2, c = (n+1)/2:
//   S[i*h+k] = (M[i][k] + M[i][n-1-k])/2 (i<c), A[i*h+k] = (M[i][k] - M[i][n-1-k])/2 (i<h), Mid[i] = M[i][h] (n odd).
// out[i] = E_i + O_i, out[n-1-i] = E_i - O_i with E = S (in + flip in) + Mid in[h], O = A (in - flip in): about half
// the multiplications of the plain product.
struct EOTab {
    double S[20], A[16], Mid[5];
};

struct ApplyParams {
    const double* X;
    const double* Z;
    double* Y;
    const double* eps;
    const double* sm;  // N: mu_g M_gg^{-1/2}
    const double* WV;  // cells*n^3
    const double *hx, *hy, *hz;
    int B, cx, cy, cz;
    long long Nx, NxNy;
    double alpha, beta, c;
    double w[9];  // Gauss weights
    // colour-ordered scatter (variant 4): this launch covers the cells (2i+ox, 2j+oy, 2k+oz) only; cells of one colour
    // share no node, so launching the 8 colours in order makes every sum order fixed (bit-reproducible results)
    int coloured, ox, oy, oz, ccx, ccy;
    int nokin;  // potential-only operator M^{-1/2} M_U M^{-1/2} (fe_apply_potential): the stiffness factors are 0
    EOTab eoN, eoNT, eoG;  // even-odd split of N, N^T and G (all centro-symmetric: GLL and Gauss points are symmetric)
};

__global__ void k_build_scaling(const double* __restrict__ sx, const double* __restrict__ sy,
                                const double* __restrict__ sz, long long Nx, long long Ny, long long Nz,
                                double* __restrict__ sm)
{
    long long total = Nx * Ny * Nz;
    for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < total; g += (long long)gridDim.x * blockDim.x) {
        long long gx = g % Nx, gy = (g / Nx) % Ny, gz = g / (Nx * Ny);
        sm[g] = sx[gx] * sy[gy] * sz[gz];
    }
}

inline void launch_build_scaling(const double* sx, const double* sy, const double* sz, long long Nx, long long Ny,
                                 long long Nz, double* sm, int sms, cudaStream_t st)
{
    k_build_scaling<<<sms * 8, 256, 0, st>>>(sx, sy, sz, Nx, Ny, Nz, sm);
}

// WV[e][q] = J_e w_qx w_qy w_qz V[e][q];  VZ = first tile of the cell record of the TMA kernel:
// rec[e*REC + (qx*n+qy)*NP+qz] = V[e][q] hz^2/2, NP = n rounded up to even, REC = 3 n n NP + 8
__global__ void k_weight_potential(const __grid_constant__ ApplyParams prm, int n, const double* __restrict__ V,
                                   double* __restrict__ WV, double* __restrict__ VZ, long long ncells)
{
    const int NP = n + (n & 1);
    const int n3 = n * n * n;
    long long total = ncells * n3;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        long long e = i / n3;
        int q = (int)(i - e * n3);
        int qx = q % n, qy = (q / n) % n, qz = q / (n * n);
        int ex = (int)(e % prm.cx), ey = (int)((e / prm.cx) % prm.cy), ez = (int)(e / ((long long)prm.cx * prm.cy));
        double J = prm.hx[ex] * prm.hy[ey] * prm.hz[ez] * 0.125;
        WV[i] = J * prm.w[qx] * prm.w[qy] * prm.w[qz] * V[i];
        VZ[e * (3 * n * n * NP + 8) + (qx * n + qy) * NP + qz] = 0.5 * prm.hz[ez] * prm.hz[ez] * V[i];
    }
}

inline void launch_weight_potential(const ApplyParams& prm, int p, const double* V, double* WV, double* VZ,
                                    long long ncells, int sms, cudaStream_t st)
{
    k_weight_potential<<<sms * 8, 256, 0, st>>>(prm, p + 1, V, WV, VZ, ncells);
}

// ---- even-odd form of the 1-D contractions (shared by every kernel generation) ---------------------------------------
template <int n>
__device__ __forceinline__ void mat1d_eo(const EOTab& T, const double (&in)[n], double (&out)[n])
{
    constexpr int h = n / 2, c = (n + 1) / 2;
    double e[h], o[h];
#pragma unroll
    for (int k = 0; k < h; ++k) {
        e[k] = in[k] + in[n - 1 - k];
        o[k] = in[k] - in[n - 1 - k];
    }
#pragma unroll
    for (int i = 0; i < c; ++i) {
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
        if (i < h) {
            double so = T.A[i * h] * o[0];
#pragma unroll
            for (int k = 1; k < h; ++k) so = fma(T.A[i * h + k], o[k], so);
            out[i] = se + so;
            out[n - 1 - i] = se - so;
        } else {
            out[i] = se;
        }
    }
}

// ---- legacy generation (variant 3): per-thread gather, potential and scaling tiles in shared memory, cp.async
//      prefetch of the owner rows of X and Z, red.global.add.f64 scatter into a zero-filled Y.  Takes the blocks the
//      TMA kernel cannot (odd B, unaligned bases) and serves as an independent cross-check in the tests.
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc, bool valid)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int sz = valid ? 8 : 0;  // src-size 0 zero-fills the 8 destination bytes
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gsrc), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int P, int BT, int MINB>
__global__ void __launch_bounds__((P + 1) * BT, MINB) k_apply_v3(const __grid_constant__ ApplyParams prm)
{
    constexpr int n = P + 1, n3 = n * n * n;
    extern __shared__ double smem[];
    double* sA = smem;             // [n^3][BT]
    double* sA2 = smem + n3 * BT;  // [n^3][BT]
    double* sWV = sA2 + n3 * BT;   // [n^3]  J w V of this cell
    double* sS = sWV + n3;         // [n^3]  mu * M^{-1/2} at the cell's nodes
    const int lane = threadIdx.x, pl = threadIdx.y;
    int cell = blockIdx.x;
    int ex = cell % prm.cx, ey = (cell / prm.cx) % prm.cy, ez = cell / (prm.cx * prm.cy);
    if (prm.coloured) {
        ex = 2 * (cell % prm.ccx) + prm.ox;
        ey = 2 * ((cell / prm.ccx) % prm.ccy) + prm.oy;
        ez = 2 * (cell / (prm.ccx * prm.ccy)) + prm.oz;
        cell = ex + prm.cx * (ey + prm.cy * ez);
    }
    const int j = blockIdx.y * BT + lane;
    const bool act = j < prm.B;
    const long long B = prm.B;
    const long long g0 = (long long)ex * P + prm.Nx * ((long long)ey * P) + prm.NxNy * ((long long)ez * P);
    const long long gpl = g0 + prm.NxNy * pl;
    const double* Xp = prm.X + gpl * B + j;
    const double hx = prm.hx[ex], hy = prm.hy[ey], hz = prm.hz[ez];
    const double J = hx * hy * hz * 0.125;
    const double kin = prm.nokin ? 0.0 : 2.0 * J;
    const double kx = kin / (hx * hx), ky = kin / (hy * hy), kz = kin / (hz * hz);

    double v[n][n], t[n], o[n];
    // ---- plane phase 1 ---------------------------------------------------------------------------------------------
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) v[ay][ax] = act ? Xp[(ax + prm.Nx * ay) * B] : 0.0;
    {
        const double* WVc = prm.WV + (long long)cell * n3;
        for (int i = pl * BT + lane; i < n3; i += n * BT) {
            sWV[i] = WVc[i];
            const int ax = i % n, ay = (i / n) % n, az = i / (n * n);
            sS[i] = prm.sm[g0 + ax + prm.Nx * ay + prm.NxNy * az];
        }
    }
    __syncthreads();
#pragma unroll
    for (int ay = 0; ay < n; ++ay)
#pragma unroll
        for (int ax = 0; ax < n; ++ax) {  // Dirichlet rows of caller data may hold NaN / Inf: select, do not multiply by 0
            const double sg = sS[(pl * n + ay) * n + ax];
            v[ay][ax] = __double2hiint(sg) != 0 ? v[ay][ax] * sg : 0.0;
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
        for (int q = 0; q < n; ++q) v[q][qx] = o[q];
    }
    {
        double v2[n][n];
#pragma unroll
        for (int qy = 0; qy < n; ++qy) {
            mat1d_eo<n>(prm.eoG, v[qy], o);
            const double f = kx * prm.w[qy];
#pragma unroll
            for (int qx = 0; qx < n; ++qx) v2[qy][qx] = f * o[qx];
        }
#pragma unroll
        for (int qx = 0; qx < n; ++qx) {
#pragma unroll
            for (int a = 0; a < n; ++a) t[a] = v[a][qx];
            mat1d_eo<n>(prm.eoG, t, o);
            const double f = ky * prm.w[qx];
#pragma unroll
            for (int qy = 0; qy < n; ++qy) v2[qy][qx] = fma(f, o[qy], v2[qy][qx]);
        }
#pragma unroll
        for (int qy = 0; qy < n; ++qy)
#pragma unroll
            for (int qx = 0; qx < n; ++qx) {
                const int idx = ((pl * n + qy) * n + qx) * BT + lane;
                sA[idx] = v[qy][qx];
                sA2[idx] = v2[qy][qx];
            }
    }
    __syncthreads();
    // ---- line phase ------------------------------------------------------------------------------------------------
    {
        const int qx = pl;
        const double kzwx = kz * prm.w[qx];
#pragma unroll 1
        for (int qy = 0; qy < n; ++qy) {
            double a[n], a2[n], u[n], u2[n], gu[n];
#pragma unroll
            for (int az = 0; az < n; ++az) {
                const int idx = ((az * n + qy) * n + qx) * BT + lane;
                a[az] = sA[idx];
                a2[az] = sA2[idx];
            }
            mat1d_eo<n>(prm.eoN, a, u);
            mat1d_eo<n>(prm.eoN, a2, u2);
            mat1d_eo<n>(prm.eoG, u, gu);
            const double kzw = kzwx * prm.w[qy];
#pragma unroll
            for (int qz = 0; qz < n; ++qz) {
                const double wv = sWV[(qz * n + qy) * n + qx];
                t[qz] = fma(wv, u[qz], fma(prm.w[qz], u2[qz], kzw * gu[qz]));
            }
            mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
            for (int az = 0; az < n; ++az) sA[((az * n + qy) * n + qx) * BT + lane] = o[az];
        }
    }
    __syncthreads();
    // ---- plane phase 2 ---------------------------------------------------------------------------------------------
    // The A2 rows of this thread's plane are dead now: prefetch the owner rows of Z (and of X, for the diagonal
    // term) into them with cp.async while the back-interpolation runs.  Row (ay,ax) of Z -> sA2 plane row (ay,ax);
    // row (ay,ax) of X -> the unused last row/column slots and, for the rest, sA after R has been consumed.
    const bool zterm = prm.Z != nullptr;
    const bool own_pl = pl < P;
    double* zbuf = sA2 + (size_t)pl * n * n * BT + lane;
    double* xbuf = sA + (size_t)pl * n * n * BT + lane;
    if (own_pl && zterm) {
        const double* Zp = prm.Z + gpl * B + j;
#pragma unroll
        for (int ay = 0; ay < P; ++ay)
#pragma unroll
            for (int ax = 0; ax < P; ++ax) cp_async8(zbuf + (ay * n + ax) * BT, Zp + (ax + prm.Nx * ay) * B, act);
    }
    cp_async_commit();
#pragma unroll
    for (int qy = 0; qy < n; ++qy)
#pragma unroll
        for (int qx = 0; qx < n; ++qx) v[qy][qx] = sA[((pl * n + qy) * n + qx) * BT + lane];
#pragma unroll
    for (int qx = 0; qx < n; ++qx) {
#pragma unroll
        for (int q = 0; q < n; ++q) t[q] = v[q][qx];
        mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
        for (int a = 0; a < n; ++a) v[a][qx] = o[a];
    }
    // every R value of this plane has been consumed by the arithmetic above: its sA rows can take the X rows
    if (own_pl) {
#pragma unroll
        for (int ay = 0; ay < P; ++ay)
#pragma unroll
            for (int ax = 0; ax < P; ++ax) cp_async8(xbuf + (ay * n + ax) * BT, Xp + (ax + prm.Nx * ay) * B, act);
    }
    cp_async_commit();
#pragma unroll
    for (int ay = 0; ay < n; ++ay) {
        mat1d_eo<n>(prm.eoNT, v[ay], o);
#pragma unroll
        for (int a = 0; a < n; ++a) v[ay][a] = o[a];
    }
    cp_async_wait_all();
    if (act) {
        const double ashift = -prm.alpha * (prm.c + (prm.eps ? prm.eps[j] : 0.0));
        double* Yp = prm.Y + gpl * B + j;
#pragma unroll
        for (int ay = 0; ay < n; ++ay)
#pragma unroll
            for (int ax = 0; ax < n; ++ax) {
                const double sc = sS[(pl * n + ay) * n + ax];
                double val = (prm.alpha * sc) * v[ay][ax];
                if (ax < P && ay < P) {
                    if (own_pl && __double2hiint(sc) != 0) {  // owner of a free node adds the diagonal terms once
                        val = fma(ashift, xbuf[(ay * n + ax) * BT], val);
                        if (zterm) val = fma(prm.beta, zbuf[(ay * n + ax) * BT], val);
                    }
                }
                atomicAdd(Yp + (ax + prm.Nx * ay) * B, val);
            }
    }
}

template <int P, int BT, int MINB>
cudaError_t launch_v3(const ApplyParams& prm, long long ncells, cudaStream_t st)
{
    constexpr int n = P + 1;
    const size_t smem = ((size_t)2 * n * n * n * BT + 2 * n * n * n) * sizeof(double);
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_apply_v3<P, BT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    dim3 grid((unsigned)ncells, (unsigned)((prm.B + BT - 1) / BT)), block(BT, n);
    k_apply_v3<P, BT, MINB><<<grid, block, smem, st>>>(prm);
    return cudaGetLastError();
}

inline bool variant_supported(int p, int variant)
{
    (void)p;
    return variant == 0 || variant == 3 || variant == 4 || (variant >= 5 && variant <= 9);
}

// One fused operator step.  *nlaunch = kernels (and memsets) enqueued.
inline cudaError_t launch_apply(const ApplyParams& prm, int p, int variant, long long N, long long ncells,
                                cudaStream_t st, int* nlaunch)
{
    cudaError_t e = cudaMemsetAsync(prm.Y, 0, (size_t)N * prm.B * sizeof(double), st);
    if (e != cudaSuccess) return e;
    *nlaunch = 1;  // kernels only; the zero-fill is a cudaMemsetAsync
    auto launch = [&](const ApplyParams& q, long long nc) -> cudaError_t {
        switch (p) {
            case 1: return launch_v3<1, 32, 8>(q, nc, st);
            case 2: return launch_v3<2, 32, 6>(q, nc, st);
            case 3: return launch_v3<3, 32, 4>(q, nc, st);
            case 4: return launch_v3<4, 32, 3>(q, nc, st);
            case 5: return launch_v3<5, 32, 1>(q, nc, st);
            case 6: return launch_v3<6, 16, 2>(q, nc, st);
            case 7: return launch_v3<7, 16, 1>(q, nc, st);
            case 8: return launch_v3<8, 16, 1>(q, nc, st);
        }
        return cudaErrorInvalidValue;
    };
    if (variant != 4) return launch(prm, ncells);
    // colour-ordered: 8 launches over the 2x2x2 parity classes of the cell grid, in a fixed order
    *nlaunch = 0;
    for (int col = 0; col < 8; ++col) {
        ApplyParams q = prm;
        q.coloured = 1;
        q.ox = col & 1; q.oy = (col >> 1) & 1; q.oz = (col >> 2) & 1;
        const int ccx = (prm.cx - q.ox + 1) / 2, ccy = (prm.cy - q.oy + 1) / 2, ccz = (prm.cz - q.oz + 1) / 2;
        if (ccx <= 0 || ccy <= 0 || ccz <= 0) continue;
        q.ccx = ccx; q.ccy = ccy;
        e = launch(q, (long long)ccx * ccy * ccz);
        if (e != cudaSuccess) return e;
        *nlaunch += 1;
    }
    return cudaSuccess;
    return cudaErrorInvalidValue;
}

}  // namespace fecheb
