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
// Threads: lane = vector j (BT per cell tile), threadIdx.y = a line slot.  Each of the 12 sweeps is a loop over the n^2
// lines of its direction, dealt to the line slots; a thread holds one line (n values) in registers, every 1-D matrix entry
// is a warp-uniform operand, and the cell tile lives in shared memory (three fields of n^3 x BT doubles: x/A/U/t/R, gy/fy,
// gz/fz) with a CTA barrier where the direction changes.  Gather and scatter go through the explicit l2g; hanging
// nodes read the expanded values X_h = C_h (s . X) (k_gen_expand) and scatter into Y_h, which k_gen_collapse distributes
// to the unconstrained nodes with C_h^T.  The shift and recurrence terms are written by k_gen_init, which replaces the
// zero-fill of Y.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "fe_apply_tma.cuh"
#include "fe_kernels.cuh"

namespace fecheb {

struct GenParams {
    const double* X;     // N * B
    const double* Xh;    // (N_all - N) * B: expanded hanging values
    double* Y;           // N * B
    double* Yh;          // (N_all - N) * B
    const int32_t* l2g;  // ncells * n^3
    const double* sc;    // ncells * n^3: s_g = mu_g M_c,gg^{-1/2} at the cell's unconstrained nodes, 1 at its hanging nodes
    const double* rec;   // ncells * GREC: per-cell record, 6 metric fields (fe_general.h) then WV = w_q |J| V_q, n^3 each
    const int32_t* cell_list;  // NULL: all cells 0..ncells-1; else the ncells cells of one colour (colour-ordered scatter)
    long long N, ncells;
    int B;
    double alpha;
    // even-odd halves (fe_kernels.cuh): N and N^T are centro-symmetric, the collocation derivative D and D^T are
    // centro-ANTIsymmetric (D[n-1-s][n-1-q] = -D[s][q]); for those the row i = h of S holds the middle row D[h][k], k < h
    EOTab eoN, eoNT, eoD, eoDT;
};

// Block shape of the row-wise helper kernels: lanes run over the vectors j of a row, threadIdx.y over rows
constexpr int kGenRows = 8;

// Y = mu (kappa_j X + beta Z), kappa_j = -alpha (c + eps_j): the part of the step that is diagonal in the nodes
__global__ void k_gen_init(double* __restrict__ Y, const double* __restrict__ X, const double* __restrict__ Z,
                           const double* __restrict__ s, const double* __restrict__ eps, double alpha, double beta,
                           double c, long long N, int B)
{
    for (long long g = blockIdx.x * (long long)kGenRows + threadIdx.y; g < N; g += (long long)gridDim.x * kGenRows) {
        const bool fr = s[g] != 0.0;
        for (int j = threadIdx.x; j < B; j += 32) {
            const long long i = g * B + j;
            double v = 0.0;
            if (fr) {
                const double kappa = -alpha * (c + (eps ? eps[j] : 0.0));
                if (kappa != 0.0) v = kappa * X[i];
                if (Z) v = fma(beta, Z[i], v);
            }
            Y[i] = v;
        }
    }
}

// Sparse rows times a block:  dst[out_r, j] (+)= alpha sum_k w_rk src[col_k, j].
//   expansion  X_h = C_h (s . X):        src = X,   dst = X_h, w = cval * s[col] (entries of Dirichlet nodes, s = 0, are dropped
//                                        when the bundles are packed: their rows of X are never read)
//   collapse   Y += alpha s . C_h^T Y_h:  k_gen_collapse below, the same bundles read the other way
// The hanging nodes of one coarse face all depend on the same n^2 nodes (and the nodes of a coarse face all feed the same
// hanging nodes), so the host sorts the rows by their column lists and packs rows with IDENTICAL lists into bundles of up to
// kGenBundle rows (GenBundles in fe_cheb.cu): a warp (lanes = vectors) works on one bundle, reads every row of src once for
// all its rows and the bundle's weights as one 64-byte line per entry -- row by row the kernel moved n^2 x the block through
// L2 and was bound by L2 bandwidth.  bptr[b] .. bptr[b+1]: entries of bundle b (col, 8 weights each); brow[b] .. brow[b+1]:
// its rows in `out`.
constexpr int kGenBundle = 8;

__global__ void __launch_bounds__(32 * kGenRows, 4)
k_gen_rows_times_block(double* __restrict__ dst, const double* __restrict__ src, const long long* __restrict__ bptr,
                       const int32_t* __restrict__ bcol, const double* __restrict__ bw, const int32_t* __restrict__ brow,
                       const int32_t* __restrict__ out, long long nb, int B, double alpha, int accumulate,
                       double* __restrict__ zero)  // zero != NULL: the same rows of this second block are cleared (Y_h of the step)
{
    // A warp stages 32 entries of its bundle (column ids and the 8 weights each, coalesced) in shared memory and then walks
    // them with the rows of src as INDEPENDENT loads, eight in flight: read straight from global memory the chain
    // column id -> row address -> value made every entry two dependent round trips, and the kernel was bound by that latency.
    __shared__ int32_t s_col[kGenRows][32];
    __shared__ __align__(16) double s_w[kGenRows][32][kGenBundle];
    const int ty = threadIdx.y, lane = threadIdx.x;
    for (long long b = blockIdx.x * (long long)kGenRows + ty; b < nb; b += (long long)gridDim.x * kGenRows) {
        const long long k0 = bptr[b], k1 = bptr[b + 1];
        const int r0 = brow[b], m = brow[b + 1] - r0;
        for (int j0 = 0; j0 < B; j0 += 32) {
            const int j = j0 + lane;
            const bool act = j < B;
            const double* sj = src + (act ? j : 0);
            double v[kGenBundle];
#pragma unroll
            for (int u = 0; u < kGenBundle; ++u) v[u] = 0.0;
            for (long long kc = k0; kc < k1; kc += 32) {
                __syncwarp();
                if (kc + lane < k1) {
                    s_col[ty][lane] = bcol[kc + lane];
                    const double4* wsrc = reinterpret_cast<const double4*>(bw + (kc + lane) * kGenBundle);
                    *reinterpret_cast<double4*>(&s_w[ty][lane][0]) = wsrc[0];
                    *reinterpret_cast<double4*>(&s_w[ty][lane][4]) = wsrc[1];
                }
                __syncwarp();
                const int cnt = (int)((k1 - kc) < 32 ? (k1 - kc) : 32);
#pragma unroll 8
                for (int e = 0; e < cnt; ++e) {
                    const double x = sj[(long long)s_col[ty][e] * B];
                    const double4 w0 = *reinterpret_cast<const double4*>(&s_w[ty][e][0]);
                    const double4 w1 = *reinterpret_cast<const double4*>(&s_w[ty][e][4]);
                    // no test of the weights: entries of Dirichlet nodes (all weights 0, data to be ignored) are not in the bundles
                    v[0] = fma(w0.x, x, v[0]); v[1] = fma(w0.y, x, v[1]); v[2] = fma(w0.z, x, v[2]); v[3] = fma(w0.w, x, v[3]);
                    v[4] = fma(w1.x, x, v[4]); v[5] = fma(w1.y, x, v[5]); v[6] = fma(w1.z, x, v[6]); v[7] = fma(w1.w, x, v[7]);
                }
            }
            if (act) {
#pragma unroll
                for (int u = 0; u < kGenBundle; ++u)
                    if (u < m) {
                        const long long i = (long long)out[r0 + u] * B + j;
                        dst[i] = accumulate ? fma(alpha, v[u], dst[i]) : alpha * v[u];
                        if (zero) zero[i] = 0.0;
                    }
            }
        }
    }
}

// Y[col_k, j] += alpha sum_u w_ku Y_h[out_u, j] over the bundles of the expansion: the transpose of k_gen_rows_times_block
// from the SAME packed rows -- the (up to 8) hanging rows of a bundle are read once, every entry costs one red.global.add of the
// bundle's combined contribution (an eighth of the atomics of a row-by-row transpose; sorting the transposed rows instead
// does not bundle, because exactly-zero weights make the column lists of neighbouring nodes differ)
__global__ void __launch_bounds__(32 * kGenRows, 4)
k_gen_collapse(double* __restrict__ Y, const double* __restrict__ Yh, const long long* __restrict__ bptr,
               const int32_t* __restrict__ bcol, const double* __restrict__ bw, const int32_t* __restrict__ brow,
               const int32_t* __restrict__ out, long long nb, int B, double alpha)
{
    for (long long b = blockIdx.x * (long long)kGenRows + threadIdx.y; b < nb; b += (long long)gridDim.x * kGenRows) {
        const long long k0 = bptr[b], k1 = bptr[b + 1];
        const int r0 = brow[b], m = brow[b + 1] - r0;
        for (int j = threadIdx.x; j < B; j += 32) {
            double y[kGenBundle];
#pragma unroll
            for (int u = 0; u < kGenBundle; ++u) y[u] = u < m ? alpha * Yh[(long long)out[r0 + u] * B + j] : 0.0;
#pragma unroll 2
            for (long long k = k0; k < k1; ++k) {
                const double4 w0 = *reinterpret_cast<const double4*>(bw + k * kGenBundle);
                const double4 w1 = *reinterpret_cast<const double4*>(bw + k * kGenBundle + 4);
                double v = w0.x * y[0];
                v = fma(w0.y, y[1], v); v = fma(w0.z, y[2], v); v = fma(w0.w, y[3], v);
                v = fma(w1.x, y[4], v); v = fma(w1.y, y[5], v); v = fma(w1.z, y[6], v); v = fma(w1.w, y[7], v);
                atomicAdd(Y + (long long)bcol[k] * B + j, v);  // unconditional: a predicated red.global becomes a branch (fe_gbox.cuh)
            }
        }
    }
}

// diagonal of the assembled kinetic matrix over ALL nodes (MINRES preconditioner, l.225): kd[g] += sum_q grad^ Phi_a(q)^T G_q
// grad^ Phi_a(q), one thread per (cell, local node), an explicit loop over the cell's quadrature points (setup, not hot).
// Nt[q*n+a] = l_a(gl_q), DNt[q*n+a] = l_a'(gl_q).
struct GenDiagTables {
    double Nt[81], DNt[81];
};
__global__ void k_gen_kinetic_diag(double* __restrict__ kd, const double* __restrict__ rec, const int32_t* __restrict__ l2g,
                                   long long ncells, int n, int grec, const __grid_constant__ GenDiagTables tb)
{
    const int n3 = n * n * n;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ncells * n3; i += (long long)gridDim.x * blockDim.x) {
        const long long e = i / n3;
        const int a = (int)(i - e * n3), ax = a % n, ay = (a / n) % n, az = a / (n * n);
        const double* M = rec + e * grec;
        double sum = 0.0;
        for (int qz = 0; qz < n; ++qz)
            for (int qy = 0; qy < n; ++qy)
                for (int qx = 0; qx < n; ++qx) {
                    const int q = qx + n * (qy + n * qz);
                    const double lx = tb.Nt[qx * n + ax], ly = tb.Nt[qy * n + ay], lz = tb.Nt[qz * n + az];
                    const double dx = tb.DNt[qx * n + ax] * ly * lz, dy = lx * tb.DNt[qy * n + ay] * lz, dz = lx * ly * tb.DNt[qz * n + az];
                    sum += M[q] * dx * dx + M[3 * n3 + q] * dy * dy + M[5 * n3 + q] * dz * dz +
                           2.0 * (M[n3 + q] * dx * dy + M[2 * n3 + q] * dx * dz + M[4 * n3 + q] * dy * dz);
                }
        atomicAdd(kd + l2g[i], sum);
    }
}

// per-cell record of the general kernel: 7 fields of n^3 doubles (6 metric entries, WV), padded to a multiple of 16 bytes
inline int gen_rec_doubles(int n) { const int r = 7 * n * n * n; return r + (r & 1); }

// field 6 of every record: WV[e][q] = w_q |J| V[e][q]
__global__ void k_gen_weight_potential(double* __restrict__ rec, const double* __restrict__ V,
                                       const double* __restrict__ wdet, long long ncells, int n3, int grec)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ncells * n3; i += (long long)gridDim.x * blockDim.x) {
        const long long e = i / n3;
        rec[e * grec + 6 * n3 + (i - e * n3)] = wdet[i] * V[i];
    }
}

// even-odd product with a centro-ANTIsymmetric matrix: out[i] = E + O, out[n-1-i] = O - E (mat1d_eo has E - O there)
template <int n>
__device__ __forceinline__ void mat1d_eoa(const EOTab& T, const double (&in)[n], double (&out)[n])
{
    constexpr int h = n / 2;
    double e[h > 0 ? h : 1], o[h > 0 ? h : 1];
#pragma unroll
    for (int k = 0; k < h; ++k) {
        e[k] = in[k] + in[n - 1 - k];
        o[k] = in[k] - in[n - 1 - k];
    }
#pragma unroll
    for (int i = 0; i < h; ++i) {
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
        double so = T.A[i * h] * o[0];
#pragma unroll
        for (int k = 1; k < h; ++k) so = fma(T.A[i * h + k], o[k], so);
        out[i] = se + so;
        out[n - 1 - i] = so - se;
    }
    if (n % 2 == 1) {
        double sm = 0.0;
        if (h > 0) {
            sm = T.S[h * h] * o[0];
#pragma unroll
            for (int k = 1; k < h; ++k) sm = fma(T.S[h * h + k], o[k], sm);
        }
        out[h] = sm;
    }
}

template <int P, int BT, bool PERSIST>
constexpr size_t gen_smem_bytes()
{
    constexpr int n3 = (P + 1) * (P + 1) * (P + 1), NB = PERSIST ? 2 : 1;
    return (size_t)3 * n3 * BT * sizeof(double) + (size_t)NB * (7 * n3 + 1) * sizeof(double) +
           (size_t)NB * (n3 + 1) * (sizeof(double) + sizeof(int32_t)) + 64;
}

// line slots of a CTA: every sweep has n^2 lines per vector; ceil(n^2 / 2) slots take them in two rounds
template <int P>
struct GenShape {
    static constexpr int LS = ((P + 1) * (P + 1) + 1) / 2;
};

// One CTA = one cell x BT vectors.  lane = vector, threadIdx.y = line slot.  Every sweep is a loop over the n^2 lines of
// one direction (a line = n values, stride sx/sy/sz in the field); the fields live in shared memory, a thread holds one
// line in registers.  The loops are NOT unrolled over lines, so the whole kernel is a few hundred FP64 instructions per
// sweep and stays in the instruction cache (the plane-in-registers version of this kernel, 150 KB of straight-line code run
// by 3.5 warps, spent 4 of 5 issue slots waiting for instructions).
// PERSIST: the CTA walks units (cell, vector tile) u = blockIdx.x, + gridDim.x, ...; while unit u runs its last two sweeps the
// node rows of unit u + gridDim.x are already being fetched into the field that sweep 7 has freed, and its ids, scales and
// metric record were requested at the start of unit u (second set of buffers), so the gather latency -- a quarter of the
// one-unit-per-CTA kernel's time (ncu) -- hides behind arithmetic.  The three fields rotate roles from unit to unit.
template <int P, int BT, int MINB, bool PERSIST>
__global__ void __launch_bounds__(GenShape<P>::LS * BT, MINB) k_apply_gen(const __grid_constant__ GenParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n, LS = GenShape<P>::LS, NB = PERSIST ? 2 : 1;
    constexpr int SX = BT, SY = n * BT, SZ = n2 * BT;  // strides of the three directions in a field [z][y][x][BT]
    constexpr int GREC = 7 * n3 + ((7 * n3) & 1), N3E = n3 + (n3 & 1);
    extern __shared__ __align__(128) double smem[];
    double* F0 = smem;                  // x -> A -> U -> t -> T -> R
    double* F1 = F0 + (size_t)n3 * BT;  // gy -> fy          (then the next unit's x)
    double* F2 = F1 + (size_t)n3 * BT;  // gz -> fz
    double* sRecB = F2 + (size_t)n3 * BT;  // [NB] the cell's record (6 metric fields, WV): one bulk copy, needed from sweep 5 on
    double* sScB = sRecB + NB * GREC;      // [NB][n^3] gather / scatter scale of the cell's nodes
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(sScB + NB * N3E);  // [2]
    int32_t* sIdB = reinterpret_cast<int32_t*>(bar + 2);  // [NB][n^3] global ids
    const int lane = threadIdx.x, slot = threadIdx.y, tid = slot * BT + lane;
    const int ntile = (prm.B + BT - 1) / BT;
    const long long nunits = prm.ncells * ntile;
    double t[n], o[n];
    // the (at most) two lines of this slot in every sweep, as field offsets: x-lines (i1, i2), y-lines (i0, i2), z-lines (i0, i1)
    const bool two = slot + LS < n2;
    int lx[2], ly[2], lz[2], ll[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int l = (r == 0 || two) ? slot + r * LS : slot;
        ll[r] = l;
        lx[r] = l * n * BT + lane;
        ly[r] = ((l / n) * n2 + (l % n)) * BT + lane;
        lz[r] = l * BT + lane;
    }
    // requests for a unit: ids and scales (4- / 8-byte cp.async) and the record (bulk copy on bar[buf]) ...
    auto request_tables = [&](long long u, int buf) {
        const long long cu = u / ntile;
        const long long c = prm.cell_list ? prm.cell_list[cu] : cu;
        if (tid == 0) {
            mbar_expect_tx(bar + buf, (unsigned)(GREC * sizeof(double)));
            bulk_load(sRecB + buf * GREC, prm.rec + c * GREC, (unsigned)(GREC * sizeof(double)), bar + buf);
        }
        for (int a = tid; a < n3; a += LS * BT) {
            const unsigned di = (unsigned)__cvta_generic_to_shared(sIdB + buf * n3 + a);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(di), "l"(prm.l2g + c * n3 + a) : "memory");
            cp_async8(sScB + buf * N3E + a, prm.sc + c * n3 + a, true);
        }
        cp_async_commit();
    };
    // ... and its node rows, once the ids are in shared memory: independent 8-byte cp.async straight into the field
    // node addresses in 32-bit pieces (ids and N fit 32 bits): row of node g = base + g * (8 B) bytes with one wide
    // multiply-add, base = X (unconstrained) or X_h - N * 8 B (hanging) -- fe_gbox.cuh
    const unsigned N32 = (unsigned)prm.N, B8 = (unsigned)prm.B * 8u;
    const unsigned long long hoff = (unsigned long long)N32 * B8;
    auto request_rows = [&](long long u, int buf, double* F) {
        const int jn = (int)(u % ntile) * BT + lane;
        const bool an = jn < prm.B;
        const char* bX = reinterpret_cast<const char*>(prm.X + (an ? jn : 0));
        const char* bH = reinterpret_cast<const char*>(prm.Xh + (an ? jn : 0)) - hoff;
        for (int a = slot; a < n3; a += LS) {
            const unsigned g = (unsigned)sIdB[buf * n3 + a];
            cp_async8(F + (size_t)a * BT + lane, (g < N32 ? bX : bH) + (unsigned long long)g * B8, an);
        }
        cp_async_commit();
    };
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 1, 1);
    }
    __syncthreads();
    if ((long long)blockIdx.x < nunits) {
        request_tables(blockIdx.x, 0);
        cp_async_wait_all();
        __syncthreads();
        request_rows(blockIdx.x, 0, F0);
    }
    unsigned ph0 = 0, ph1 = 0;  // phases of the two record barriers
    int buf = 0;
    for (long long u = blockIdx.x; u < nunits; u += gridDim.x, buf ^= (PERSIST ? 1 : 0)) {
    const long long un = u + gridDim.x;
    const bool more = PERSIST && un < nunits;
    const int j = (int)(u % ntile) * BT + lane;
    const bool act = j < prm.B;
    const double* sRec = sRecB + buf * GREC;
    const double* sSc = sScB + buf * N3E;
    const int32_t* sId = sIdB + buf * n3;
    cp_async_wait_all();
    __syncthreads();  // this unit's rows are in F0; the previous unit has left its buffers
    if (more) request_tables(un, buf ^ 1);
    // ---- sweep 1: x-lines (ay, az) of the nodal values: scale (mask, M^-1/2), interpolate (table N) -----------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        double* f = F0 + lx[r];
        const double* sc = sSc + l * n;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double sg = sc[k];
            t[k] = sg != 0.0 ? sg * f[k * SX] : 0.0;  // Dirichlet rows of caller data are ignored (R5)
        }
        mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SX] = o[k];
    }
    __syncthreads();
    // ---- sweep 2: y-lines (qx, az) (table N) -----------------------------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        double* f = F0 + ly[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SY];
        mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SY] = o[k];
    }
    __syncthreads();
    // ---- sweep 3: z-lines (qx, qy): U = Nz A (table N), then gz = Dz U on the same lines (table D) -------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        double* f = F0 + lz[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SZ];
        mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SZ] = o[k];
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        const int off = lz[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = F0[off + k * SZ];
        mat1d_eoa<n>(prm.eoD, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) F2[off + k * SZ] = o[k];
    }
    __syncthreads();
    // ---- sweep 4: y-lines (qx, qz): gy = Dy U (table D) ---------------------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        const int off = ly[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = F0[off + k * SY];
        mat1d_eoa<n>(prm.eoD, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) F1[off + k * SY] = o[k];
    }
    __syncthreads();
    // ---- sweep 5: x-lines (qy, qz): gx = Dx U (table D), the metric at the line's points, t = WV U + Dx^T fx (table D^T) -------------
    if (buf == 0) { mbar_wait(bar, ph0); ph0 ^= 1; } else { mbar_wait(bar + 1, ph1); ph1 ^= 1; }
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        const int off = lx[r];
        const double* Mq = sRec + l * n;  // + c * n3 + qx
        double u[n];
#pragma unroll
        for (int k = 0; k < n; ++k) u[k] = F0[off + k * SX];
        mat1d_eoa<n>(prm.eoD, u, o);
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double gxv = o[k], gyv = F1[off + k * SX], gzv = F2[off + k * SX];
            const double g0 = Mq[k], g1 = Mq[n3 + k], g2 = Mq[2 * n3 + k], g3 = Mq[3 * n3 + k], g4 = Mq[4 * n3 + k],
                         g5 = Mq[5 * n3 + k];
            t[k] = fma(g0, gxv, fma(g1, gyv, g2 * gzv));
            F1[off + k * SX] = fma(g1, gxv, fma(g3, gyv, g4 * gzv));
            F2[off + k * SX] = fma(g2, gxv, fma(g4, gyv, g5 * gzv));
        }
        mat1d_eoa<n>(prm.eoDT, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) F0[off + k * SX] = fma(Mq[6 * n3 + k], u[k], o[k]);
    }
    __syncthreads();
    // ---- sweep 6: y-lines (qx, qz): t += Dy^T fy (table D^T) ------------------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        const int off = ly[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = F1[off + k * SY];
        mat1d_eoa<n>(prm.eoDT, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) F0[off + k * SY] += o[k];
    }
    __syncthreads();
    // ---- sweep 7: z-lines (qx, qy): T = t + Dz^T fz (table D^T), then R = Nz^T T on the same lines (table N^T) -------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        const int off = lz[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = F2[off + k * SZ];
        mat1d_eoa<n>(prm.eoDT, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) F0[off + k * SZ] += o[k];
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        double* f = F0 + lz[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SZ];
        mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SZ] = o[k];
    }
    if (more) cp_async_wait_all();  // the next unit's ids and scales (requested at the top of this unit)
    __syncthreads();
    if (more) request_rows(un, buf ^ 1, F1);  // F1 and F2 are free from here on
    // ---- sweep 8: y-lines (qx, az) (table N^T) ----------------------------------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        double* f = F0 + ly[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SY];
        mat1d_eo<n>(prm.eoNT, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SY] = o[k];
    }
    __syncthreads();
    // ---- sweep 9: x-lines (ay, az) (table N^T) and the scatter of the line's n nodes through the l2g -----------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) if (r == 0 || two) {
        const int l = ll[r];
        const double* f = F0 + lx[r];
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SX];
        mat1d_eo<n>(prm.eoNT, t, o);
        {   // unconditional adds: a predicated red.global becomes a branch with uniform-register spills around it (fe_gbox.cuh);
            // Dirichlet nodes (scale 0) and idle lanes (column 0 of their node) add +0.0, which changes nothing
            const int jj = act ? j : 0;
            char* yX = reinterpret_cast<char*>(prm.Y + jj);
            char* yH = reinterpret_cast<char*>(prm.Yh + jj) - hoff;
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const unsigned g = (unsigned)sId[l * n + k];
                const double sg = sSc[l * n + k];
                const bool master = g < N32;
                double* dst = reinterpret_cast<double*>((master ? yX : yH) + (unsigned long long)g * B8);
                atomicAdd(dst, (act && sg != 0.0) ? (master ? prm.alpha * sg * o[k] : o[k]) : 0.0);
            }
        }
    }
    double* Fr = F0; F0 = F1; F1 = F2; F2 = Fr;  // the field that holds the next unit's rows becomes F0
    }  // units
}

// Electron density at the quadrature points on a general mesh (Eq. 4 l.73-77): rho[e][q] = sum_j f_j psi_j(x_q)^2 with
// psi = M_c^{-1/2} psi~ expanded through the constraints -- the gather and the three interpolation sweeps of k_apply_gen,
// then f_j U^2 summed over the BT vectors of the tile (shuffles inside the lane group) and added to rho.
struct GenDensityParams {
    const double* X;
    const double* Xh;
    const double* f;
    double* rho;
    const int32_t* l2g;
    const double* sc;
    long long N;
    int B;
    EOTab eoN;
};

template <int P, int BT, int MINB>
__global__ void __launch_bounds__(GenShape<P>::LS * BT, MINB) k_density_gen(const __grid_constant__ GenDensityParams prm)
{
    constexpr int n = P + 1, n2 = n * n, n3 = n * n * n, LS = GenShape<P>::LS;
    constexpr int SX = BT, SY = n * BT, SZ = n2 * BT;
    extern __shared__ __align__(128) double smem[];
    double* F0 = smem;
    double* sSc = F0 + (size_t)n3 * BT;
    int32_t* sId = reinterpret_cast<int32_t*>(sSc + n3 + (n3 & 1));
    const int lane = threadIdx.x, slot = threadIdx.y, tid = slot * BT + lane;
    const long long cell = blockIdx.x;
    const int j = blockIdx.y * BT + lane;
    const bool act = j < prm.B;
    const long long B = prm.B;
    double t[n], o[n];
    for (int a = tid; a < n3; a += LS * BT) {
        sId[a] = prm.l2g[cell * n3 + a];
        sSc[a] = prm.sc[cell * n3 + a];
    }
    __syncthreads();
    for (int a = slot; a < n3; a += LS) {
        const long long g = sId[a];
        const double* src = g < prm.N ? prm.X + g * B + j : prm.Xh + (g - prm.N) * B + j;
        cp_async8(F0 + (size_t)a * BT + lane, act ? src : prm.X, act);
    }
    cp_async_commit();
    cp_async_wait_all();
    __syncthreads();
    for (int l = slot; l < n2; l += LS) {  // x-lines: scale, interpolate
        double* f = F0 + (size_t)l * n * BT + lane;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            const double sg = sSc[l * n + k];
            t[k] = sg != 0.0 ? sg * f[k * SX] : 0.0;
        }
        mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SX] = o[k];
    }
    __syncthreads();
    for (int l = slot; l < n2; l += LS) {  // y-lines
        double* f = F0 + ((size_t)(l / n) * n2 + (l % n)) * BT + lane;
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SY];
        mat1d_eo<n>(prm.eoN, t, o);
#pragma unroll
        for (int k = 0; k < n; ++k) f[k * SY] = o[k];
    }
    __syncthreads();
    const double fj = act ? prm.f[j] : 0.0;
    for (int l = slot; l < n2; l += LS) {  // z-lines (qx, qy) = (l % n, l / n): psi at the Gauss points, squared and summed
        const double* f = F0 + (size_t)l * BT + lane;
#pragma unroll
        for (int k = 0; k < n; ++k) t[k] = f[k * SZ];
        mat1d_eo<n>(prm.eoN, t, o);
        const unsigned peers = __activemask();  // the lane groups of this warp that have a line in this round
#pragma unroll
        for (int k = 0; k < n; ++k) {
            double v = fj * o[k] * o[k];
#pragma unroll
            for (int d = BT / 2; d > 0; d >>= 1) v += __shfl_xor_sync(peers, v, d, BT);
            if (lane == 0) atomicAdd(prm.rho + cell * n3 + (size_t)k * n2 + l, v);
        }
    }
}

template <int P, int BT, int MINB>
cudaError_t launch_density_gen_t(const GenDensityParams& prm, long long ncells, cudaStream_t st)
{
    constexpr int n3 = (P + 1) * (P + 1) * (P + 1);
    constexpr size_t smem = (size_t)n3 * BT * sizeof(double) + (size_t)(n3 + 1) * (sizeof(double) + sizeof(int32_t)) + 16;
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_density_gen<P, BT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    dim3 grid((unsigned)ncells, (unsigned)((prm.B + BT - 1) / BT)), block(BT, GenShape<P>::LS);
    k_density_gen<P, BT, MINB><<<grid, block, smem, st>>>(prm);
    return cudaGetLastError();
}

inline cudaError_t launch_density_gen(const GenDensityParams& prm, int p, long long ncells, cudaStream_t st)
{
    switch (p) {
        case 1: return launch_density_gen_t<1, 32, 8>(prm, ncells, st);
        case 2: return launch_density_gen_t<2, 32, 6>(prm, ncells, st);
        case 3: return launch_density_gen_t<3, 32, 4>(prm, ncells, st);
        case 4: return launch_density_gen_t<4, 32, 2>(prm, ncells, st);
        case 5: return launch_density_gen_t<5, 16, 2>(prm, ncells, st);
        case 6: return launch_density_gen_t<6, 16, 2>(prm, ncells, st);
        case 7: return launch_density_gen_t<7, 8, 2>(prm, ncells, st);
        case 8: return launch_density_gen_t<8, 8, 2>(prm, ncells, st);
    }
    return cudaErrorInvalidValue;
}

template <int P, int BT, int MINB, bool PERSIST>
cudaError_t launch_gen(const GenParams& prm, long long ncells, int sms, cudaStream_t st)
{
    constexpr size_t smem = gen_smem_bytes<P, BT, PERSIST>();
    static PerDeviceOnce once;
    cudaError_t e0 = once_per_device(once, [&] {
        return cudaFuncSetAttribute(k_apply_gen<P, BT, MINB, PERSIST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    });
    if (e0 != cudaSuccess) return e0;
    const long long nunits = ncells * ((prm.B + BT - 1) / BT);
    const long long ctas = PERSIST ? std::min<long long>(nunits, (long long)sms * MINB) : nunits;
    dim3 grid((unsigned)ctas), block(BT, GenShape<P>::LS);
    k_apply_gen<P, BT, MINB, PERSIST><<<grid, block, smem, st>>>(prm);
    return cudaGetLastError();
}

// vector-tile width per order: three fields of n^3 x BT doubles + the cell record per CTA, several CTAs per SM where they
// fit.  The persistent walk with prefetched rows pays where only ONE CTA fits an SM (p = 7: 27.1 -> 31.2 GDoF-vec/s on the
// adaptive workload); with two CTAs per SM the hardware already overlaps one CTA's gather with the other's arithmetic and
// the loop state costs 3-4 % (p = 4, 6); p = 8 has no room for the second set of buffers.
inline cudaError_t launch_apply_gen(const GenParams& prm, int p, long long ncells, int sms, cudaStream_t st)
{
    switch (p) {
        case 1: return launch_gen<1, 32, 8, false>(prm, ncells, sms, st);
        case 2: return launch_gen<2, 32, 6, false>(prm, ncells, sms, st);
        case 3: return launch_gen<3, 32, 4, false>(prm, ncells, sms, st);
        case 4: return launch_gen<4, 32, 2, false>(prm, ncells, sms, st);
        case 5: return launch_gen<5, 16, 2, false>(prm, ncells, sms, st);
        case 6: return launch_gen<6, 8, 2, false>(prm, ncells, sms, st);
        case 7: return launch_gen<7, 8, 1, true>(prm, ncells, sms, st);
        case 8: return launch_gen<8, 8, 1, false>(prm, ncells, sms, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace fecheb
