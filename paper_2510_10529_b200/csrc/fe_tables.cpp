// Host-side 1-D tables, computed by a route that shares nothing with the CPU oracle (which uses Newton on
// Legendre polynomials and the literal product formula): here the quadrature nodes are eigenvalues of Jacobi
// matrices (Golub-Welsch), the basis is evaluated with the barycentric formula, and the derivative at the
// Gauss points is the collocation differentiation matrix of the Gauss-point Lagrange basis.
#include "fe_tables.h"

#include <algorithm>
#include <cmath>

namespace fecheb {
namespace {

typedef long double real;

// Cyclic Jacobi eigen-decomposition of a symmetric m x m matrix (m <= 9).  A is destroyed; eigenvalues on its
// diagonal, eigenvectors in the columns of V.
void jacobi_eig(int m, real A[kMaxN][kMaxN], real V[kMaxN][kMaxN])
{
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) V[i][j] = (i == j) ? 1.0L : 0.0L;
    for (int sweep = 0; sweep < 100; ++sweep) {
        real off = 0.0L;
        for (int i = 0; i < m; ++i)
            for (int j = i + 1; j < m; ++j) off += A[i][j] * A[i][j];
        if (off < 1e-60L) break;
        for (int pi = 0; pi < m; ++pi)
            for (int qi = pi + 1; qi < m; ++qi) {
                if (A[pi][qi] == 0.0L) continue;
                real theta = (A[qi][qi] - A[pi][pi]) / (2.0L * A[pi][qi]);
                real t = ((theta >= 0) ? 1.0L : -1.0L) / (fabsl(theta) + sqrtl(theta * theta + 1.0L));
                real c = 1.0L / sqrtl(t * t + 1.0L), s = t * c;
                for (int k = 0; k < m; ++k) {
                    real akp = A[k][pi], akq = A[k][qi];
                    A[k][pi] = c * akp - s * akq;
                    A[k][qi] = s * akp + c * akq;
                }
                for (int k = 0; k < m; ++k) {
                    real apk = A[pi][k], aqk = A[qi][k];
                    A[pi][k] = c * apk - s * aqk;
                    A[qi][k] = s * apk + c * aqk;
                }
                for (int k = 0; k < m; ++k) {
                    real vkp = V[k][pi], vkq = V[k][qi];
                    V[k][pi] = c * vkp - s * vkq;
                    V[k][qi] = s * vkp + c * vkq;
                }
            }
    }
}

// nodes/weights of the m-point Gauss rule for the weight (1-x^2)^alpha, alpha in {0,1}; mu0 = integral of the weight
void golub_welsch(int m, int alpha, real* x, real* w)
{
    real A[kMaxN][kMaxN], V[kMaxN][kMaxN];
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) A[i][j] = 0.0L;
    for (int k = 1; k < m; ++k) {
        real b2 = (alpha == 0) ? (real)k * k / (4.0L * k * k - 1.0L)
                               : (real)k * (k + 2) / ((2.0L * k + 1.0L) * (2.0L * k + 3.0L));
        A[k - 1][k] = A[k][k - 1] = sqrtl(b2);
    }
    jacobi_eig(m, A, V);
    real mu0 = (alpha == 0) ? 2.0L : 4.0L / 3.0L;
    int idx[kMaxN];
    for (int i = 0; i < m; ++i) idx[i] = i;
    std::sort(idx, idx + m, [&](int a, int b) { return A[a][a] < A[b][b]; });
    for (int i = 0; i < m; ++i) {
        x[i] = A[idx[i]][idx[i]];
        w[i] = mu0 * V[0][idx[i]] * V[0][idx[i]];
    }
    // the rules are symmetric: average the mirrored pairs
    for (int i = 0; i < m / 2; ++i) {
        real xm = 0.5L * (x[m - 1 - i] - x[i]), wm = 0.5L * (w[i] + w[m - 1 - i]);
        x[i] = -xm; x[m - 1 - i] = xm;
        w[i] = w[m - 1 - i] = wm;
    }
    if (m % 2 == 1) x[m / 2] = 0.0L;
}

}  // namespace

void build_tables(int p, Tables1D* t)
{
    const int n = p + 1;
    t->p = p;
    t->n = n;
    real gx[kMaxN], gw[kMaxN], lx[kMaxN], lw[kMaxN];
    golub_welsch(n, 0, gx, gw);  // Gauss-Legendre, n_q = p+1 (R1)
    // GLL: +-1 and the p-1 Gauss-Jacobi(1,1) points; interior weight = Jacobi weight / (1-x^2); end weight 2/(p(p+1))
    lx[0] = -1.0L; lx[p] = 1.0L;
    lw[0] = lw[p] = 2.0L / ((real)p * (p + 1));
    if (p > 1) {
        real jx[kMaxN], jw[kMaxN];
        golub_welsch(p - 1, 1, jx, jw);
        for (int i = 0; i < p - 1; ++i) {
            lx[i + 1] = jx[i];
            lw[i + 1] = jw[i] / (1.0L - jx[i] * jx[i]);
        }
    }
    for (int i = 0; i < n; ++i) {
        t->gll_x[i] = (double)lx[i]; t->gll_w[i] = (double)lw[i];
        t->gl_x[i] = (double)gx[i]; t->gl_w[i] = (double)gw[i];
    }
    // barycentric weights of the GLL nodes and of the Gauss points
    real bl[kMaxN], bg[kMaxN];
    for (int a = 0; a < n; ++a) {
        real pl = 1.0L, pg = 1.0L;
        for (int j = 0; j < n; ++j)
            if (j != a) { pl *= (lx[a] - lx[j]); pg *= (gx[a] - gx[j]); }
        bl[a] = 1.0L / pl;
        bg[a] = 1.0L / pg;
    }
    // N[q][a] = l_a(gx[q]) (Eq. 12 in barycentric form); the centre point coincides with a node when p is even
    for (int q = 0; q < n; ++q) {
        int hit = -1;
        for (int j = 0; j < n; ++j)
            if (gx[q] == lx[j]) hit = j;
        if (hit >= 0) {
            for (int a = 0; a < n; ++a) t->N[q * n + a] = (a == hit) ? 1.0 : 0.0;
            continue;
        }
        real den = 0.0L;
        for (int j = 0; j < n; ++j) den += bl[j] / (gx[q] - lx[j]);
        for (int a = 0; a < n; ++a) t->N[q * n + a] = (double)((bl[a] / (gx[q] - lx[a])) / den);
    }
    // collocation derivative on the Gauss points: D[s][q] = l^_q'(gx[s])
    real D[kMaxN][kMaxN];
    for (int s = 0; s < n; ++s) {
        real diag = 0.0L;
        for (int q = 0; q < n; ++q)
            if (q != s) {
                D[s][q] = (bg[q] / bg[s]) / (gx[s] - gx[q]);
                diag -= D[s][q];
            }
        D[s][s] = diag;
    }
    for (int s = 0; s < n; ++s)
        for (int q = 0; q < n; ++q) t->D[s * n + q] = (double)D[s][q];
    for (int q = 0; q < n; ++q)
        for (int r = 0; r < n; ++r) {
            real g = 0.0L;
            for (int s = 0; s < n; ++s) g += gw[s] * D[s][q] * D[s][r];
            t->G[q * n + r] = (double)g;
        }
}

void lagrange_gll(const Tables1D& t, double x, double* out)
{
    const int n = t.n;
    for (int j = 0; j < n; ++j)
        if (x == t.gll_x[j]) {
            for (int a = 0; a < n; ++a) out[a] = (a == j) ? 1.0 : 0.0;
            return;
        }
    real b[kMaxN], den = 0.0L;
    for (int a = 0; a < n; ++a) {
        real pr = 1.0L;
        for (int j = 0; j < n; ++j)
            if (j != a) pr *= ((real)t.gll_x[a] - (real)t.gll_x[j]);
        b[a] = 1.0L / (pr * ((real)x - (real)t.gll_x[a]));
        den += b[a];
    }
    for (int a = 0; a < n; ++a) out[a] = (double)(b[a] / den);
}

}  // namespace fecheb
