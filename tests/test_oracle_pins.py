"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage or closed form it pins: a plausible mistake in the oracle (dropped term, wrong sign or
index, transposed operand, wrong quadrature weight) fails at least one of them.
"""
import os

import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla
from numpy.polynomial import Polynomial

import oracle
import workloads


def _read(golden_dir, name):
    rows = []
    with open(os.path.join(golden_dir, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


def _mesh(edges, p, V=None, assemble=True):
    m = oracle.OracleMesh(*edges, p)
    Vq = np.zeros(m.ncells * m.nq3) if V is None else V(m.quad_coords())
    m.set_potential(Vq)
    if assemble:
        m.assemble()
    return m


def _csr(m, scaled=True):
    rp, col, val = m.csr(scaled)
    return sp.csr_matrix((val, col, rp), shape=(m.N, m.N))


UNEQUAL = (np.array([0.0, 0.7, 2.0]), np.array([-1.0, -0.5, 0.4, 1.0]), np.array([0.0, 0.3, 1.0, 1.2, 2.5]))


# ---- 1-D rules and Eq. 12 -----------------------------------------------------------------------------------
def test_gll_closed_forms(golden_dir):
    for p, x, w in _read(golden_dir, "gll_rules.txt"):
        p, x, w = int(p), float(x), float(w)
        xs, ws = oracle.gll(p)
        i = int(np.argmin(np.abs(xs - x)))
        assert abs(xs[i] - x) < 5e-15 and abs(ws[i] - w) < 5e-15
        assert abs(xs[p - i] + x) < 5e-15 and abs(ws[p - i] - w) < 5e-15


@pytest.mark.parametrize("p", range(1, 9))
def test_rules_exactness(p):
    """GLL is exact to degree 2p-1, Gauss (p+1 points) to 2p+1; one degree more is not (R1)."""
    xs, ws = oracle.gll(p)
    xg, wg = oracle.gauss(p + 1)
    assert abs(ws.sum() - 2) < 1e-14 and abs(wg.sum() - 2) < 1e-14
    assert np.all(np.diff(xs) > 0) and np.all(np.diff(xg) > 0) and xs[0] == -1 and xs[-1] == 1
    for k in range(0, 2 * p + 3):
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        if k <= 2 * p - 1:
            assert abs(ws @ xs**k - exact) < 1e-14
        if k <= 2 * p + 1:
            assert abs(wg @ xg**k - exact) < 1e-14
    assert abs(ws @ xs ** (2 * p) - 2.0 / (2 * p + 1)) > 1e-6
    assert abs(wg @ xg ** (2 * p + 2) - 2.0 / (2 * p + 3)) > 1e-8


@pytest.mark.parametrize("p", [1, 2, 4, 6, 8])
def test_lagrange_eq12(p):
    """Eq. 12: l_a(x_b) = delta_ab, reproduces polynomials of degree <= p, derivative too."""
    xs, _ = oracle.gll(p)
    for a in range(p + 1):
        for b in range(p + 1):
            assert abs(oracle.lagrange(xs, a, xs[b]) - (a == b)) < 1e-14
    for x in (-0.93, -0.2, 0.41, 0.77):
        for k in range(p + 1):
            v = sum(xs[a] ** k * oracle.lagrange(xs, a, x) for a in range(p + 1))
            d = sum(xs[a] ** k * oracle.lagrange_deriv(xs, a, x) for a in range(p + 1))
            assert abs(v - x**k) < 1e-13
            assert abs(d - (k * x ** (k - 1) if k else 0.0)) < 5e-12


# ---- mesh tables --------------------------------------------------------------------------------------------
def test_l2g_brute_force():
    """Reading R3 against brute force: nodes are identified by their coordinates."""
    p = 2
    m = oracle.OracleMesh(*UNEQUAL, p)
    l2g, xyz, mask = m.l2g(), m.node_coords(), m.mask()
    cx, cy, cz = 2, 3, 4
    assert m.N == (cx * p + 1) * (cy * p + 1) * (cz * p + 1) and len(np.unique(l2g)) == m.N
    xs = np.array([-1.0, 0.0, 1.0])  # closed-form GLL p=2
    seen = {}
    for e in range(m.ncells):
        ex, ey, ez = e % cx, (e // cx) % cy, e // (cx * cy)
        for a in range(27):
            ax, ay, az = a % 3, (a // 3) % 3, a // 9
            c = []
            for edges, ec, aa in ((UNEQUAL[0], ex, ax), (UNEQUAL[1], ey, ay), (UNEQUAL[2], ez, az)):
                c.append(edges[ec] + 0.5 * (xs[aa] + 1) * (edges[ec + 1] - edges[ec]))
            g = l2g[e, a]
            assert np.allclose(xyz[g], c, atol=1e-14)
            key = tuple(np.round(c, 10))
            assert seen.setdefault(key, g) == g  # same point <-> same id
    assert len(seen) == m.N
    lo, hi = [u[0] for u in UNEQUAL], [u[-1] for u in UNEQUAL]
    on_bnd = np.any((np.abs(xyz - lo) < 1e-13) | (np.abs(xyz - hi) < 1e-13), axis=1)
    assert np.array_equal(mask, (~on_bnd).astype(np.uint8))
    assert mask.sum() == m.N_free == (cx * p - 1) * (cy * p - 1) * (cz * p - 1)
    # x fastest
    assert l2g[0, 1] == l2g[0, 0] + 1 and l2g[1, 0] == l2g[0, 2]


def test_coords_r4():
    m = oracle.OracleMesh(*UNEQUAL, 3)
    xyz, l2g = m.node_coords(), m.l2g()
    # last local node of a cell sits exactly on the upper edge, first on the lower one
    assert xyz[l2g[0, 0], 0] == UNEQUAL[0][0] and xyz[l2g[0, 3], 0] == UNEQUAL[0][1]
    q = m.quad_coords().reshape(m.ncells, 4, 4, 4, 3)
    xg, _ = oracle.gauss(4)
    assert np.allclose(q[0, 0, 0, :, 0], 0.35 * (xg + 1), atol=1e-15)
    assert np.allclose(q[0, :, 0, 0, 2], 0.15 * (xg + 1), atol=1e-15)


@pytest.mark.parametrize("p", [2, 3])
def test_mass(p):
    """l.185: GLL-lumped mass; sum = volume; equals the row sums of the Gauss-integrated mass matrix (V == 1)."""
    m = oracle.OracleMesh(*UNEQUAL, p)
    M = m.mass()
    vol = np.prod([u[-1] - u[0] for u in UNEQUAL])
    assert abs(M.sum() - vol) < 1e-13 * vol
    m.set_potential(np.ones(m.ncells * m.nq3))
    l2g = m.l2g()
    rows = np.zeros(m.N)
    for e in range(m.ncells):
        MV = m.cell_matrix(e, np.ones(m.nq3), kin=0.0, pot=1.0)
        np.add.at(rows, l2g[e], MV.sum(axis=1))
    assert np.max(np.abs(rows - M)) < 1e-14


def test_config1_volume():
    w = workloads.config(1)
    m = oracle.OracleMesh(w.xe, w.ye, w.ze, w.p)
    assert abs(m.mass().sum() - 1728.0) < 1e-10 and m.N == 729 and m.N_free == 343


# ---- stiffness ----------------------------------------------------------------------------------------------
def test_trilinear_laplacian(golden_dir):
    e = np.array([0.0, 1.0])
    m = oracle.OracleMesh(e, e, e, 1)
    K = m.cell_matrix(0, None, kin=1.0, pot=0.0)
    expect = {int(k): float(v) for k, v in _read(golden_dir, "trilinear_laplacian.txt")}
    for a in range(8):
        for b in range(8):
            ndiff = bin(a ^ b).count("1")
            assert abs(K[a, b] - expect[ndiff]) < 1e-15
    K1, M1 = np.array([[1.0, -1.0], [-1.0, 1.0]]), np.array([[1 / 3, 1 / 6], [1 / 6, 1 / 3]])
    Kt = np.kron(M1, np.kron(M1, K1)) + np.kron(M1, np.kron(K1, M1)) + np.kron(K1, np.kron(M1, M1))
    assert np.max(np.abs(K - Kt)) < 1e-15


def _exact_1d(p):
    """1-D stiffness and mass of the GLL Lagrange basis on [-1,1] by EXACT polynomial integration (numpy)."""
    xs, _ = oracle.gll(p)
    L = []
    for a in range(p + 1):
        poly = Polynomial([1.0])
        for j in range(p + 1):
            if j != a:
                poly = poly * Polynomial([-xs[j], 1.0]) / (xs[a] - xs[j])
        L.append(poly)
    K1, M1 = np.empty((p + 1, p + 1)), np.empty((p + 1, p + 1))
    for a in range(p + 1):
        for b in range(p + 1):
            ik = (L[a].deriv() * L[b].deriv()).integ()
            im = (L[a] * L[b]).integ()
            K1[a, b], M1[a, b] = ik(1.0) - ik(-1.0), im(1.0) - im(-1.0)
    return K1, M1


@pytest.mark.parametrize("p", [2, 3, 4])
def test_cell_matrix_kronecker(p):
    """Eq. 17 on an axis-aligned box separates: K_e = sum_d (h/2 factors) K1 (x) M1 (x) M1 with exactly integrated
    1-D matrices; a constant V gives V * M1 (x) M1 (x) M1.  Unequal edge lengths catch axis-order mistakes."""
    m = oracle.OracleMesh(np.array([0.0, 0.7]), np.array([0.0, 1.3]), np.array([0.0, 0.4]), p)
    hx, hy, hz = 0.7, 1.3, 0.4
    K1, M1 = _exact_1d(p)
    Kx, Mx = K1 * 2 / hx, M1 * hx / 2
    Ky, My = K1 * 2 / hy, M1 * hy / 2
    Kz, Mz = K1 * 2 / hz, M1 * hz / 2
    # local index a = ax + n (ay + n az): z is the slowest -> leftmost Kronecker factor
    Kt = np.kron(Mz, np.kron(My, Kx)) + np.kron(Mz, np.kron(Ky, Mx)) + np.kron(Kz, np.kron(My, Mx))
    Mt = np.kron(Mz, np.kron(My, Mx))
    K = m.cell_matrix(0, None, kin=1.0, pot=0.0)
    MV = m.cell_matrix(0, 2.5 * np.ones(m.nq3), kin=0.0, pot=1.0)
    H = m.cell_matrix(0, 2.5 * np.ones(m.nq3))
    assert np.max(np.abs(K - Kt)) < 2e-13 * np.max(np.abs(Kt))
    assert np.max(np.abs(MV - 2.5 * Mt)) < 1e-14
    assert np.max(np.abs(H - (0.5 * Kt + 2.5 * Mt))) < 2e-13 * np.max(np.abs(Kt))


def test_potential_is_quadrature_defined():
    """R1: M_V is DEFINED by the Gauss rule: M_V[a,b] = sum_q J w_q V_q Phi_a(q) Phi_b(q); check against a direct
    numpy einsum with independently tabulated basis values, for a non-constant V and a non-cubic cell."""
    p = 3
    m = oracle.OracleMesh(np.array([0.0, 0.5]), np.array([1.0, 2.0]), np.array([-1.0, 1.0]), p)
    xs, _ = oracle.gll(p)
    xg, wg = oracle.gauss(p + 1)
    phi = np.array([[oracle.lagrange(xs, a, x) for a in range(p + 1)] for x in xg])  # [q][a]
    rng = np.random.default_rng(5)
    V = rng.normal(size=(p + 1, p + 1, p + 1))  # [qz][qy][qx]
    J = 0.5 * 1.0 * 2.0 / 8
    W = J * np.einsum("k,j,i->kji", wg, wg, wg) * V
    P3 = np.einsum("kc,jb,ia->kjicba", phi, phi, phi).reshape(p + 1, p + 1, p + 1, -1)  # [qz,qy,qx][a]
    ref = np.einsum("kji,kjia,kjib->ab", W, P3, P3)
    MV = m.cell_matrix(0, V.reshape(-1), kin=0.0, pot=1.0)
    assert np.max(np.abs(MV - ref)) < 1e-14


def test_stiffness_invariants():
    """K.1 = 0 (partition of unity); (K u)_a = -6 M_aa for u = x^2+y^2+z^2 at interior nodes (-1/2 lap is what
    1/2 K discretises, Eq. 17); H symmetric; sum of cells == assembled matrix (l.237, l.253)."""
    p = 3
    m = _mesh(UNEQUAL, p)
    # raw assembled H with V=0 is K/2
    H = _csr(m, scaled=False)
    K = 2.0 * H
    scale = abs(K).max()
    assert abs(K @ np.ones(m.N)).max() < 1e-12 * scale
    xyz, M, mask = m.node_coords(), m.mass(), m.mask().astype(bool)
    u = (xyz**2).sum(axis=1)
    assert np.max(np.abs((K @ u)[mask] + 6.0 * M[mask])) < 1e-11 * scale
    assert abs(H - H.T).max() < 1e-13 * scale
    # sum of cells, assembled densely in numpy through l2g
    l2g = m.l2g()
    D = np.zeros((m.N, m.N))
    for e in range(m.ncells):
        D[np.ix_(l2g[e], l2g[e])] += m.He[e]
    assert np.max(np.abs(D - H.toarray())) < 1e-13 * scale


def test_scaled_operator_and_applies():
    """Eq. 19-20: H~ = M^-1/2 H M^-1/2 on free nodes; boundary rows/columns zero; CSR apply == cell-wise apply ==
    row-sampled apply; the shift multiplies the identity."""
    p = 2
    m = _mesh(UNEQUAL, p, V=lambda q: -1.0 / np.sqrt((q**2).sum(axis=1) + 0.25))
    H, Ht = _csr(m, False).toarray(), _csr(m, True).toarray()
    s, mask = 1 / np.sqrt(m.mass()), m.mask().astype(bool)
    ref = (s[:, None] * H * s[None, :]) * np.outer(mask, mask)
    assert np.max(np.abs(Ht - ref)) < 1e-13 * np.max(np.abs(ref))
    assert np.max(np.abs(Ht - Ht.T)) < 1e-13 * np.max(np.abs(ref))
    B = 5
    X = workloads.random_block(11, m.N, B)  # boundary rows NOT zeroed: they must be ignored
    eps = workloads.shifts(12, B)
    Y0 = m.apply(X)
    assert np.max(np.abs(Y0 - Ht @ X)) < 1e-12 * np.max(np.abs(Y0))
    assert np.all(Y0[~mask] == 0)
    Y1 = m.apply(X, eps)
    assert np.max(np.abs(Y1 - (Ht @ X - mask[:, None] * X * eps[None, :]))) < 1e-12 * np.max(np.abs(Y0))
    Yc = m.apply(X, eps, cellwise=True)
    assert np.max(np.abs(Yc - Y1)) < 1e-12 * np.max(np.abs(Y0))
    Yt = m.apply(X, eps, nthreads=4)
    assert np.array_equal(Yt, Y1)
    rows = np.array([0, 7, 100, 233, m.N - 1, 152, 200, 41])
    Yr = m.apply_rows(X, rows, eps)
    assert np.max(np.abs(Yr - Y1[rows])) < 1e-12 * np.max(np.abs(Y0))


# ---- spectrum -----------------------------------------------------------------------------------------------
def _lowest(m, k):
    A = _csr(m, True)
    free = np.flatnonzero(m.mask())
    A = A[free][:, free].tocsc()
    vals = spla.eigsh(A, k=k, sigma=0.0, which="LM", return_eigenvectors=False)
    return np.sort(vals)


def test_harmonic_oscillator_levels(golden_dir):
    """BASELINE.json north_star: eigenvalues 1.5, 2.5 (x3), 3.5 (x6) converging with p ([-6,6]^3, 4^3 cells)."""
    levels = []
    for lv, deg in _read(golden_dir, "harmonic_levels.txt"):
        levels += [float(lv)] * int(deg)
    levels = np.array(levels)
    e = workloads.uniform_edges(-6.0, 6.0, 4)
    errs = []
    for p in (2, 3, 4, 5):
        m = _mesh((e, e, e), p, V=workloads.harmonic)
        k = 10 if p >= 4 else 4
        lam = _lowest(m, k)
        errs.append(np.max(np.abs(lam[:4] - levels[:4])))
        if p == 5:
            assert np.max(np.abs(lam - levels)) < 2e-2
    assert errs[0] > errs[2] and errs[1] > errs[3] and errs[3] < 5e-3, errs


def test_config1_spectrum(golden_dir):
    """spectrum of H~ for config 1 from the surveyor's independent probe."""
    w = workloads.config(1)
    m = _mesh((w.xe, w.ye, w.ze), w.p, V=w.V)
    free = np.flatnonzero(m.mask())
    lam = np.linalg.eigvalsh(_csr(m).toarray()[np.ix_(free, free)])
    expect_low, lam_max = [], None
    for kind, v, deg in _read(golden_dir, "cfg1_spectrum.txt"):
        if kind == "low":
            expect_low += [float(v)] * int(deg)
        else:
            lam_max = float(v)
    assert np.max(np.abs(lam[:len(expect_low)] - expect_low)) < 2e-11
    assert abs(lam[-1] - lam_max) < 1e-10


# ---- filter, Lanczos, Rayleigh-Ritz -------------------------------------------------------------------------
def _cheb_T(m, x):
    x = np.asarray(x, dtype=np.float64)
    out = np.empty_like(x)
    inside = np.abs(x) <= 1
    out[inside] = np.cos(m * np.arccos(x[inside]))
    xo = x[~inside]
    out[~inside] = np.sign(xo) ** m * np.cosh(m * np.arccosh(np.abs(xo)))
    return out


def test_filter_closed_form():
    """l.210: Y = T_m(Hbar) X.  On config 1 compare the recurrence with U T_m((L-c)/e)/T_m(x0) U^T X from LAPACK."""
    w = workloads.config(1)
    m = _mesh((w.xe, w.ye, w.ze), w.p, V=w.V)
    mask = m.mask()
    free = np.flatnonzero(mask)
    lam, U = np.linalg.eigh(_csr(m).toarray()[np.ix_(free, free)])
    X = w.X(mask)
    th_min, th_max, beta = oracle.lanczos_bounds(m, workloads.normal(3001, m.N), 20)
    assert th_min >= lam[0] - 1e-10 and th_max <= lam[-1] + 1e-10 and th_max + beta >= lam[-1]
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    for deg in (1, 2, 3, w.m):
        Y = m.filter(X, deg, a, b, a0)
        e, c = (b - a) / 2, (b + a) / 2
        rho = _cheb_T(deg, (lam - c) / e) / _cheb_T(deg, np.array([(a0 - c) / e]))[0]
        ref = np.zeros_like(X)
        ref[free] = U @ (rho[:, None] * (U.T @ X[free]))
        assert np.linalg.norm(Y - ref) < 1e-12 * np.linalg.norm(ref), deg
        assert np.all(Y[mask == 0] == 0)
    with pytest.raises(ValueError):
        m.filter(X, 3, b, a, a0)


@pytest.mark.parametrize("k", [1, 2, 6])
def test_lanczos_is_the_krylov_projection(k):
    """Reading R10 pins lanczos_bounds to what the mathematics fixes: in exact arithmetic the Lanczos vectors are the
    Gram-Schmidt basis of the Krylov space, so with Q from a Householder QR of [v, H~v, ..., H~^k v] (column signs made
    positive) alpha_i = (Q^T H~ Q)_ii, beta_i = (Q^T H~ Q)_{i+1,i} > 0, the returned beta is the LAST of them (the
    coupling to the (k+1)-th vector = norm of the last residual), and theta = eig of the leading k x k block.  A dropped
    `- beta v_prev`, a shifted off-diagonal or a wrong returned beta fails this; k <= 6 keeps the monomial Krylov basis
    well enough conditioned for 1e-9 on config 1's 343 x 343 operator."""
    w = workloads.config(1)
    m = _mesh((w.xe, w.ye, w.ze), w.p, V=w.V)
    mask = m.mask()
    free = np.flatnonzero(mask)
    H = _csr(m).toarray()[np.ix_(free, free)]
    v0 = workloads.normal(3001, m.N)
    v = v0[free] / np.linalg.norm(v0[free])
    K = np.empty((len(free), k + 1))
    K[:, 0] = v
    for i in range(k):
        K[:, i + 1] = H @ K[:, i]
        K[:, i + 1] /= np.linalg.norm(K[:, i + 1])  # column scaling changes R, not Q
    Q, R = np.linalg.qr(K)
    Q = Q * np.sign(np.diag(R))[None, :]
    T = Q.T @ H @ Q  # (k+1) x (k+1), tridiagonal up to rounding
    lo, hi, beta, alphas, betas = oracle.lanczos_bounds(m, v0, k, return_tridiagonal=True)
    scale = np.abs(H).sum(axis=1).max()
    assert len(alphas) == k and len(betas) == k
    assert np.max(np.abs(alphas - np.diag(T)[:k])) <= 1e-9 * scale
    assert np.max(np.abs(betas - np.diag(T, -1)[:k])) <= 1e-9 * scale
    assert np.all(np.diag(T, -1)[:k] > 0)
    assert beta == betas[-1] and abs(beta - T[k, k - 1]) <= 1e-9 * scale
    theta = np.linalg.eigvalsh(T[:k, :k])
    assert abs(lo - theta[0]) <= 1e-9 * scale and abs(hi - theta[-1]) <= 1e-9 * scale
    # what is outside the tridiagonal band vanishes (three-term recurrence = symmetry of H~)
    assert np.max(np.abs(np.triu(T[:k, :k], 2))) <= 1e-9 * scale
    # and the interval [theta_min, theta_max + beta] the filter uses still brackets as before
    lam = np.linalg.eigvalsh(H)
    assert lo >= lam[0] - 1e-10 and hi <= lam[-1] + 1e-10


def test_filter_cellwise_equals_csr():
    w = workloads.reduced(2, 2)
    m = _mesh((w.xe, w.ye, w.ze), 2, V=w.V)
    X = workloads.random_block(21, m.N, 3, m.mask())
    Y1 = m.filter(X, 7, 0.5, 40.0, -3.0)
    Y2 = m.filter(X, 7, 0.5, 40.0, -3.0, cellwise=True)
    assert np.linalg.norm(Y1 - Y2) < 1e-12 * np.linalg.norm(Y1)


def test_rayleigh_ritz():
    """Eq. 23-24 (R8, R9): Q orthonormal; Ritz values >= the matching eigenvalues (Cauchy interlacing); a few
    filter + RR cycles converge to the lowest eigenvalues of H~."""
    w = workloads.config(1)
    m = _mesh((w.xe, w.ye, w.ze), w.p, V=w.V)
    mask = m.mask()
    free = np.flatnonzero(mask)
    lam = np.linalg.eigvalsh(_csr(m).toarray()[np.ix_(free, free)])
    X = w.X(mask)
    th_min, th_max, beta = oracle.lanczos_bounds(m, workloads.normal(3001, m.N), 20)
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    for _ in range(6):
        Y = m.filter(X, 10, a, b, a0)
        theta, X, Q = oracle.rayleigh_ritz(m, Y)
        assert np.max(np.abs(Q.T @ Q - np.eye(w.B))) < 1e-13
        assert np.all(theta >= lam[:w.B] - 1e-11)
        a, a0 = theta[-1], theta[0]
    assert np.max(np.abs(theta[:4] - lam[:4])) < 1e-6
    # shifted apply of a converged Ritz pair has norm = its residual (l.221: (H~ - eps) is singular there)
    R = m.apply(X, theta)
    assert np.linalg.norm(R[:, 0]) < 1e-4


def test_ritz_residuals_and_residual_controlled_chfsi():
    """l.296: the eigenproblem residual || H~ x - theta x || is driven below t_eig.  Pins, on config 1's dense H~ through
    LAPACK: (i) exact eigenpairs have residual 0; (ii) for any unit vector with its Rayleigh quotient,
    ||H x - theta x||^2 = x^T H^2 x - theta^2; (iii) Bauer-Fike for symmetric matrices: every Ritz value lies within its
    residual norm of an eigenvalue; (iv) the residual-controlled loop stops at the first cycle whose gate residuals are
    <= t_eig (it reproduces a hand-rolled fixed-count loop) and its lowest values are then eigenvalues to residual^2 / gap."""
    w = workloads.config(1)
    m = _mesh((w.xe, w.ye, w.ze), w.p, V=w.V)
    mask = m.mask()
    free = np.flatnonzero(mask)
    H = _csr(m).toarray()[np.ix_(free, free)]
    lam, U = np.linalg.eigh(H)
    Xe = np.zeros((m.N, 5))
    Xe[free] = U[:, :5]
    assert np.max(oracle.ritz_residuals(m, Xe, lam[:5])) < 1e-12
    x = workloads.normal(77, m.N) * mask
    x /= np.linalg.norm(x)
    th = x[free] @ H @ x[free]
    r = oracle.ritz_residuals(m, x[:, None], [th])[0]
    assert abs(r ** 2 - (x[free] @ H @ (H @ x[free]) - th ** 2)) < 1e-10 * r ** 2
    th_min, th_max, beta = oracle.lanczos_bounds(m, workloads.normal(3001, m.N), 20)
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    X0 = w.X(mask)
    theta, X, res, cycles = oracle.chfsi(m, X0, 10, a, b, a0, t_eig=1e-6, n_gate=4, max_cycles=40)
    assert 1 < cycles < 40 and res[:4].max() <= 1e-6
    for t, rj in zip(theta, res):
        assert np.min(np.abs(lam - t)) <= rj * (1 + 1e-8) + 1e-13
    assert np.max(np.abs(theta[:4] - lam[:4])) < 1e-10
    # the same cycles by hand: the loop stopped exactly at the first cycle that met the gate
    Xh, ah, a0h = X0, a, a0
    for c in range(cycles):
        th_h, Xh, _ = oracle.rayleigh_ritz(m, m.filter(Xh, 10, ah, b, a0h))
        rh = oracle.ritz_residuals(m, Xh, th_h)
        assert (rh[:4].max() <= 1e-6) == (c == cycles - 1)
        ah, a0h = th_h[-1], th_h[0]
    assert np.array_equal(th_h, theta)


# ---- MINRES of the adjoint solve (l.221-225) -------------------------------------------------------------------------
def test_minres_against_dense_solves():
    """The oracle's MINRES is pinned to LAPACK: a regular shifted system against numpy.linalg.solve, and the singular
    system of l.221 ((H~ - theta_k) with g orthogonal to the null vector) against the pseudo-inverse solution, which is
    the component p_perp the paper's Krylov argument singles out.  The preconditioner against the CSR diagonal."""
    w = workloads.config(1)
    m = _mesh((w.xe, w.ye, w.ze), w.p, w.V)
    free = m.mask().astype(bool)
    A = _csr(m).toarray()[np.ix_(free, free)]
    lam, U = np.linalg.eigh(A)
    # preconditioner = inverse diagonal of the mass-scaled (1/2)K: compare with the CSR of the potential-free operator
    m0 = _mesh((w.xe, w.ye, w.ze), w.p, lambda q: np.zeros(len(q)))
    K = _csr(m0).toarray()
    Mi = oracle.laplacian_precond(m)
    assert np.allclose(Mi[free], 1.0 / np.diag(K)[free], rtol=1e-13) and np.all(Mi[~free] == 0) and np.all(Mi[free] > 0)
    B = 4
    G = workloads.random_block(77, m.N, B, m.mask())
    eps = np.array([-1.0, 0.3, 2.2, 5.1])  # inside the spectrum: indefinite systems
    for Minv in (None, Mi):
        X, rel, it = oracle.minres_shifted(m, G, eps, maxit=2000, tol=1e-13, Minv=Minv)
        for j in range(B):
            xref = np.linalg.solve(A - eps[j] * np.eye(A.shape[0]), G[free, j])
            assert np.linalg.norm(X[free, j] - xref) <= 1e-8 * np.linalg.norm(xref), (j, it)
        assert np.all(X[~free] == 0)
    # singular case: eps = a (3-fold degenerate) eigenvalue, g orthogonal to its null vectors Psi_k
    k = 3
    Psi = U[:, np.abs(lam - lam[k]) < 1e-8]
    assert Psi.shape[1] == 3
    Gs = G[:, :1].copy()
    Gs[free, 0] -= Psi @ (Psi.T @ Gs[free, 0])
    Xs, rel, it = oracle.minres_shifted(m, Gs, np.array([lam[k]]), maxit=2000, tol=1e-10)
    xp = np.linalg.pinv(A - lam[k] * np.eye(A.shape[0]), rcond=1e-10) @ Gs[free, 0]
    assert np.linalg.norm(Xs[free, 0] - xp) <= 1e-7 * np.linalg.norm(xp)
    assert np.max(np.abs(Psi.T @ Xs[free, 0])) <= 1e-7 * np.linalg.norm(xp)  # p_perp is orthogonal to the null vectors


# ---- density at the quadrature points (Eq. 4) -----------------------------------------------------------------------
def _bubble_fields(xyz, edges):
    """Two polynomials of degree <= 3 per variable that vanish on the box surface (exactly representable at p >= 3)."""
    (x0, x1), (y0, y1), (z0, z1) = [(e[0], e[-1]) for e in edges]
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    bub = (x - x0) * (x1 - x) * (y - y0) * (y1 - y) * (z - z0) * (z1 - z)
    return np.stack([bub * (1.0 + 0.3 * x - 0.2 * y + 0.5 * z), bub * (0.7 - 0.4 * x * y + 0.1 * z)], axis=1)


def test_density_polynomial_closed_form():
    """Eq. 4: rho(x_q) = sum_j f_j psi_j(x_q)^2.  For psi in the FE space (polynomials of degree <= p per variable that
    satisfy the Dirichlet condition) interpolation is exact, so the oracle must return f . psi(x_q)^2 evaluated from
    the closed form at the quadrature coordinates; and int rho = sum_q J w_q rho_q integrates psi^2 exactly."""
    m = oracle.OracleMesh(*UNEQUAL, 3)
    psi_nodes = _bubble_fields(m.node_coords(), UNEQUAL)
    X = psi_nodes * np.sqrt(m.mass())[:, None]  # psi~ = M^{1/2} psi (Eq. 19)
    f = np.array([2.0, 0.5])
    rho = oracle.density(m, X, f)
    ref = (_bubble_fields(m.quad_coords(), UNEQUAL) ** 2) @ f
    assert np.max(np.abs(rho.reshape(-1) - ref)) <= 1e-13 * np.max(np.abs(ref))
    # the integral with p+1 Gauss points is exact for degree 2p+1 = 7 > 6: compare with the analytic integral of the
    # first field's square computed by high-order 1-D Gauss rules on the whole box
    xq, wq = np.polynomial.legendre.leggauss(12)
    pts, wts = [], []
    for e in UNEQUAL:
        a, b = e[0], e[-1]
        pts.append(0.5 * (b - a) * xq + 0.5 * (a + b))
        wts.append(0.5 * (b - a) * wq)
    Xg, Yg, Zg = np.meshgrid(*pts, indexing="ij")
    Wg = wts[0][:, None, None] * wts[1][None, :, None] * wts[2][None, None, :]
    grid = np.stack([Xg.ravel(), Yg.ravel(), Zg.ravel()], axis=1)
    exact = ((_bubble_fields(grid, UNEQUAL) ** 2) @ f * Wg.ravel()).sum()
    n = m.p + 1
    gx, gw = oracle.gauss(n)
    hx, hy, hz = (np.diff(e) for e in UNEQUAL)
    cx, cy = len(hx), len(hy)
    total = 0.0
    for e in range(m.ncells):
        ex, ey, ez = e % cx, (e // cx) % cy, e // (cx * cy)
        J = hx[ex] * hy[ey] * hz[ez] / 8.0
        w3 = (gw[None, None, :] * gw[None, :, None] * gw[:, None, None]).reshape(-1)  # q = qx + n(qy + n qz)
        total += J * (w3 * rho[e]).sum()
    assert abs(total - exact) <= 1e-12 * abs(exact)


def test_adjoint_rhs_weak_form():
    """Eq. 18: sum_a c_a g_a^{(i)} = int f_i U psi_i phi - sum_j (D+D^T)_ij int psi_j phi for phi = sum_a c_a N_a.  With
    polynomial psi, phi (degree <= 3 per variable, zero on the boundary) and linear U the first integrand has degree 7 =
    2p+1 at p = 3: the p+1 Gauss points integrate it exactly, so it must equal a 12-point reference integral of the
    closed forms; the second term is the lumped GLL mass inner product (l.185)."""
    m = oracle.OracleMesh(*UNEQUAL, 3)
    xyz = m.node_coords()
    fields = _bubble_fields(xyz, UNEQUAL)
    psi_nodes, phi_nodes = fields[:, :1], fields[:, 1]
    sqrtM = np.sqrt(m.mass())
    U = lambda q: 1.0 + 0.5 * q[:, 0] - 0.25 * q[:, 1] + 0.125 * q[:, 2]
    f = np.array([1.7])
    D = np.array([[0.3]])
    gt = oracle.adjoint_rhs(m, psi_nodes * sqrtM[:, None], f, U(m.quad_coords()), D)
    lhs = float((gt[:, 0] * sqrtM) @ phi_nodes)  # g = M^{1/2} g~ ; sum_a c_a g_a
    xq, wq = np.polynomial.legendre.leggauss(12)
    pts, wts = [], []
    for e in UNEQUAL:
        a, b = e[0], e[-1]
        pts.append(0.5 * (b - a) * xq + 0.5 * (a + b))
        wts.append(0.5 * (b - a) * wq)
    Xg, Yg, Zg = np.meshgrid(*pts, indexing="ij")
    Wg = (wts[0][:, None, None] * wts[1][None, :, None] * wts[2][None, None, :]).ravel()
    grid = np.stack([Xg.ravel(), Yg.ravel(), Zg.ravel()], axis=1)
    F = _bubble_fields(grid, UNEQUAL)
    first = f[0] * float((U(grid) * F[:, 0] * F[:, 1] * Wg).sum())
    second = (D + D.T)[0, 0] * float((m.mass() * psi_nodes[:, 0]) @ phi_nodes)  # lumped mass: int psi phi ~ psi^T M phi
    assert abs(lhs - (first - second)) <= 1e-11 * max(abs(first), abs(second))


# ---- inputs module ------------------------------------------------------------------------------------------
def test_inputs_generator():
    z = workloads.splitmix64(0, 0, 3)
    # splitmix64(seed=0) reference outputs (public-domain generator by S. Vigna, first three values)
    assert [int(v) for v in z] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    x = workloads.normal(7, 200001)
    assert abs(x.mean()) < 0.01 and abs(x.std() - 1) < 0.01
    assert np.array_equal(workloads.normal(7, 11, start=1001), x[1001:1012])
    e = workloads.graded_edges()
    h = np.diff(e)
    assert len(e) == 41 and e[0] == -15 and e[-1] == 15 and np.allclose(e, -e[::-1])
    assert abs(h.min() - 0.2 * 0.88151901) < 1e-6 and abs(h.max() - 1.5 * 0.88151901) < 1e-6
    assert np.all(np.diff(workloads.shifts(3, 64)) >= 0)
    R, Z = workloads.atoms(1004, 20, 9)
    assert np.all(np.abs(R) <= 5) and Z.min() >= 1 and Z.max() <= 9
