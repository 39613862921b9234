"""ctypes face of oracle/fe_oracle.c plus the two harness-level algorithms that sit on top of the oracle's
apply: 20-step Lanczos bounds (reading R10), Rayleigh-Ritz (Eq. 23-24, l.210-219; readings R8, R9) and the
preconditioned MINRES of the adjoint solve (l.221-225).

TEST INFRASTRUCTURE: imported only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libfe_oracle.so")
_lib = None


def build_oracle(force=False):
    """gcc -O2 (no fast-math) build of the plain-C oracle into oracle/libfe_oracle.so."""
    src = os.path.join(_HERE, "fe_oracle.c")
    hdr = os.path.join(_HERE, "fe_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", _SO, src, "-lm"]
    subprocess.check_call(cmd)
    return _SO


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build_oracle()
    L = C.CDLL(_SO)
    dp, ip, i64p, u8p = (C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_uint8))
    vp = C.c_void_p
    sig = {
        "orc_gll": (C.c_int, [C.c_int, dp, dp]),
        "orc_gauss": (C.c_int, [C.c_int, dp, dp]),
        "orc_lagrange": (C.c_double, [C.c_int, dp, C.c_int, C.c_double]),
        "orc_lagrange_deriv": (C.c_double, [C.c_int, dp, C.c_int, C.c_double]),
        "orc_mesh_create": (vp, [dp, C.c_int, dp, C.c_int, dp, C.c_int, C.c_int]),
        "orc_mesh_destroy": (None, [vp]),
        "orc_num_nodes": (C.c_int64, [vp]),
        "orc_num_free": (C.c_int64, [vp]),
        "orc_num_cells": (C.c_int64, [vp]),
        "orc_nodes_per_cell": (C.c_int, [vp]),
        "orc_quad_per_cell": (C.c_int, [vp]),
        "orc_get_l2g": (None, [vp, ip]),
        "orc_get_node_coords": (None, [vp, dp]),
        "orc_get_quad_coords": (None, [vp, dp]),
        "orc_get_mass": (None, [vp, dp]),
        "orc_get_mask": (None, [vp, u8p]),
        "orc_cell_matrix": (None, [vp, C.c_int64, dp, C.c_double, C.c_double, dp]),
        "orc_build_cell_matrices": (None, [vp, dp, dp]),
        "orc_assemble": (vp, [vp, dp, C.c_int]),
        "orc_csr_destroy": (None, [vp]),
        "orc_csr_nnz": (C.c_int64, [vp]),
        "orc_csr_copy": (None, [vp, i64p, ip, dp]),
        "orc_csr_apply": (None, [vp, vp, dp, C.c_int, dp, dp, C.c_int]),
        "orc_cellwise_apply": (None, [vp, dp, dp, C.c_int, dp, dp]),
        "orc_apply_rows": (None, [vp, dp, dp, C.c_int, dp, i64p, C.c_int64, dp]),
        "orc_filter": (C.c_int, [vp, vp, dp, dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def gll(p):
    x, w = np.empty(p + 1), np.empty(p + 1)
    _load().orc_gll(p, _d(x), _d(w))
    return x, w


def gauss(nq):
    x, w = np.empty(nq), np.empty(nq)
    _load().orc_gauss(nq, _d(x), _d(w))
    return x, w


def lagrange(nodes, a, x):
    nodes = _f64(nodes)
    return _load().orc_lagrange(len(nodes), _d(nodes), a, float(x))


def lagrange_deriv(nodes, a, x):
    nodes = _f64(nodes)
    return _load().orc_lagrange_deriv(len(nodes), _d(nodes), a, float(x))


class OracleMesh:
    """Mesh + operator of the oracle.  set_potential() builds every cell matrix by explicit quadrature;
    assemble() builds the CSR of H~ (configs 1, 2, 5); without it, apply() uses the cell-wise form."""

    def __init__(self, xe, ye, ze, p):
        L = _load()
        self.xe, self.ye, self.ze = _f64(xe), _f64(ye), _f64(ze)
        self.p = int(p)
        self._h = L.orc_mesh_create(_d(self.xe), len(self.xe) - 1, _d(self.ye), len(self.ye) - 1,
                                    _d(self.ze), len(self.ze) - 1, self.p)
        if not self._h:
            raise ValueError("orc_mesh_create failed")
        self.N = L.orc_num_nodes(self._h)
        self.N_free = L.orc_num_free(self._h)
        self.ncells = L.orc_num_cells(self._h)
        self.nc = L.orc_nodes_per_cell(self._h)
        self.nq3 = L.orc_quad_per_cell(self._h)
        self.He = None
        self.Vq = None
        self._csr = None
        self._csr_raw = None

    def __del__(self):
        try:
            L = _load()
            for h in (self._csr, self._csr_raw):
                if h:
                    L.orc_csr_destroy(h)
            if self._h:
                L.orc_mesh_destroy(self._h)
        except Exception:
            pass

    # ---- tables -------------------------------------------------------------------------------------------
    def l2g(self):
        a = np.empty((self.ncells, self.nc), dtype=np.int32)
        _load().orc_get_l2g(self._h, a.ctypes.data_as(C.POINTER(C.c_int32)))
        return a

    def node_coords(self):
        a = np.empty((self.N, 3))
        _load().orc_get_node_coords(self._h, _d(a))
        return a

    def quad_coords(self):
        a = np.empty((self.ncells * self.nq3, 3))
        _load().orc_get_quad_coords(self._h, _d(a))
        return a

    def mass(self):
        a = np.empty(self.N)
        _load().orc_get_mass(self._h, _d(a))
        return a

    def mask(self):
        a = np.empty(self.N, dtype=np.uint8)
        _load().orc_get_mask(self._h, a.ctypes.data_as(C.POINTER(C.c_uint8)))
        return a

    # ---- operator -----------------------------------------------------------------------------------------
    def cell_matrix(self, e, Vq_cell=None, kin=0.5, pot=1.0):
        He = np.empty((self.nc, self.nc))
        v = _f64(Vq_cell) if Vq_cell is not None else None
        _load().orc_cell_matrix(self._h, int(e), _d(v), float(kin), float(pot), _d(He))
        return He

    def set_potential(self, Vq, build=True):
        self.Vq = _f64(Vq).reshape(-1)
        assert self.Vq.size == self.ncells * self.nq3
        L = _load()
        for name in ("_csr", "_csr_raw"):
            if getattr(self, name):
                L.orc_csr_destroy(getattr(self, name))
                setattr(self, name, None)
        self.He = None
        if build:
            self.He = np.empty((self.ncells, self.nc, self.nc))
            L.orc_build_cell_matrices(self._h, _d(self.Vq), _d(self.He))

    def assemble(self):
        if self._csr is None:
            self._csr = _load().orc_assemble(self._h, _d(self.He), 1)
        return self

    def csr(self, scaled=True):
        """(row_ptr, col, val) of H~ (scaled) or of the raw assembled H."""
        L = _load()
        if scaled:
            self.assemble()
            h = self._csr
        else:
            if self._csr_raw is None:
                self._csr_raw = L.orc_assemble(self._h, _d(self.He), 0)
            h = self._csr_raw
        nnz = L.orc_csr_nnz(h)
        rp, col, val = np.empty(self.N + 1, dtype=np.int64), np.empty(nnz, dtype=np.int32), np.empty(nnz)
        L.orc_csr_copy(h, rp.ctypes.data_as(C.POINTER(C.c_int64)), col.ctypes.data_as(C.POINTER(C.c_int32)), _d(val))
        return rp, col, val

    def apply(self, X, eps=None, nthreads=1, cellwise=False):
        X = _f64(X)
        B = X.shape[1]
        e = _f64(eps) if eps is not None else None
        Y = np.empty_like(X)
        L = _load()
        if self._csr is not None and not cellwise:
            L.orc_csr_apply(self._h, self._csr, _d(X), B, _d(e), _d(Y), int(nthreads))
        else:
            L.orc_cellwise_apply(self._h, _d(self.He), _d(X), B, _d(e), _d(Y))
        return Y

    def apply_rows(self, X, rows, eps=None):
        X = _f64(X)
        B = X.shape[1]
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        e = _f64(eps) if eps is not None else None
        Y = np.empty((len(rows), B))
        _load().orc_apply_rows(self._h, _d(self.Vq), _d(X), B, _d(e), rows.ctypes.data_as(C.POINTER(C.c_int64)),
                               len(rows), _d(Y))
        return Y

    def filter(self, X, m, a, b, a0, nthreads=1, cellwise=False):
        Y = _f64(X).copy()
        B = Y.shape[1]
        use_csr = self._csr is not None and not cellwise
        rc = _load().orc_filter(self._h, self._csr if use_csr else None, _d(self.He), _d(Y), B, int(m),
                                float(a), float(b), float(a0), int(nthreads))
        if rc != 0:
            raise ValueError("orc_filter: need a0 < a < b and m >= 1")
        return Y


def lanczos_bounds(mesh, v0, k=20, nthreads=1, return_tridiagonal=False):
    """Reading R10 (survey 8(c) step 8): k Lanczos steps on H~ (free rows) from the given start vector, no
    re-orthogonalisation; returns (theta_min, theta_max, beta_k).  b = theta_max + beta_k, a0 = theta_min.
    return_tridiagonal: also return the recurrence coefficients (alphas, betas) -- betas[i] couples steps i and i+1,
    betas[-1] is the norm of the last residual vector -- so that the pin in tests/test_oracle_pins.py can compare them
    with Q^T H~ Q from a Householder QR of the Krylov matrix."""
    mask = mesh.mask().astype(np.float64)
    v = _f64(v0).reshape(-1) * mask
    v = v / np.linalg.norm(v)
    v_prev = np.zeros_like(v)
    beta = 0.0
    alphas, betas = [], []
    for _ in range(k):
        w = mesh.apply(v.reshape(-1, 1), nthreads=nthreads).reshape(-1)
        alpha = float(w @ v)
        w = w - alpha * v - beta * v_prev
        beta = float(np.linalg.norm(w))
        alphas.append(alpha)
        betas.append(beta)
        if beta == 0.0:
            break
        v_prev, v = v, w / beta
    T = np.diag(alphas) + np.diag(betas[:-1], 1) + np.diag(betas[:-1], -1)
    theta = np.linalg.eigvalsh(T)
    if return_tridiagonal:
        return float(theta[0]), float(theta[-1]), float(betas[-1]), np.array(alphas), np.array(betas)
    return float(theta[0]), float(theta[-1]), float(betas[-1])


def rayleigh_ritz(mesh, Y, nthreads=1):
    """PAPER.md Eq. 23-24 (l.210-219) with readings R8 (H~_Y = Y^T H~ Y) and R9 (CholQR2):
    S = Y^T Y = L L^T, Q = Y L^{-T} (twice), G = Q^T H~ Q, G v = theta v, X = Q V.  Returns (theta, X, Q)."""
    mask = mesh.mask().astype(np.float64)[:, None]
    Q = _f64(Y) * mask
    for _ in range(2):
        S = Q.T @ Q
        Lc = np.linalg.cholesky(S)
        Q = np.linalg.solve(Lc, Q.T).T  # Q L^{-T}
    HQ = mesh.apply(Q, nthreads=nthreads)
    G = Q.T @ HQ
    G = 0.5 * (G + G.T)
    theta, V = np.linalg.eigh(G)
    return theta, Q @ V, Q


def ritz_residuals(mesh, X, theta, nthreads=1):
    """|| H~ x_j - theta_j x_j ||_2 over the free rows, column by column: the residual of the eigenvalue problem that the
    tolerance t_eig of PAPER.md l.296 is applied to."""
    X = _f64(X)
    free = mesh.mask().astype(bool)
    R = mesh.apply(X, nthreads=nthreads) - X * _f64(theta)[None, :]
    return np.sqrt(np.sum(R[free] ** 2, axis=0))


def chfsi(mesh, X, deg, a, b, a0, t_eig, n_gate, max_cycles=50, nthreads=1):
    """Chebyshev-filtered subspace iteration with the residual stopping rule of PAPER.md l.296 (t_eig = e_L2^2 / c_eig is
    handed in as a number): repeat { filter (l.208-210), Rayleigh-Ritz (Eq. 23-24), residuals } until the n_gate lowest
    pairs have residual <= t_eig; after each cycle a = largest, a0 = smallest Ritz value of the block (survey 8(c) step 8).
    Returns (theta, X, residuals, cycles)."""
    cycles = 0
    while True:
        theta, X, _ = rayleigh_ritz(mesh, mesh.filter(X, deg, a, b, a0, nthreads=nthreads), nthreads=nthreads)
        res = ritz_residuals(mesh, X, theta, nthreads=nthreads)
        cycles += 1
        if res[:n_gate].max() <= t_eig or cycles >= max_cycles:
            return theta, X, res, cycles
        a, a0 = float(theta[-1]), float(theta[0])


def laplacian_precond(mesh):
    """Inverse diagonal of the mass-scaled negative Laplacian, 1 / diag(M^{-1/2} (1/2 K) M^{-1/2}) on free rows and 0
    on Dirichlet rows: the MINRES preconditioner of PAPER.md l.225.  Diagonal taken entry by entry from the cell
    matrices of Eq. 17 with the potential switched off."""
    l2g = mesh.l2g()
    d = np.zeros(mesh.N)
    for e in range(mesh.ncells):
        Ke = mesh.cell_matrix(e, None, kin=0.5, pot=0.0)
        np.add.at(d, l2g[e], np.diag(Ke))
    mask = mesh.mask().astype(bool)
    out = np.zeros(mesh.N)
    out[mask] = mesh.mass()[mask] / d[mask]
    return out


def minres_shifted(mesh, G, eps=None, maxit=200, tol=1e-10, Minv=None, nthreads=1):
    """Preconditioned MINRES (Paige & Saunders 1975, the method PAPER.md l.223-225 names, ref. [59]; statement order and
    variable names after the canonical SOL `minres.m` / scipy.sparse.linalg.minres formulation of that algorithm) for
    (H~ - eps_j I) x_j = g_j, column by column, x_0 = 0, on the free rows.  Minv: diagonal preconditioner (N) or None.
    A column stops when phibar <= tol * beta1 (estimate of the preconditioned residual norm).
    Returns (X, phibar / beta1, iterations of the slowest column)."""
    G = _f64(G)
    N, B = G.shape
    mask = mesh.mask().astype(np.float64)
    Mi = mask if Minv is None else _f64(Minv) * mask
    X = np.zeros((N, B))
    rel = np.zeros(B)
    itmax = 0
    for j in range(B):
        ej = None if eps is None else np.array([eps[j]])
        b = G[:, j] * mask
        r1 = b.copy()
        y = Mi * r1
        beta1 = np.sqrt(max(r1 @ y, 0.0))
        if beta1 == 0.0:
            continue
        oldb, beta, dbar, epsln, phibar = 0.0, beta1, 0.0, 0.0, beta1
        cs, sn = -1.0, 0.0
        w = np.zeros(N)
        w2 = np.zeros(N)
        r2 = r1.copy()
        x = np.zeros(N)
        itn = 0
        while itn < maxit and phibar > tol * beta1 and beta > 0.0:
            itn += 1
            v = y / beta
            y = mesh.apply(v[:, None], ej, nthreads=nthreads)[:, 0]
            if itn >= 2:
                y = y - (beta / oldb) * r1
            alfa = v @ y
            y = y - (alfa / beta) * r2
            r1, r2 = r2, y
            y = Mi * r2
            oldb, beta = beta, np.sqrt(max(r2 @ y, 0.0))
            oldeps = epsln
            delta = cs * dbar + sn * alfa
            gbar = sn * dbar - cs * alfa
            epsln = sn * beta
            dbar = -cs * beta
            gamma = max(np.hypot(gbar, beta), np.finfo(float).eps)
            cs, sn = gbar / gamma, beta / gamma
            phi = cs * phibar
            phibar = sn * phibar
            w1, w2 = w2, w
            w = (v - oldeps * w1 - delta * w2) / gamma
            x = x + phi * w
        X[:, j] = x
        rel[j] = phibar / beta1
        itmax = max(itmax, itn)
    return X, rel, itmax


def density(mesh, X, f):
    """rho[e, q] = sum_j f_j psi_j(x_q)^2 at the Gauss points of every cell (Eq. 4, l.73-77), psi = M^{-1/2} psi~
    with zero Dirichlet rows; psi_j(x_q) = sum_a Phi_a(x_q) psi_{j,a} written out with the Lagrange basis of Eq. 12."""
    X = _f64(X)
    p, n = mesh.p, mesh.p + 1
    xg, _ = gll(p)
    xq, _ = gauss(n)
    L1 = np.array([[lagrange(xg, a, xq[q]) for a in range(n)] for q in range(n)])  # L1[q, a]
    s = np.zeros(mesh.N)
    free = mesh.mask().astype(bool)
    s[free] = 1.0 / np.sqrt(mesh.mass()[free])
    psi = X * s[:, None]
    l2g = mesh.l2g()
    rho = np.zeros((mesh.ncells, n ** 3))
    fw = _f64(f)
    for e in range(mesh.ncells):
        loc = psi[l2g[e]].reshape(n, n, n, -1)  # [az, ay, ax, j]
        val = np.einsum("ra,sb,tc,cbaj->rstj", L1, L1, L1, loc)  # [qx, qy, qz, j]: Phi_a = l_ax l_ay l_az
        r = np.einsum("rstj,j->rst", val ** 2, fw)
        rho[e] = r.transpose(2, 1, 0).reshape(-1)  # q = qx + n (qy + n qz)
    return rho


def adjoint_rhs(mesh, Psi, f, Uq, D):
    """g~ of PAPER.md Eq. 18 (l.174-177) in the scaled space of Eq. 19-20, for one block of orbitals Psi~ (N x B):
    g_a^{(i)} = int [ f_i U psi^{(i)} - sum_j (D + D^T)_{ij} psi^{(j)} ] N_a dr with U = 4 w (rho_data - rho) given at the
    quadrature points;  g~ = M^{-1/2} g, psi = M^{-1/2} psi~.  The first integral is M_U psi with (M_U)_ab = int N_a U N_b
    taken entry by entry from the cell matrices of Eq. 17 with the kinetic part switched off; the second is M psi with
    the lumped GLL mass (l.185), i.e. the identity in the scaled space.  Dirichlet rows are 0."""
    Psi = _f64(Psi)
    N, B = Psi.shape
    free = mesh.mask().astype(bool)
    s = np.zeros(N)
    s[free] = 1.0 / np.sqrt(mesh.mass()[free])
    psi = Psi * s[:, None]
    l2g = mesh.l2g()
    Uq = _f64(Uq).reshape(mesh.ncells, -1)
    g = np.zeros((N, B))
    for e in range(mesh.ncells):
        MU = mesh.cell_matrix(e, Uq[e], kin=0.0, pot=1.0)
        g[l2g[e]] += MU @ psi[l2g[e]]
    g = g * _f64(f)[None, :]
    DD = _f64(D) + _f64(D).T
    gt = g * s[:, None] - (Psi * free[:, None]) @ DD.T  # column i: sum_j (D + D^T)_{ij} psi~^{(j)}
    gt[~free] = 0.0
    return gt
