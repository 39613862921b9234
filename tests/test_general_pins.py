"""Pins of the general-hexahedral / hanging-node oracle (oracle/fe_general.py; NEXT-3) against what the mathematics fixes.
None of them calls the CUDA path."""
import numpy as np
import pytest
from numpy.polynomial import Polynomial

import oracle
import workloads


def _affine(A, b=(0.0, 0.0, 0.0)):
    A, b = np.asarray(A, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return lambda x: x @ A.T + b


SHEAR = np.array([[1.0, 0.3, -0.2], [0.1, 0.9, 0.25], [-0.15, 0.2, 1.1]])


def _refined(p, deform=None, levels=1, roots=3):
    e = workloads.uniform_edges(-1.5, 1.5, roots)
    radius = {0: 0.9, 1: 0.45}
    mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: np.linalg.norm((lo + hi) / 2) < radius[l], levels, deform)
    return mesh, oracle.GeneralOracleMesh(mesh, p)


@pytest.mark.parametrize("p", [1, 2, 4])
def test_unrefined_undeformed_mesh_is_the_tensor_oracle(p):
    """No refinement, no deformation: numbering, coordinates, mass, mask and H~ must be those of the (separately pinned)
    tensor-product oracle -- ties the general code path to fe_oracle.c."""
    xe, ye, ze = np.array([0.0, 0.7, 2.0]), np.array([-1.0, -0.5, 0.4, 1.0]), np.array([0.0, 0.3, 1.0])
    mesh = workloads.octree_mesh(xe, ye, ze, lambda l, lo, hi: False, 1)
    g = oracle.GeneralOracleMesh(mesh, p)
    t = oracle.OracleMesh(xe, ye, ze, p)
    assert (g.N, g.N_all, g.N_free, g.ncells) == (t.N, t.N, t.N_free, t.ncells)
    # the tensor oracle numbers nodes lexicographically (R3), the general one by first appearance (R23): compare through
    # the coordinates
    perm = np.empty(t.N, dtype=np.int64)
    perm[t.l2g().reshape(-1)] = g.l2g().reshape(-1)      # tensor id -> general id
    assert np.array_equal(np.sort(perm), np.arange(t.N))
    assert np.max(np.abs(g.node_coords()[perm] - t.node_coords())) < 1e-14
    assert np.max(np.abs(g.quad_coords() - t.quad_coords())) < 1e-14
    assert np.max(np.abs(g.mass()[perm] / t.mass() - 1)) < 1e-13
    assert np.array_equal(g.mask()[perm], t.mask())
    V = lambda q: -4.0 / np.sqrt((q ** 2).sum(axis=1) + 0.25)
    Vq = V(t.quad_coords())
    t.set_potential(Vq)
    t.assemble()
    g.set_potential(Vq)
    X = workloads.random_block(40 + p, t.N, 3, t.mask())
    Xg = np.empty_like(X)
    Xg[perm] = X
    eps = np.array([-1.0, 0.0, 0.5])
    Yt, Yg = t.apply(X, eps), g.apply(Xg, eps)
    assert np.linalg.norm(Yg[perm] - Yt) < 1e-12 * np.linalg.norm(Yt)
    Ft, Fg = t.filter(X, 5, 2.0, 300.0, -8.0), g.filter(Xg, 5, 2.0, 300.0, -8.0)
    assert np.linalg.norm(Fg[perm] - Ft) < 1e-12 * np.linalg.norm(Ft)


def _ref_1d(p):
    """Exactly integrated 1-D reference matrices on [-1,1] from the polynomial coefficients of the Lagrange basis:
    M[a,b] = int l_a l_b, D[a,b] = int l_a l_b', K[a,b] = int l_a' l_b'."""
    x, _ = oracle.gll(p)
    L = [Polynomial.fromroots(np.delete(x, a)) / np.prod(x[a] - np.delete(x, a)) for a in range(p + 1)]

    def integ(f):
        F = f.integ()
        return F(1.0) - F(-1.0)
    M = np.array([[integ(la * lb) for lb in L] for la in L])
    D = np.array([[integ(la * lb.deriv()) for lb in L] for la in L])
    K = np.array([[integ(la.deriv() * lb.deriv()) for lb in L] for la in L])
    return M, D, K


@pytest.mark.parametrize("p", [1, 2, 3])
def test_affine_cell_matrix_is_the_transformed_reference_matrix(p):
    """Sheared parallelepiped x = A xi + b: K_e = |det A| sum_ij (A^-1 A^-T)_ij int d_i Phi_a d_j Phi_b and the mass-like
    potential term |det A| V0 int Phi_a Phi_b, with the reference integrals built from independently, exactly integrated
    1-D matrices (Kronecker products; the n_q = p+1 Gauss rule is exact for them)."""
    A = SHEAR * 0.7
    corners = np.array([[(-1.0, 1.0)[v & 1], (-1.0, 1.0)[(v >> 1) & 1], (-1.0, 1.0)[v >> 2]] for v in range(8)])
    verts = corners @ A.T + np.array([0.3, -0.2, 1.0])
    mesh = workloads.OctreeMesh(1, 1, 1, [[0, 0, 0, 0]], verts[None], 0)
    g = oracle.GeneralOracleMesh(mesh, p)
    M, D, K = _ref_1d(p)
    G = np.linalg.inv(A) @ np.linalg.inv(A).T
    # index a = ax + n (ay + n az): Kronecker order (z, y, x)
    d = [[None] * 3 for _ in range(3)]
    one = {"M": M, "K": K, "D": D, "Dt": D.T}
    for i in range(3):
        for j in range(3):
            f = []
            for axis in (2, 1, 0):  # z, y, x factors
                if axis == i and axis == j:
                    f.append(K)
                elif axis == i:
                    f.append(D.T)   # int l_a' l_b
                elif axis == j:
                    f.append(D)     # int l_a l_b'
                else:
                    f.append(M)
            d[i][j] = np.kron(np.kron(f[0], f[1]), f[2])
    Kref = abs(np.linalg.det(A)) * sum(G[i, j] * d[i][j] for i in range(3) for j in range(3))
    Ke = g.cell_matrix(0, None, kin=1.0, pot=0.0)
    assert np.max(np.abs(Ke - Kref)) < 1e-12 * np.max(np.abs(Kref))
    Mref = abs(np.linalg.det(A)) * np.kron(np.kron(M, M), M)
    Me = g.cell_matrix(0, np.full(g.nq3, 2.5), kin=0.0, pot=1.0)
    assert np.max(np.abs(Me - 2.5 * Mref)) < 1e-12 * np.max(np.abs(Mref))
    assert abs(g._m_all.sum() - 8 * abs(np.linalg.det(A))) < 1e-12  # lumped mass sums to the volume


@pytest.mark.parametrize("p,levels", [(2, 1), (3, 1), (2, 2), (4, 1)])
def test_hanging_node_constraints(p, levels):
    """Refined, sheared (affine) mesh.  (i) every constraint row sums to one and refers to unconstrained nodes only;
    (ii) CONTINUITY: for a random vector on the unconstrained nodes, the expanded field of a fine cell and of the coarse
    cell it hangs on agree at random points of the shared face (evaluated with the Lagrange basis of Eq. 12);
    (iii) PATCH TESTS through the hanging faces: K_c (linear field) = 0 and, p >= 2, K_c (x^2+y^2+z^2) = -6 M_c at the
    free nodes -- the second pins the lumped constrained mass C^T m (reading R25) as well; (iv) symmetry of H_c."""
    mesh, g = _refined(p, _affine(SHEAR), levels)
    assert g.N_all > g.N and (mesh.cells[:, 0] == levels).any()
    Ch = g.constraint_matrix()
    assert np.max(np.abs(Ch.sum(axis=1) - 1.0)) < 1e-13
    # (ii) continuity at the nodes: a polynomial of degree p per cell that agrees at all (p+1)^2 face nodes agrees on the face
    u = workloads.normal(70 + p, g.N)
    u_all = g.Cfull @ u
    lev = mesh.cells[:, 0]
    n = p + 1
    x, _ = oracle.gll(p)
    checked = 0
    for h, row in list(g.constraints.items())[::7]:
        # the hanging value must equal the coarse cell's interpolant at the node's physical position: find a coarse cell
        # containing it and evaluate its field there through the inverse of the affine map
        pos = g.node_coords()[h]
        for e in np.flatnonzero(lev < levels):
            V = mesh.verts[e]
            A = np.stack([(V[1] - V[0]) / 2, (V[2] - V[0]) / 2, (V[4] - V[0]) / 2], axis=1)
            xi = np.linalg.solve(A, pos - V.mean(axis=0))
            if np.all(np.abs(xi) <= 1 + 1e-10) and not np.any(g.l2g()[e] == h):
                xi = np.clip(xi, -1, 1)
                w = [[oracle.lagrange(x, b, xi[d]) for b in range(n)] for d in range(3)]
                val = sum(w[0][b % n] * w[1][(b // n) % n] * w[2][b // (n * n)] * u_all[g.l2g()[e, b]] for b in range(n ** 3))
                assert abs(val - u_all[h]) < 1e-11 * max(1.0, np.abs(u).max())
                checked += 1
                break
    assert checked > 3
    # (iii) patch tests
    g.set_potential(np.zeros(g.ncells * g.nq3), kin=1.0)
    xyz = g.node_coords()[:g.N]
    free = g.mask().astype(bool)
    Kc = g.Hc
    lin = 0.3 + xyz @ np.array([1.0, -2.0, 0.5])
    assert np.max(np.abs((Kc @ lin)[free])) < 1e-11 * np.abs(Kc).max()
    if p >= 2:
        quad = (xyz ** 2).sum(axis=1)
        r = (Kc @ quad)[free] + 6.0 * g.mass()[free]
        assert np.max(np.abs(r)) < 1e-10 * np.abs(Kc).max()
    assert abs(Kc - Kc.T).max() < 1e-12 * np.abs(Kc).max()
    assert abs(g.mass().sum() - 27.0 * abs(np.linalg.det(SHEAR))) < 1e-11  # C^T m keeps the volume (rows of C sum to one)


def test_refinement_improves_the_oscillator_ground_state():
    """3-D harmonic oscillator on [-6,6]^3, p=3: refining the 8 central root cells moves the lowest eigenvalues towards
    1.5 and 2.5 (x3) (BASELINE.json's convergence pin, here through hanging nodes)."""
    e = workloads.uniform_edges(-6.0, 6.0, 4)
    errs = []
    for refine in (False, True):
        mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: refine and np.abs((lo + hi) / 2).max() < 3.0, 1)
        g = oracle.GeneralOracleMesh(mesh, 3)
        g.set_potential(workloads.harmonic(g.quad_coords()))
        free = np.flatnonzero(g.mask())
        lam = np.linalg.eigvalsh(g.Ht.toarray()[np.ix_(free, free)])
        errs.append((abs(lam[0] - 1.5), np.abs(lam[1:4] - 2.5).max()))
    assert errs[1][0] < 0.25 * errs[0][0] and errs[1][1] < 0.5 * errs[0][1]
    assert errs[1][0] < 2e-3


def test_density_preconditioner_and_potential_apply_on_constrained_meshes():
    """(i) unrefined mesh: the general preconditioner equals the tensor oracle's (diag of the potential-free operator);
    (ii) refined sheared mesh, a polynomial field of degree <= p sampled at the unconstrained nodes: the hanging values
    reproduce it, so rho(x_q) = f poly(x_q)^2 in closed form and sum_q w|J| rho = the exactly known integral is matched by
    the weights; (iii) potential_apply through its weak form: v^T (C^T M_U C) u = sum_q w|J| U u v for polynomial u, v;
    (iv) the preconditioner is positive on free rows."""
    xe, ye, ze = np.array([0.0, 0.7, 2.0]), np.array([-1.0, -0.5, 0.4, 1.0]), np.array([0.0, 0.3, 1.0])
    p = 3
    g0 = oracle.GeneralOracleMesh(workloads.octree_mesh(xe, ye, ze, lambda l, lo, hi: False, 0), p)
    t0 = oracle.OracleMesh(xe, ye, ze, p)
    perm = np.empty(t0.N, dtype=np.int64)
    perm[t0.l2g().reshape(-1)] = g0.l2g().reshape(-1)
    t0.set_potential(np.zeros(t0.ncells * t0.nq3))
    assert np.max(np.abs(g0.laplacian_precond()[perm] - oracle.laplacian_precond(t0))) < 1e-12
    mesh, g = _refined(p, _affine(SHEAR), 1)
    xyz = g.node_coords()[:g.N]
    free = g.mask().astype(bool)
    poly = lambda x: 0.3 + x[:, 0] - 0.5 * x[:, 1] * x[:, 2] + 0.25 * x[:, 0] ** 2 * x[:, 2]  # degree <= 3 per variable
    # psi~ = M_c^{1/2} psi with psi the polynomial; Dirichlet rows carry the polynomial too but are ignored by the density
    sq = np.sqrt(g.mass())
    X = np.stack([poly(xyz) * sq, (0.2 - xyz[:, 1]) * sq], axis=1)
    # the density ignores Dirichlet rows; compare only in cells that do not touch the boundary
    rho = g.density(X, np.array([2.0, 1.0]))
    q = g.quad_coords().reshape(g.ncells, -1, 3)
    touches = np.array([not free[g.l2g()[e][g.l2g()[e] < g.N]].all() for e in range(g.ncells)])
    ref = 2.0 * poly(q.reshape(-1, 3)) ** 2 + (0.2 - q.reshape(-1, 3)[:, 1]) ** 2
    ref = ref.reshape(g.ncells, -1)
    inner = ~touches
    assert inner.sum() >= 8
    assert np.max(np.abs(rho[inner] - ref[inner])) < 1e-11 * np.abs(ref).max()
    Mi = g.laplacian_precond()
    assert np.all(Mi[free] > 0) and np.all(Mi[~free] == 0)
    # weak form of the potential-only operator with U = 1 + x: v^T S^-1 [S C^T M_U C S] S^-1 u over interior-supported u, v
    U = 1.0 + q.reshape(-1, 3)[:, 0]
    u = np.where(free, poly(xyz), 0.0)
    Y = g.potential_apply(U, (u * sq)[:, None])[:, 0]
    # bilinear form with v = u: u^T C^T M_U C u = sum over cells of quadrature of U (u_h)^2, u_h = the FE interpolant of u
    u_all = g.Cfull @ u
    n = p + 1
    x1, _ = oracle.gll(p)
    xq, wq = oracle.gauss(n)
    L1 = np.array([[oracle.lagrange(x1, a, xq[k]) for a in range(n)] for k in range(n)])
    total = 0.0
    for e in range(g.ncells):
        loc = u_all[g.l2g()[e]].reshape(n, n, n)
        val = np.einsum("ra,sb,tc,cba->rst", L1, L1, L1, loc).transpose(2, 1, 0).reshape(-1)
        V = mesh.verts[e]
        det = abs(np.linalg.det(np.stack([(V[1] - V[0]) / 2, (V[2] - V[0]) / 2, (V[4] - V[0]) / 2], axis=1)))
        w3 = np.array([wq[a] * wq[b] * wq[c] for c in range(n) for b in range(n) for a in range(n)])
        total += np.sum(w3 * det * U.reshape(g.ncells, -1)[e] * val ** 2)
    assert abs(u @ (Y * sq) - total) < 1e-11 * abs(total)


def test_apply_rows_equals_the_assembled_operator():
    """apply_rows (the row-by-row definition used at sizes where nothing can be assembled) against the assembled H~ on a
    two-level refined sheared mesh: every row, including unconstrained nodes that hanging nodes depend on."""
    mesh, g = _refined(2, _affine(SHEAR), 2)
    Vq = -4.0 / np.sqrt((g.quad_coords() ** 2).sum(axis=1) + 0.25)
    g.set_potential(Vq)
    X = workloads.random_block(90, g.N, 3, g.mask())
    eps = np.array([-0.5, 0.0, 0.7])
    rows = np.arange(0, g.N, 3)
    Yr = g.apply_rows(X, rows, Vq, eps)
    Y = g.apply(X, eps)
    assert np.linalg.norm(Yr - Y[rows]) < 1e-12 * np.linalg.norm(Y[rows])
