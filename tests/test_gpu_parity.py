"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star, reading R16): relative Frobenius error over free rows <= 1e-11 for one apply
(plain and shifted), <= 1e-9 after cheb_filter; l2g and Dirichlet mask byte-identical.
"""
import numpy as np
import pytest

import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_APPLY = 1e-11
TOL_FILTER = 1e-9

UNEQUAL = (np.array([0.0, 0.7, 2.0]), np.array([-1.0, -0.5, 0.4, 1.0]), np.array([0.0, 0.3, 1.0, 1.2, 2.5]))


def _fe():
    import paper_2510_10529_b200 as fe
    return fe


def _pair(edges, p, V):
    """(oracle mesh with cell matrices + CSR, GPU mesh) with the same potential, evaluated ONCE at the oracle's points."""
    import oracle
    fe = _fe()
    om = oracle.OracleMesh(*edges, p)
    Vq = V(om.quad_coords())
    om.set_potential(Vq)
    om.assemble()
    gm = fe.FEMesh(*edges, p)
    gm.set_potential(Vq)
    return om, gm


def _relerr(Yg, Yo, mask):
    free = mask.astype(bool)
    return np.linalg.norm(Yg[free] - Yo[free]) / max(np.linalg.norm(Yo[free]), 1e-300)


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


def _coulomb(q):
    return -4.0 / np.sqrt((q**2).sum(axis=1) + 0.25)


# ---- T1: setup tables ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_tables_match_oracle(p):
    import oracle
    fe = _fe()
    om = oracle.OracleMesh(*UNEQUAL, p)
    gm = fe.FEMesh(*UNEQUAL, p)
    assert (gm.N, gm.N_free, gm.ncells, gm.nc, gm.nq3) == (om.N, om.N_free, om.ncells, om.nc, om.nq3)
    assert np.array_equal(gm.l2g(), om.l2g())  # bit-exact (BASELINE.json)
    assert np.array_equal(gm.mask(), om.mask())
    assert np.max(np.abs(gm.node_coords() - om.node_coords())) <= 2 * np.spacing(2.5)
    assert np.max(np.abs(gm.quad_coords() - om.quad_coords())) <= 2 * np.spacing(2.5)
    Mo, Mg = om.mass(), gm.mass()
    assert np.max(np.abs(Mg - Mo) / Mo) < 2e-15


# ---- T2: one apply -------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_apply_all_orders(p):
    e = (np.array([0.0, 0.9, 2.0]), np.array([-1.0, 0.1, 1.0]), np.array([0.0, 0.6, 1.0]))
    om, gm = _pair(e, p, _coulomb)
    B = 5
    X = workloads.random_block(100 + p, om.N, B)  # boundary rows NOT zeroed: must be ignored
    Yo = om.apply(X)
    Yg = gm.apply_H(_dev(X)).cpu().numpy()
    assert _relerr(Yg, Yo, om.mask()) <= TOL_APPLY
    assert np.all(Yg[om.mask() == 0] == 0)


@pytest.mark.parametrize("variant", [3, 5])
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_apply_all_orders_both_kernel_generations(p, variant):
    """Even B takes the TMA kernel (variant 5 = default), variant 3 forces the legacy atomics kernel; B = 6 is a
    ragged tail of the 16/32-wide vector box (out-of-bounds columns of the tensor tile)."""
    e = (np.array([0.0, 0.9, 2.0]), np.array([-1.0, 0.1, 1.0]), np.array([0.0, 0.6, 1.0]))
    om, gm = _pair(e, p, _coulomb)
    gm.set_variant(variant)
    B = 6
    X = workloads.random_block(200 + p, om.N, B)  # boundary rows NOT zeroed: must be ignored
    eps = workloads.shifts(2100 + p, B)
    Yo = om.apply(X, eps)
    Yg = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert _relerr(Yg, Yo, om.mask()) <= TOL_APPLY
    assert np.all(Yg[om.mask() == 0] == 0)


@pytest.mark.parametrize("p,B,deg,variant", [(1, 4, 5, 5), (3, 10, 4, 5), (4, 34, 6, 5), (5, 6, 3, 5), (6, 18, 5, 5),
                                             (7, 4, 2, 5), (8, 2, 4, 5), (6, 18, 5, 3), (4, 7, 4, 0), (6, 3, 3, 0)])
def test_filter_unequal_mesh_all_paths(p, B, deg, variant):
    """cheb_filter on the 2x3x4 unequal mesh: pre-initialised TMA recurrence (even B) and the legacy path (odd B or
    variant 3); caller data in the Dirichlet rows of X must be ignored (R5) and come back as 0."""
    om, gm = _pair(UNEQUAL, p, _coulomb)
    gm.set_variant(variant)
    mask = om.mask()
    X = workloads.random_block(300 + p, om.N, B)  # garbage in boundary rows
    X0 = X * mask[:, None]
    import oracle
    th_min, th_max, beta = oracle.lanczos_bounds(om, workloads.normal(3100 + p, om.N), 20)
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    Yo = om.filter(X0, deg, a, b, a0)
    work = torch.full((2 * om.N * B,), 7.5, dtype=torch.float64, device="cuda")  # dirty work space
    Yg = gm.cheb_filter(_dev(X).clone(), deg, a, b, a0, work).cpu().numpy()
    assert _relerr(Yg, Yo, mask) <= TOL_FILTER
    assert np.all(Yg[mask == 0] == 0)


@pytest.mark.parametrize("p,B", [(2, 1), (2, 8), (3, 33), (4, 64), (2, 70)])
def test_apply_unequal_mesh_ragged_B(p, B):
    """2x3x4 cells with unequal edges (axis-order bugs), B = 1, a ragged tail, several tiles."""
    om, gm = _pair(UNEQUAL, p, _coulomb)
    X = workloads.random_block(7, om.N, B, om.mask())
    Yo = om.apply(X)
    Yg = gm.apply_H(_dev(X)).cpu().numpy()
    assert _relerr(Yg, Yo, om.mask()) <= TOL_APPLY


def test_shifted_apply():
    """Config 5 shape on a reduced mesh: (H~ - eps_j I) X_j with sorted eps in [-2, 0] (Eq. 20, R18)."""
    w = workloads.reduced(5, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    X = workloads.random_block(w.x_seed, om.N, w.B, om.mask())
    eps = w.eps()
    Yo = om.apply(X, eps)
    Yg = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert _relerr(Yg, Yo, om.mask()) <= TOL_APPLY
    # eps == 0 reproduces the plain apply up to summation order
    Y0 = gm.apply_H(_dev(X), eps=torch.zeros(w.B, dtype=torch.float64, device="cuda")).cpu().numpy()
    assert _relerr(Y0, om.apply(X), om.mask()) <= TOL_APPLY


def test_degenerate_meshes():
    """One cell (a single free node at p=2) and the smallest mesh with a free node at p=1."""
    e1 = np.array([0.0, 1.0])
    om, gm = _pair((e1, e1, e1), 2, workloads.harmonic)
    X = workloads.random_block(3, om.N, 4)
    assert om.N_free == 1
    assert _relerr(gm.apply_H(_dev(X)).cpu().numpy(), om.apply(X), om.mask()) <= TOL_APPLY
    e2 = np.array([0.0, 1.0, 2.5])
    om, gm = _pair((e2, e2, e2), 1, workloads.harmonic)
    X = workloads.random_block(4, om.N, 3)
    assert om.N_free == 1
    assert _relerr(gm.apply_H(_dev(X)).cpu().numpy(), om.apply(X), om.mask()) <= TOL_APPLY
    # all-boundary mesh: p=1, one cell -> Y == 0
    om, gm = _pair((e1, e1, e1), 1, workloads.harmonic)
    Y = gm.apply_H(_dev(workloads.random_block(5, om.N, 2))).cpu().numpy()
    assert om.N_free == 0 and np.all(Y == 0)


# ---- T3: filter ----------------------------------------------------------------------------------------------------
def test_filter_config1():
    """BASELINE.json config 1: 4^3 cells, p=2, V = r^2/2, B=8, m=10, bounds from 20 Lanczos steps (R10)."""
    import oracle
    w = workloads.config(1)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    X = w.X(mask)
    th_min, th_max, beta = oracle.lanczos_bounds(om, workloads.normal(3001, om.N), 20)
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    for deg in (1, 2, 3, w.m):
        Yo = om.filter(X, deg, a, b, a0)
        Yg = gm.cheb_filter(_dev(X).clone(), deg, a, b, a0).cpu().numpy()
        assert _relerr(Yg, Yo, mask) <= TOL_FILTER, deg
        assert np.all(Yg[mask == 0] == 0)


def test_filter_reduced_config2_and_ritz_values():
    """Config 2 recipe on 4^3 cells: lock-step filter parity per cycle and Ritz values of the free-running GPU cycles
    (Eq. 23-24; R20)."""
    import oracle
    w = workloads.reduced(2, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    B = 16
    Xo = workloads.random_block(w.x_seed, om.N, B, mask)
    Xg = Xo.copy()
    th_min, th_max, beta = oracle.lanczos_bounds(om, workloads.normal(3002, om.N), 20)
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    ag, a0g = a, a0
    for cycle in range(3):
        Yo = om.filter(Xo, w.m, a, b, a0)
        Ylock = gm.cheb_filter(_dev(Xo).clone(), w.m, a, b, a0).cpu().numpy()
        assert _relerr(Ylock, Yo, mask) <= TOL_FILTER, cycle
        theta_o, Xo, _ = oracle.rayleigh_ritz(om, Yo)
        # free-running GPU cycle, all on the device: its own filter output, then fe_rayleigh_ritz (NEXT-1)
        Xgd = gm.cheb_filter(_dev(Xg).clone(), w.m, ag, b, a0g)
        theta_g = gm.rayleigh_ritz(Xgd)
        Xg = Xgd.cpu().numpy()
        assert np.max(np.abs(theta_g - theta_o) / np.maximum(1.0, np.abs(theta_o))) <= 1e-9, cycle
        a, a0 = theta_o[-1], theta_o[0]
        ag, a0g = theta_g[-1], theta_g[0]


@pytest.mark.parametrize("p,B", [(2, 8), (4, 16), (3, 37), (2, 128)])
def test_device_rayleigh_ritz(p, B):
    """fe_rayleigh_ritz (NEXT-1: device Gram / rotation kernels, host B x B Cholesky and eigensolver) against the oracle's
    Eq. 23-24: Ritz values <= 1e-9 (R16); vectors are compared through what is unique (R17): orthonormality, the
    spanned subspace, and the Ritz residual relation Q^T H~ Q = diag(theta)."""
    import oracle
    w = workloads.reduced(2, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), p, w.V)
    mask = om.mask()
    free = mask.astype(bool)
    Y = workloads.random_block(500 + p, om.N, B)  # garbage in the Dirichlet rows: must not take part
    th_min, th_max, beta = oracle.lanczos_bounds(om, workloads.normal(3200 + p, om.N), 20)
    b, a0 = th_max + beta, th_min
    Yf = om.filter(Y * mask[:, None], 4, a0 + 0.1 * (b - a0), b, a0)  # mildly filtered block (conditioned, not orthogonal)
    Yin = Yf.copy()
    Yin[~free] = 3.25
    theta_o, Xo, _ = oracle.rayleigh_ritz(om, Yf)
    Xd = _dev(Yin)
    theta_g = gm.rayleigh_ritz(Xd)
    Xg = Xd.cpu().numpy()
    assert np.max(np.abs(theta_g - theta_o) / np.maximum(1.0, np.abs(theta_o))) <= 1e-9
    assert np.all(Xg[~free] == 0)
    assert np.max(np.abs(Xg.T @ Xg - np.eye(B))) <= 1e-12
    # same subspace: projecting the oracle's Ritz vectors onto span(Xg) loses nothing
    assert np.linalg.norm(Xo - Xg @ (Xg.T @ Xo)) <= 1e-9 * np.linalg.norm(Xo)
    G = Xg.T @ om.apply(Xg)
    assert np.max(np.abs(G - np.diag(theta_g))) <= 1e-9 * max(1.0, np.max(np.abs(theta_g)))


@pytest.mark.parametrize("precondition", [False, True])
def test_block_minres_shifted(precondition):
    """fe_minres_shifted (NEXT-2) on the config-5 recipe (reduced mesh): same Paige-Saunders iteration as the oracle,
    column by column; compared after a FIXED number of steps (the iterates of the two sides then differ by rounding
    only) and at convergence, where the true residual of the GPU solution is checked with the oracle's operator."""
    import oracle
    w = workloads.reduced(5, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    free = mask.astype(bool)
    B = 12
    G = workloads.random_block(600, om.N, B)  # Dirichlet rows hold data that must be ignored
    eps = workloads.shifts(2600, B)
    Mi = oracle.laplacian_precond(om) if precondition else None
    Xo, relo, ito = oracle.minres_shifted(om, G, eps, maxit=25, tol=0.0, Minv=Mi)
    Xg, relg, itg = gm.minres_shifted(_dev(G), _dev(eps), maxit=25, tol=0.0, precondition=precondition)
    Xg = Xg.cpu().numpy()
    assert itg == 25 and ito == 25
    assert _relerr(Xg, Xo, mask) <= 1e-9
    assert np.max(np.abs(relg - relo)) <= 1e-9
    assert np.all(Xg[~free] == 0)
    # run to convergence; the residual is measured with the oracle's operator, not with the solver's own estimate
    Xc, relc, itc = gm.minres_shifted(_dev(G), _dev(eps), maxit=3000, tol=1e-9, precondition=precondition)
    Xc = Xc.cpu().numpy()
    R = (om.apply(Xc, eps) - G * mask[:, None])[free]
    assert np.all(relc <= 1e-9) and itc < 3000
    assert np.linalg.norm(R) <= 1e-6 * np.linalg.norm(G[free])
    if precondition:  # l.225: the preconditioner has to pay for itself
        _, _, it_plain = gm.minres_shifted(_dev(G), _dev(eps), maxit=3000, tol=1e-9, precondition=False)
        assert itc < it_plain


@pytest.mark.parametrize("B", [7, 66, 128])
def test_block_minres_block_widths(B):
    """The elementwise passes of a MINRES step have three launch shapes: 16-byte accesses with one tile of 64 columns (even
    B <= 64, covered above), with two tiles (even B up to 128), and 8-byte accesses for odd B.  Fixed 12 steps, all columns."""
    import oracle
    w = workloads.reduced(5, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    G = workloads.random_block(610 + B, om.N, B)
    eps = workloads.shifts(2610 + B, B)
    Mi = oracle.laplacian_precond(om)
    Xo, relo, ito = oracle.minres_shifted(om, G, eps, maxit=12, tol=0.0, Minv=Mi)
    Xg, relg, itg = gm.minres_shifted(_dev(G), _dev(eps), maxit=12, tol=0.0, precondition=True)
    Xg = Xg.cpu().numpy()
    assert itg == 12 and ito == 12
    assert _relerr(Xg, Xo, mask) <= 1e-9
    assert np.max(np.abs(relg - relo)) <= 1e-9
    assert np.all(Xg[~mask.astype(bool)] == 0)


def test_adjoint_null_space_completion():
    """l.221-223: eps_k = Ritz values, g orthogonal to the Ritz vectors; after the MINRES solve the component along
    Psi is replaced by d (Eq. 8 supplies d; here seeded): P += Psi (d - Psi^T P)."""
    import oracle
    w = workloads.reduced(2, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    B = 6
    Y = workloads.random_block(610, om.N, B, mask)
    th_min, th_max, beta = oracle.lanczos_bounds(om, workloads.normal(3300, om.N), 20)
    b, a0 = th_max + beta, th_min
    Xd = _dev(Y)
    a = a0 + 0.05 * (b - a0)
    for _ in range(8):  # converge the lowest Ritz pairs on the device
        gm.cheb_filter(Xd, 20, a, b, a0)
        theta = gm.rayleigh_ritz(Xd)
        a, a0 = theta[-1] + 0.05 * (b - theta[-1]), theta[0]
    Psi = Xd.clone()
    Ph = Psi.cpu().numpy()
    G = workloads.random_block(611, om.N, B, mask)
    G -= Ph @ (Ph.T @ G)  # orthogonal to every Ritz vector (degenerate levels included)
    # With Ritz (not exact) pairs the system is only nearly singular and, preconditioned (l.225), M^{-1} g is not
    # orthogonal to Psi either: the Psi-component of the iterate is whatever the near-null space amplifies (the exact
    # case of l.221-223 is pinned on the oracle in test_oracle_pins).  The library therefore SETS that component: P += Psi (d - Psi^T P) with d from Eq. 8 (here a seeded matrix).  fe_gram and
    # fe_add_subspace are the two device pieces of that completion.
    P, rel, it = gm.minres_shifted(_dev(G), _dev(theta), maxit=600, tol=1e-7, precondition=True)
    C = gm.gram(Psi, P)
    Pn = P.cpu().numpy()
    assert np.max(np.abs(C - Ph.T @ Pn)) <= 1e-11 * max(1.0, np.max(np.abs(C)))
    d = np.diag(workloads.normal(612, B))
    gm.add_subspace(Psi, d - C, P)
    Pf = P.cpu().numpy()
    assert np.max(np.abs(Ph.T @ Pf - d)) <= 1e-9 * max(1.0, np.max(np.abs(C)))
    Pref = Pn + Ph @ (d - C)
    assert np.linalg.norm(Pf - Pref) <= 1e-12 * np.linalg.norm(Pref)


@pytest.mark.parametrize("p,B", [(1, 2), (2, 8), (3, 33), (4, 64), (6, 40), (8, 5)])
def test_density_at_quadrature_points(p, B):
    """fe_density (NEXT-4, Eq. 4) against the oracle's definition on the unequal 2x3x4 mesh: several vector tiles, a
    ragged tail, data in the Dirichlet rows that must not contribute."""
    import oracle
    fe = _fe()
    om = oracle.OracleMesh(*UNEQUAL, p)
    gm = fe.FEMesh(*UNEQUAL, p)
    X = workloads.random_block(700 + p, om.N, B)
    f = 2.0 * workloads.uniform01(701 + p, 0, B)
    rho_o = oracle.density(om, X, f).reshape(-1)
    rho_g = gm.density(_dev(X), _dev(f)).cpu().numpy()
    assert np.linalg.norm(rho_g - rho_o) <= 1e-12 * np.linalg.norm(rho_o)


def test_device_lanczos_bounds_and_chfsi_cycles():
    """fe_lanczos_bounds against the oracle's 20-step Lanczos (R10), then BASELINE config 2's recipe end to end on the
    device — bounds, five filter + Rayleigh-Ritz cycles (R20) — against the same cycles on the oracle: Ritz values of
    the final cycle <= 1e-9 (R16)."""
    import oracle
    w = workloads.reduced(2, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    v0 = workloads.normal(3400, om.N)
    lo_o, hi_o, be_o = oracle.lanczos_bounds(om, v0, 20)
    lo_g, hi_g, be_g = gm.lanczos_bounds(_dev(v0), 20)
    scale = max(abs(hi_o), 1.0)
    assert abs(lo_g - lo_o) <= 1e-8 * scale and abs(hi_g - hi_o) <= 1e-8 * scale and abs(be_g - be_o) <= 1e-7 * scale
    B = 16
    Xo = workloads.random_block(w.x_seed, om.N, B, mask)
    Xg = _dev(Xo)
    bo, a0o = hi_o + be_o, lo_o
    ao = a0o + 0.1 * (bo - a0o)
    bg, a0g = hi_g + be_g, lo_g
    ag = a0g + 0.1 * (bg - a0g)
    for cycle in range(5):
        theta_o, Xo, _ = oracle.rayleigh_ritz(om, om.filter(Xo, w.m, ao, bo, a0o))
        gm.cheb_filter(Xg, w.m, ag, bg, a0g)
        theta_g = gm.rayleigh_ritz(Xg)
        ao, a0o = theta_o[-1], theta_o[0]
        ag, a0g = theta_g[-1], theta_g[0]
    assert np.max(np.abs(theta_g - theta_o) / np.maximum(1.0, np.abs(theta_o))) <= 1e-9


def test_ritz_residuals_and_residual_controlled_chfsi():
    """fe_ritz_residuals and fe_chfsi (NEXT-4, l.296) on the config-2 recipe (reduced mesh): residual norms of a given
    block against the oracle's definition, then the residual-controlled loop from device Lanczos bounds -- same number
    of cycles, Ritz values <= 1e-9, residuals of the gated pairs below t_eig on both sides."""
    import oracle
    w = workloads.reduced(2, 4)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    B, n_gate, t_eig = 16, 6, 1e-7
    X0 = workloads.random_block(w.x_seed, om.N, B, mask)
    th_min, th_max, beta = oracle.lanczos_bounds(om, workloads.normal(3500, om.N), 20)
    b, a0 = th_max + beta, th_min
    a = a0 + 0.1 * (b - a0)
    # residuals of a half-converged block with garbage in its Dirichlet rows
    th1, X1, _ = oracle.rayleigh_ritz(om, om.filter(X0, w.m, a, b, a0))
    Xin = X1.copy()
    Xin[mask == 0] = -4.5
    r_o = oracle.ritz_residuals(om, X1, th1)
    r_g = gm.ritz_residuals(_dev(Xin), th1)
    assert np.max(np.abs(r_g - r_o)) <= 1e-11 * max(1.0, r_o.max())
    theta_o, _, res_o, cyc_o = oracle.chfsi(om, X0, w.m, a, b, a0, t_eig, n_gate, max_cycles=30)
    Xg = _dev(X0)
    theta_g, res_g, cyc_g = gm.chfsi(Xg, w.m, a, b, a0, t_eig, n_gate, max_cycles=30)
    assert cyc_g == cyc_o and 1 < cyc_g < 30
    assert res_g[:n_gate].max() <= t_eig and res_o[:n_gate].max() <= t_eig
    assert np.max(np.abs(theta_g - theta_o) / np.maximum(1.0, np.abs(theta_o))) <= 1e-9
    Q = Xg.cpu().numpy()
    assert np.max(np.abs(Q.T @ Q - np.eye(B))) <= 1e-12
    assert np.max(np.abs(oracle.ritz_residuals(om, Q, theta_g) - res_g)) <= 1e-9  # the library's own claim, checked


@pytest.mark.parametrize("B", [6, 64, 96])
def test_filter_from_host_buffers(B):
    """cheb_filter_host (H2D, filter, D2H through the C ABI; chunks of 32 columns on two streams when B % 32 == 0)
    against the oracle and against the device-resident call."""
    w = workloads.config(1)
    om, gm = _pair((w.xe, w.ye, w.ze), w.p, w.V)
    mask = om.mask()
    X = workloads.random_block(800 + B, om.N, B)  # data in the Dirichlet rows: ignored, returned as 0
    a0, a, b = 1.0, 3.0, 25.0
    Yo = om.filter(X * mask[:, None], 7, a, b, a0)
    Xh = torch.as_tensor(X.copy()).pin_memory()
    gm.cheb_filter_host(Xh, 7, a, b, a0)
    assert _relerr(Xh.numpy(), Yo, mask) <= TOL_FILTER
    assert np.all(Xh.numpy()[mask == 0] == 0)
    Xn = X.copy()  # pageable numpy memory works too
    gm.cheb_filter_host(Xn, 7, a, b, a0)
    Yd = gm.cheb_filter(_dev(X).clone(), 7, a, b, a0).cpu().numpy()
    assert _relerr(Xn, Yd, mask) <= 1e-13


@pytest.mark.parametrize("B", [64, 128])
def test_filter_from_host_buffers_edge_chunks(B):
    """cheb_filter_host at p = 6, where the first and the last column chunk are 16 wide (16, 32, ..., 32, 16: the exposed
    copy-in / copy-out halves) and run the 16-wide launch shape while the middle chunks run the 32-wide one: against the
    oracle and against the device-resident call."""
    xe, ye, ze = np.array([0.0, 0.8, 2.0]), np.array([-1.0, -0.2, 0.5, 1.4]), np.array([0.0, 0.9, 1.7])
    om, gm = _pair((xe, ye, ze), 6, lambda q: -3.0 / np.sqrt(((q - 0.7) ** 2).sum(axis=1) + 0.25))
    mask = om.mask()
    X = workloads.random_block(900 + B, om.N, B)
    a0, a, b = -4.0, 30.0, 2600.0
    Xh = torch.as_tensor(X.copy()).pin_memory()
    gm.cheb_filter_host(Xh, 5, a, b, a0)
    Yd = gm.cheb_filter(_dev(X).clone(), 5, a, b, a0).cpu().numpy()
    assert _relerr(Xh.numpy(), Yd, mask) <= 1e-13 and np.all(Xh.numpy()[mask == 0] == 0)
    if B == 64:
        assert _relerr(Xh.numpy(), om.filter(X * mask[:, None], 5, a, b, a0), mask) <= TOL_FILTER


def test_colour_ordered_scatter_is_reproducible_and_agrees():
    """Variant 4 (SURVEY a3 "atomic or colour-ordered"): two runs are bit-identical, and the atomic paths (TMA bulk
    reduce-add, legacy red.global) agree with it to rounding — the deterministic mode doubles as a race oracle (R17)."""
    om, gm = _pair(UNEQUAL, 4, _coulomb)
    mask = om.mask()
    B = 10
    X = workloads.random_block(900, om.N, B, mask)
    eps = workloads.shifts(2900, B)
    Xd, ed = _dev(X), _dev(eps)
    gm.set_variant(4)
    Y1 = gm.apply_H(Xd, eps=ed).clone()
    Y2 = gm.apply_H(Xd, eps=ed).clone()
    F1 = gm.cheb_filter(Xd.clone(), 6, -2.0, 400.0, -12.0)
    F2 = gm.cheb_filter(Xd.clone(), 6, -2.0, 400.0, -12.0)
    assert torch.equal(Y1, Y2) and torch.equal(F1, F2)
    assert _relerr(Y1.cpu().numpy(), om.apply(X, eps), mask) <= TOL_APPLY
    for variant in (0, 3):
        gm.set_variant(variant)
        Ya = gm.apply_H(Xd, eps=ed)
        Fa = gm.cheb_filter(Xd.clone(), 6, -2.0, 400.0, -12.0)
        assert float(torch.linalg.norm(Ya - Y1) / torch.linalg.norm(Y1)) <= 1e-14
        assert float(torch.linalg.norm(Fa - F1) / torch.linalg.norm(F1)) <= 1e-13


@pytest.mark.parametrize("p,B", [(2, 4), (4, 10), (6, 7)])
def test_adjoint_right_hand_side(p, B):
    """Eq. 18 assembled from the device pieces — fe_apply_potential (int N_a U psi), the occupancy scaling, and
    fe_add_subspace for the (D + D^T) term — against the oracle's explicit-quadrature g~ (NEXT-4)."""
    import oracle
    fe = _fe()
    om = oracle.OracleMesh(*UNEQUAL, p)
    gm = fe.FEMesh(*UNEQUAL, p)
    gm.set_potential(_coulomb(gm.quad_coords()))  # the stored potential must not leak into the result
    mask = om.mask()
    Psi = workloads.random_block(950 + p, om.N, B, mask)
    f = 2.0 * workloads.uniform01(951 + p, 0, B)
    D = workloads.normal(952 + p, B * B).reshape(B, B)
    Uq = np.cos(om.quad_coords()).prod(axis=1) - 0.3  # any smooth field at the quadrature points (4 w (rho_data - rho))
    Go = oracle.adjoint_rhs(om, Psi, f, Uq, D)
    Pd = _dev(Psi)
    G = gm.apply_potential(_dev(Uq), Pd)
    G *= _dev(f)[None, :]
    gm.add_subspace(Pd, -(D + D.T), G)
    assert _relerr(G.cpu().numpy(), Go, mask) <= TOL_APPLY
    assert np.all(G.cpu().numpy()[mask == 0] == 0)
    # the operator set by fe_set_potential is untouched
    X = workloads.random_block(953, om.N, 4, mask)
    om.set_potential(_coulomb(om.quad_coords()))
    om.assemble()
    assert _relerr(gm.apply_H(_dev(X)).cpu().numpy(), om.apply(X), mask) <= TOL_APPLY


# ---- full BASELINE sizes: sampled rows ------------------------------------------------------------------------------
def _sample_rows(w, count, seed):
    """Rows spread over cell interiors, faces, edges, vertices and the boundary."""
    nx, ny, nz = w.nodes_per_axis
    u = workloads.uniform01(seed, 0, 3 * count).reshape(count, 3)
    gx, gy, gz = (np.minimum((u[:, d] * n).astype(np.int64), n - 1) for d, n in enumerate((nx, ny, nz)))
    # force a share of the rows onto cell faces / edges / vertices
    k = count // 4
    gx[:k] = (gx[:k] // w.p) * w.p
    gy[:k // 2] = (gy[:k // 2] // w.p) * w.p
    gz[:k // 4] = (gz[:k // 4] // w.p) * w.p
    return np.unique(gx + nx * (gy + ny * gz))


@pytest.mark.parametrize("cfg", [2, 5, 3])
def test_apply_full_size_sampled_rows(cfg):
    """Full BASELINE sizes in the launch configuration bench.py times; the oracle computes sampled rows one by one
    straight from Eq. 17 (orc_apply_rows)."""
    import oracle
    fe = _fe()
    w = workloads.config(cfg)
    om = oracle.OracleMesh(w.xe, w.ye, w.ze, w.p)
    Vq = w.V(om.quad_coords())
    om.set_potential(Vq, build=False)
    gm = fe.FEMesh(w.xe, w.ye, w.ze, w.p)
    gm.set_potential(Vq)
    assert np.array_equal(gm.mask(), om.mask())
    X = w.X(om.mask())
    eps = w.eps()
    rows = _sample_rows(w, 96 if cfg != 3 else 48, 9000 + cfg)
    Yo = om.apply_rows(X, rows, eps)
    Xd = _dev(X)
    Yg = gm.apply_H(Xd, eps=_dev(eps) if eps is not None else None)
    Ys = Yg[torch.as_tensor(rows, device="cuda")].cpu().numpy()
    assert np.linalg.norm(Ys - Yo) <= TOL_APPLY * np.linalg.norm(Yo)
    # boundary rows are written 0 everywhere
    bnd = torch.as_tensor(np.flatnonzero(om.mask() == 0), device="cuda")
    assert float(Yg[bnd].abs().max()) == 0.0


# ---- the persistent loop of k_apply_tma (default at p = 5, 7, 8 and the 32-wide p = 6 shape; variants 7 / 8 elsewhere) ----
BIG = (np.array([0.0, 0.5, 1.1, 1.5, 2.2, 2.6, 3.3]), np.array([-1.0, -0.6, 0.1, 0.5, 1.2, 1.5, 2.0]),
       np.array([0.0, 0.4, 0.7, 1.3, 1.6, 2.1]))  # 6 x 6 x 5 = 180 unequal cells: more units than the 148 persistent CTAs


@pytest.mark.parametrize("p,B,variant", [(5, 6, 0), (5, 34, 0), (5, 34, 7), (7, 6, 0), (7, 34, 0), (8, 6, 0), (8, 34, 0), (6, 34, 0),
                                         (2, 130, 7), (3, 130, 7), (4, 130, 7), (6, 34, 7), (6, 6, 8), (6, 34, 8), (6, 34, 6)])
def test_persistent_loop_parity(p, B, variant):
    """(p = 5, variant 0 is the two-CTAs-per-SM SLIM shape, one unit per CTA; variant 7 its persistent predecessor.)
    A mesh with more units than resident CTAs, so that every persistent CTA walks several units (bar[1] handshake,
    rec / recN swap, mid-unit next-tile request, the BT = 16 shape with two planes per warp at p = 7, 8; B = 130 gives
    the several-CTAs-per-SM shapes of p <= 4 more units than their 888 / 592 / 444 resident CTAs).  One shifted
    apply: sampled rows against the oracle's entry-by-entry Eq. 17 and ALL rows against the colour-ordered legacy kernel
    (variant 4, the race oracle of R17).  A degree-5 filter: against the legacy kernel's recurrence."""
    import oracle
    fe = _fe()
    om = oracle.OracleMesh(*BIG, p)
    Vq = _coulomb(om.quad_coords())
    om.set_potential(Vq, build=False)
    gm = fe.FEMesh(*BIG, p)
    gm.set_potential(Vq)
    mask = om.mask()
    X = workloads.random_block(1300 + p, om.N, B)  # data in the Dirichlet rows: ignored
    eps = workloads.shifts(2300 + p, B)
    rows = np.unique((workloads.uniform01(9300 + p, 0, 120) * om.N).astype(np.int64))
    Yo = om.apply_rows(X * mask[:, None], rows, eps)
    Xd, ed = _dev(X), _dev(eps)
    gm.set_variant(4)
    Yref = gm.apply_H(Xd, eps=ed).clone()
    Fref = gm.cheb_filter(Xd.clone(), 5, -2.0, 900.0, -12.0)
    gm.set_variant(variant)
    Yg = gm.apply_H(Xd, eps=ed)
    Ys = Yg[torch.as_tensor(rows, device="cuda")].cpu().numpy()
    assert np.linalg.norm(Ys - Yo) <= TOL_APPLY * np.linalg.norm(Yo)
    assert float(torch.linalg.norm(Yg - Yref) / torch.linalg.norm(Yref)) <= 1e-13
    assert np.all(Yg.cpu().numpy()[mask == 0] == 0)
    Fg = gm.cheb_filter(Xd.clone(), 5, -2.0, 900.0, -12.0)
    assert float(torch.linalg.norm(Fg - Fref) / torch.linalg.norm(Fref)) <= 1e-12
    assert np.all(Fg.cpu().numpy()[mask == 0] == 0)


def test_adjoint_scratch_survives_host_filter():
    """One handle: fe_apply_potential, then cheb_filter_host on a wider block (its staging is regrown), then
    fe_apply_potential again -- the adjoint scratch must stay valid across the regrowth."""
    import oracle
    fe = _fe()
    p = 3
    om = oracle.OracleMesh(*UNEQUAL, p)
    gm = fe.FEMesh(*UNEQUAL, p)
    Vq = _coulomb(om.quad_coords())
    om.set_potential(Vq)
    om.assemble()
    gm.set_potential(Vq)
    mask = om.mask()
    Uq = np.cos(om.quad_coords()).prod(axis=1) - 0.3
    Psi = workloads.random_block(1400, om.N, 6, mask)
    Go = oracle.adjoint_rhs(om, Psi, np.ones(6), Uq, np.zeros((6, 6)))
    G1 = gm.apply_potential(_dev(Uq), _dev(Psi)).cpu().numpy()
    assert _relerr(G1, Go, mask) <= TOL_APPLY
    for B in (4, 64, 96):  # growing staging
        Xh = workloads.random_block(1401 + B, om.N, B, mask)
        Yo = om.filter(Xh, 4, 3.0, 2500.0, -10.0)
        gm.cheb_filter_host(Xh, 4, 3.0, 2500.0, -10.0)
        assert _relerr(Xh, Yo, mask) <= TOL_FILTER
        G2 = gm.apply_potential(_dev(Uq), _dev(Psi)).cpu().numpy()
        assert _relerr(G2, Go, mask) <= TOL_APPLY


def test_nan_in_dirichlet_rows_is_ignored():
    """R5: boundary rows of X are IGNORED -- even NaN / Inf there (an uninitialised block) must not reach any free node, in
    fe_apply_H (both kernel generations), cheb_filter, fe_density and fe_apply_potential."""
    om, gm = _pair(UNEQUAL, 4, _coulomb)
    mask = om.mask()
    B = 6
    X = workloads.random_block(1500, om.N, B, mask)
    Xbad = X.copy()
    bnd = np.flatnonzero(mask == 0)
    Xbad[bnd[0::3]] = np.nan
    Xbad[bnd[1::3]] = np.inf
    Xbad[bnd[2::3]] = -np.inf
    Yo = om.apply(X)
    for variant in (0, 3):
        gm.set_variant(variant)
        Yg = gm.apply_H(_dev(Xbad)).cpu().numpy()
        assert np.all(np.isfinite(Yg)) and _relerr(Yg, Yo, mask) <= TOL_APPLY and np.all(Yg[mask == 0] == 0)
        Fg = gm.cheb_filter(_dev(Xbad).clone(), 5, -2.0, 400.0, -12.0).cpu().numpy()
        assert np.all(np.isfinite(Fg)) and _relerr(Fg, om.filter(X, 5, -2.0, 400.0, -12.0), mask) <= TOL_FILTER
    gm.set_variant(0)
    import oracle
    f = np.ones(B)
    rho = gm.density(_dev(Xbad), _dev(f)).cpu().numpy()
    assert np.all(np.isfinite(rho)) and np.linalg.norm(rho - oracle.density(om, X, f).reshape(-1)) <= 1e-12 * np.linalg.norm(rho)
    Uq = np.cos(om.quad_coords()).prod(axis=1)
    G = gm.apply_potential(_dev(Uq), _dev(Xbad)).cpu().numpy()
    assert np.all(np.isfinite(G))


@pytest.mark.parametrize("p,B", [(2, 6), (4, 34), (6, 8), (3, 5)])
def test_apply_chain(p, B):
    """fe_apply_H_chain on the unequal mesh: three chained applies into two alternating blocks equal three fe_apply_H calls;
    B = 5 takes the fallback (plain apply + memset of the next target)."""
    om, gm = _pair(UNEQUAL, p, _coulomb)
    mask = om.mask()
    eps = workloads.shifts(2700 + p, B)
    Xs = [workloads.random_block(1700 + p + i, om.N, B) for i in range(3)]  # Dirichlet rows hold data
    Y = [torch.full((om.N, B), 9.0, dtype=torch.float64, device="cuda"), torch.full((om.N, B), -7.0, dtype=torch.float64, device="cuda")]
    for t in range(3):
        gm.apply_H_chain(_dev(Xs[t]), Y[t % 2], Y[(t + 1) % 2], _dev(eps), y_is_clear=(t > 0))
        Yg = Y[t % 2].cpu().numpy()
        assert _relerr(Yg, om.apply(Xs[t], eps), mask) <= TOL_APPLY, t
        assert np.all(Yg[mask == 0] == 0)
    gm.apply_H_chain(_dev(Xs[0]), Y[1], None, None, y_is_clear=True)  # last link: nothing to clear, no shift
    assert _relerr(Y[1].cpu().numpy(), om.apply(Xs[0]), mask) <= TOL_APPLY


# ---- error behaviour -------------------------------------------------------------------------------------------------
def test_error_codes():
    fe = _fe()
    e = np.array([0.0, 1.0, 2.0])
    with pytest.raises(fe.FEError):
        fe.FEMesh(e, e, e, 9)
    with pytest.raises(fe.FEError):
        fe.FEMesh(np.array([0.0, 1.0, 1.0]), e, e, 2)
    gm = fe.FEMesh(e, e, e, 2)
    X = torch.zeros(gm.N, 4, dtype=torch.float64, device="cuda")
    with pytest.raises(fe.FEError) as ei:
        gm.apply_H(X)
    assert ei.value.code == -4  # before fe_set_potential
    gm.set_potential(np.zeros(gm.ncells * gm.nq3))
    with pytest.raises(fe.FEError):
        fe.fe_apply_H(gm.h, X, X)  # aliasing
    with pytest.raises(fe.FEError):
        gm.cheb_filter(X, 3, 2.0, 1.0, 0.0)  # needs a0 < a < b
    with pytest.raises(fe.FEError):
        gm.cheb_filter(X, 0, 1.0, 2.0, 0.0)
    assert gm.launches >= 2
