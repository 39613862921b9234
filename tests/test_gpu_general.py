"""GPU parity of the general-hexahedral / hanging-node path (NEXT-3: fe_mesh_create_general; fe_general.cuh) against its
oracle (oracle/fe_general.py) on the same seeded inputs: <= 1e-11 for one apply (plain and shifted), <= 1e-9 after
cheb_filter and on Ritz values (R16); Dirichlet rows of the input ignored, of the output exactly 0."""
import numpy as np
import pytest

import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_APPLY = 1e-11
TOL_FILTER = 1e-9


def _dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


def _relerr(Yg, Yo, mask):
    free = mask.astype(bool)
    return np.linalg.norm(Yg[free] - Yo[free]) / max(np.linalg.norm(Yo[free]), 1e-300)


def _wave(x):
    return x + 0.06 * np.sin(1.3 * x[:, [1, 2, 0]] + 0.4)


def _atom_mesh(levels, roots=4, half=4.0, deform=_wave):
    """Root grid on [-half, half]^3 refined `levels` times around the atom at the origin (a mesh vertex, l.151)."""
    e = workloads.uniform_edges(-half, half, roots)
    r = {0: 0.45 * half, 1: 0.25 * half}
    return workloads.octree_mesh(e, e, e, lambda l, lo, hi: np.linalg.norm((lo + hi) / 2) < r[l], levels, deform)


def _pair(mesh, p, V):
    import oracle
    import paper_2510_10529_b200 as fe
    om = oracle.GeneralOracleMesh(mesh, p)
    Vq = V(om.quad_coords())
    om.set_potential(Vq)
    gm = fe.FEMesh.general(mesh, p)
    gm.set_potential(Vq)
    assert np.array_equal(gm.l2g(), om.l2g()) and np.array_equal(gm.mask(), om.mask())
    return om, gm


def _coulomb(q):
    return -4.0 / np.sqrt((q ** 2).sum(axis=1) + 0.25)


@pytest.mark.parametrize("p,B", [(1, 5), (2, 34), (3, 6), (4, 33), (5, 6), (6, 18), (7, 5), (7, 34), (8, 10)])
def test_apply_refined_deformed_mesh_all_orders(p, B):
    """One-level refinement of a 3^3 root grid with smoothly displaced vertices (non-constant Jacobians, hanging faces and
    edges): plain and shifted apply, ragged vector tiles, data in the Dirichlet rows.  (7, 34): 83 leaves x 5 vector tiles are
    more units than resident CTAs, so the persistent p = 7 kernel walks several units per CTA (prefetched rows, rotating fields)."""
    e = workloads.uniform_edges(-1.5, 1.5, 3)
    mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: np.linalg.norm((lo + hi) / 2) < 0.9, 1, _wave)
    om, gm = _pair(mesh, p, _coulomb)
    mask = om.mask()
    X = workloads.random_block(1500 + p, om.N, B)  # boundary rows NOT zeroed
    eps = workloads.shifts(2500 + p, B)
    Yg = gm.apply_H(_dev(X)).cpu().numpy()
    assert _relerr(Yg, om.apply(X), mask) <= TOL_APPLY
    assert np.all(Yg[mask == 0] == 0)
    Yg = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert _relerr(Yg, om.apply(X, eps), mask) <= TOL_APPLY
    assert np.all(Yg[mask == 0] == 0)
    Xbad = X.copy()
    Xbad[mask == 0] = np.nan  # R5: even NaN in the Dirichlet rows (also those feeding hanging nodes) is ignored
    Yg = gm.apply_H(_dev(Xbad)).cpu().numpy()
    assert np.all(np.isfinite(Yg)) and _relerr(Yg, om.apply(X), mask) <= TOL_APPLY


@pytest.mark.parametrize("p,B,deg", [(2, 8, 7), (4, 16, 10), (6, 6, 4)])
def test_two_level_refinement_around_an_atom(p, B, deg):
    """The verdict's target case: a mesh refined twice around one soft-Coulomb atom sitting on a mesh vertex (l.151, l.273),
    sheared so that the metric is a full 3 x 3 matrix.  Apply <= 1e-11, cheb_filter <= 1e-9 with bounds from the oracle's
    20-step Lanczos (R10), the device Lanczos bounds against the oracle's."""
    import oracle
    shear = lambda x: x @ np.array([[1.0, 0.15, -0.1], [0.05, 0.95, 0.12], [-0.08, 0.1, 1.05]]).T
    mesh = _atom_mesh(2, deform=shear)
    assert (mesh.cells[:, 0] == 2).any()
    om, gm = _pair(mesh, p, _coulomb)
    assert om.N_all > om.N
    mask = om.mask()
    X = workloads.random_block(1600 + p, om.N, B)
    Yg = gm.apply_H(_dev(X)).cpu().numpy()
    assert _relerr(Yg, om.apply(X), mask) <= TOL_APPLY
    v0 = workloads.normal(3600 + p, om.N)
    lo_o, hi_o, be_o = oracle.lanczos_bounds(om, v0, 20)
    lo_g, hi_g, be_g = gm.lanczos_bounds(_dev(v0), 20)
    scale = max(abs(hi_o), 1.0)
    assert abs(lo_g - lo_o) <= 1e-8 * scale and abs(hi_g - hi_o) <= 1e-8 * scale and abs(be_g - be_o) <= 1e-7 * scale
    b, a0 = hi_o + be_o, lo_o
    a = a0 + 0.1 * (b - a0)
    Fo = om.filter(X, deg, a, b, a0)
    work = torch.full((2 * om.N * B,), -3.25, dtype=torch.float64, device="cuda")  # dirty work space
    Fg = gm.cheb_filter(_dev(X).clone(), deg, a, b, a0, work).cpu().numpy()
    assert _relerr(Fg, Fo, mask) <= TOL_FILTER
    assert np.all(Fg[mask == 0] == 0)


def test_chfsi_on_a_refined_mesh():
    """Filter + Rayleigh-Ritz cycles with the residual stopping rule (l.296) on a hanging-node mesh: harmonic oscillator on
    [-6,6]^3, p=3, the 8 central root cells refined -- same number of cycles as the oracle, Ritz values <= 1e-9, and the
    lowest level near 1.5 (the refinement pin of tests/test_general_pins.py, now through the device path)."""
    import oracle
    e = workloads.uniform_edges(-6.0, 6.0, 4)
    mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: np.abs((lo + hi) / 2).max() < 3.0, 1)
    om, gm = _pair(mesh, 3, workloads.harmonic)
    mask = om.mask()
    B, n_gate, t_eig = 10, 4, 1e-6
    X0 = workloads.random_block(1700, om.N, B, mask)
    lo, hi, be = oracle.lanczos_bounds(om, workloads.normal(3700, om.N), 20)
    b, a0 = hi + be, lo
    a = a0 + 0.1 * (b - a0)
    theta_o, _, res_o, cyc_o = oracle.chfsi(om, X0, 12, a, b, a0, t_eig, n_gate, max_cycles=40)
    Xg = _dev(X0)
    theta_g, res_g, cyc_g = gm.chfsi(Xg, 12, a, b, a0, t_eig, n_gate, max_cycles=40)
    assert cyc_g == cyc_o and 1 < cyc_g < 40
    assert np.max(np.abs(theta_g - theta_o) / np.maximum(1.0, np.abs(theta_o))) <= 1e-9
    assert res_g[:n_gate].max() <= t_eig
    assert abs(theta_g[0] - 1.5) < 2e-3
    Q = Xg.cpu().numpy()
    assert np.max(np.abs(Q.T @ Q - np.eye(B))) <= 1e-12 and np.all(Q[mask == 0] == 0)


def test_unrefined_box_mesh_agrees_with_the_tensor_product_path():
    """The same box mesh through both generations of the library: the general kernel (explicit l2g, 12 sweeps, full metric)
    and the TMA kernel (closed-form l2g, 10 sweeps) must agree to rounding once the rows are matched through the l2g."""
    import paper_2510_10529_b200 as fe
    xe, ye, ze = np.array([0.0, 0.7, 2.0, 2.6]), np.array([-1.0, -0.5, 0.4, 1.0]), np.array([0.0, 0.3, 1.0])
    mesh = workloads.octree_mesh(xe, ye, ze, lambda l, lo, hi: False, 0)
    p, B = 4, 8
    gt = fe.FEMesh(xe, ye, ze, p)
    gg = fe.FEMesh.general(mesh, p)
    Vq = _coulomb(gt.quad_coords())
    assert np.max(np.abs(gg.quad_coords() - gt.quad_coords())) < 1e-14
    gt.set_potential(Vq)
    gg.set_potential(Vq)
    perm = np.empty(gt.N, dtype=np.int64)
    perm[gt.l2g().reshape(-1)] = gg.l2g().reshape(-1)  # tensor id -> general id
    X = workloads.random_block(1800, gt.N, B)
    Xg = np.empty_like(X)
    Xg[perm] = X
    Yt = gt.apply_H(_dev(X)).cpu().numpy()
    Yg = gg.apply_H(_dev(Xg)).cpu().numpy()[perm]
    assert np.linalg.norm(Yg - Yt) <= 1e-13 * np.linalg.norm(Yt)


@pytest.mark.parametrize("precondition", [False, True])
def test_block_minres_on_a_hanging_node_mesh(precondition):
    """fe_minres_shifted (l.221-225) on a refined, smoothly deformed mesh: the same Paige-Saunders iteration as the oracle's,
    compared after a fixed 25 steps (<= 1e-9) and at convergence through the true residual with the oracle's operator; the
    preconditioner of reading R27 against the oracle's (through the iterates: both sides build their own)."""
    import oracle
    e = workloads.uniform_edges(-1.5, 1.5, 3)
    mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: np.linalg.norm((lo + hi) / 2) < 0.9, 1, _wave)
    om, gm = _pair(mesh, 3, _coulomb)
    mask = om.mask()
    free = mask.astype(bool)
    B = 6
    G = workloads.random_block(1900, om.N, B)  # Dirichlet rows hold data that must be ignored
    eps = workloads.shifts(2900, B)
    Mi = om.laplacian_precond() if precondition else None
    Xo, relo, ito = oracle.minres_shifted(om, G, eps, maxit=25, tol=0.0, Minv=Mi)
    Xg, relg, itg = gm.minres_shifted(_dev(G), _dev(eps), maxit=25, tol=0.0, precondition=precondition)
    Xg = Xg.cpu().numpy()
    assert itg == 25 and ito == 25
    assert _relerr(Xg, Xo, mask) <= 1e-9
    assert np.max(np.abs(relg - relo)) <= 1e-9
    assert np.all(Xg[~free] == 0)
    Xc, relc, itc = gm.minres_shifted(_dev(G), _dev(eps), maxit=4000, tol=1e-9, precondition=precondition)
    R = (om.apply(Xc.cpu().numpy(), eps) - G * mask[:, None])[free]
    assert np.all(relc <= 1e-9) and itc < 4000
    assert np.linalg.norm(R) <= 1e-6 * np.linalg.norm(G[free])
    if precondition:
        _, _, it_plain = gm.minres_shifted(_dev(G), _dev(eps), maxit=4000, tol=1e-9, precondition=False)
        assert itc < it_plain


@pytest.mark.parametrize("p,B", [(1, 3), (2, 8), (3, 33), (4, 20), (6, 9), (7, 12), (8, 5)])
def test_density_and_potential_apply_on_a_hanging_node_mesh(p, B):
    """fe_density (Eq. 4) and fe_apply_potential (the integral of Eq. 18) on a refined, smoothly deformed mesh against the
    oracle's definitions: several vector tiles, ragged tails, data in the Dirichlet rows; the operator set by
    fe_set_potential is untouched afterwards."""
    e = workloads.uniform_edges(-1.5, 1.5, 3)
    mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: np.linalg.norm((lo + hi) / 2) < 0.9, 1, _wave)
    om, gm = _pair(mesh, p, _coulomb)
    mask = om.mask()
    X = workloads.random_block(2000 + p, om.N, B)
    f = 2.0 * workloads.uniform01(2001 + p, 0, B)
    rho_o = om.density(X, f).reshape(-1)
    rho_g = gm.density(_dev(X), _dev(f)).cpu().numpy()
    assert np.linalg.norm(rho_g - rho_o) <= 1e-12 * np.linalg.norm(rho_o)
    Uq = np.cos(om.quad_coords()).prod(axis=1) - 0.3
    Yo = om.potential_apply(Uq, X * mask[:, None])
    Yg = gm.apply_potential(_dev(Uq), _dev(X)).cpu().numpy()
    assert _relerr(Yg, Yo, mask) <= TOL_APPLY
    assert np.all(Yg[mask == 0] == 0)
    assert _relerr(gm.apply_H(_dev(X)).cpu().numpy(), om.apply(X), mask) <= TOL_APPLY


def test_colour_ordered_scatter_on_a_hanging_node_mesh():
    """Variant 4 on a general mesh (S8(a) a3 "atomic or colour-ordered"): cells launched colour by colour, collapse over the
    transposed rows -- two runs are bit-identical, the result matches the oracle, and the atomic path agrees with it to
    rounding (the deterministic mode doubles as a race oracle, R17)."""
    mesh = _atom_mesh(2)
    om, gm = _pair(mesh, 3, _coulomb)
    mask = om.mask()
    B = 10
    X = workloads.random_block(2100, om.N, B, mask)
    eps = workloads.shifts(3100, B)
    Xd, ed = _dev(X), _dev(eps)
    gm.set_variant(4)
    Y1 = gm.apply_H(Xd, eps=ed).clone()
    Y2 = gm.apply_H(Xd, eps=ed).clone()
    F1 = gm.cheb_filter(Xd.clone(), 6, -2.0, 400.0, -12.0)
    F2 = gm.cheb_filter(Xd.clone(), 6, -2.0, 400.0, -12.0)
    assert torch.equal(Y1, Y2) and torch.equal(F1, F2)
    assert _relerr(Y1.cpu().numpy(), om.apply(X, eps), mask) <= TOL_APPLY
    gm.set_variant(0)
    Ya = gm.apply_H(Xd, eps=ed)
    Fa = gm.cheb_filter(Xd.clone(), 6, -2.0, 400.0, -12.0)
    assert float(torch.linalg.norm(Ya - Y1) / torch.linalg.norm(Y1)) <= 1e-14
    assert float(torch.linalg.norm(Fa - F1) / torch.linalg.norm(F1)) <= 1e-13


def test_adaptive_workload_full_size_properties():
    """The adaptive-molecule workload bench.py times (4 066 leaves on three levels, p = 6, 857 011 unconstrained + 100 507
    hanging nodes, B = 64), where the oracle's cell matrices are out of reach: (i) the operator is symmetric,
    <X, H~Y> = <H~X, Y> column by column -- gather, constraint expansion, scatter and collapse are transposes of each other at
    this size too; (ii) cheb_filter at the timed degree equals the three-term recurrence assembled from fe_apply_H calls,
    which the small-mesh tests tie to the oracle; (iii) Dirichlet rows stay exactly 0."""
    import paper_2510_10529_b200 as fe
    mesh, V = workloads.adaptive_molecule()
    gm = fe.FEMesh.general(mesh, 6)
    assert gm.N_all > gm.N and gm.ncells == mesh.ncells
    gm.set_potential(V(gm.quad_coords()))
    B, m = 64, 30
    mask = _dev(gm.mask().astype(np.float64))[:, None]
    gen = torch.Generator(device="cuda")
    gen.manual_seed(6100)
    X = torch.randn(gm.N, B, dtype=torch.float64, device="cuda", generator=gen) * mask
    Y = torch.randn(gm.N, B, dtype=torch.float64, device="cuda", generator=gen) * mask
    HX, HY = gm.apply_H(X), gm.apply_H(Y)
    # (0) sampled rows of one apply against the oracle's row-by-row definition (cell matrices by explicit quadrature on demand):
    # nodes inside refined cells, on coarse faces that hanging nodes depend on, and near the boundary
    import oracle
    om = oracle.GeneralOracleMesh(mesh, 6)
    assert np.array_equal(om.l2g(), gm.l2g())
    rp, col, _ = gm.constraints()
    masters_with_dependents = np.unique(col)
    pick = np.concatenate([masters_with_dependents[:: max(1, len(masters_with_dependents) // 5)][:5],
                           (workloads.uniform01(9600, 0, 7) * om.N).astype(np.int64)])
    rows = np.unique(pick)
    Yo = om.apply_rows(X.cpu().numpy(), rows, V(om.quad_coords()))
    Ys = HX[torch.as_tensor(rows, device="cuda")].cpu().numpy()
    assert np.linalg.norm(Ys - Yo) <= TOL_APPLY * np.linalg.norm(Yo)
    gm.set_variant(4)  # ALL rows against the colour-ordered deterministic path (no atomics anywhere): a race check at scale
    HXd = gm.apply_H(X)
    gm.set_variant(0)
    assert float(torch.linalg.norm(HX - HXd) / torch.linalg.norm(HXd)) <= 1e-14
    del HXd
    lhs, rhs = (X * HY).sum(dim=0), (HX * Y).sum(dim=0)
    scale = torch.sqrt((X * X).sum(dim=0) * (HY * HY).sum(dim=0))
    assert float(((lhs - rhs).abs() / scale).max()) <= 1e-12
    assert float((HX * (1 - mask)).abs().max()) == 0.0
    a0, a, b = -40.0, 20.0, 4000.0
    e, c = (b - a) / 2, (b + a) / 2
    s1 = e / (a0 - c)
    s = s1
    Ykm, Yk = X, (s1 / e) * (gm.apply_H(X) - c * X)
    for _ in range(1, m):
        sn = 1.0 / (2.0 / s1 - s)
        Ykm, Yk = Yk, (2 * sn / e) * (gm.apply_H(Yk) - c * Yk) - s * sn * Ykm
        s = sn
    Yf = gm.cheb_filter(X.clone(), m, a, b, a0)
    assert float(torch.linalg.norm(Yf - Yk) / torch.linalg.norm(Yk)) <= 1e-12
    assert float((Yf * (1 - mask)).abs().max()) == 0.0


def _graded_box_mesh(levels=1):
    """Undeformed octree leaves on an UNEQUALLY spaced root grid (hx != hy != hz, graded): every cell an axis-aligned box,
    one or two levels of refinement near a corner region so that hanging faces and edges appear."""
    ex = np.array([-1.6, -0.7, 0.1, 1.4])
    ey = np.array([-1.2, -0.5, 0.4, 1.3])
    ez = np.array([-1.5, -0.2, 0.5, 1.1])
    r = {0: 1.0, 1: 0.55}
    return workloads.octree_mesh(ex, ey, ez, lambda l, lo, hi: np.linalg.norm((lo + hi) / 2 - 0.2) < r[l], levels)


@pytest.mark.parametrize("p,B", [(1, 5), (2, 34), (3, 6), (4, 66), (5, 40), (6, 18), (6, 70), (7, 5), (7, 34), (8, 10)])
def test_box_cell_fast_path_on_octree_leaves(p, B):
    """A general mesh whose cells are all axis-aligned boxes (the paper's adaptive meshes: octree leaves of a box, l.273)
    takes the 10-sweep box-cell kernel of fe_gbox.cuh (p <= 7): apply (plain, shifted, NaN in the Dirichlet rows) against the
    oracle <= 1e-11, agreement with the generic 12-sweep kernel (variant 9), the colour-ordered mode bit-reproducible, and a
    filter <= 1e-9.  The larger B make the persistent CTAs walk several units (prefetched records and rows)."""
    mesh = _graded_box_mesh(2 if p <= 3 else 1)
    om, gm = _pair(mesh, p, _coulomb)
    assert om.N_all > om.N
    mask = om.mask()
    X = workloads.random_block(1900 + p, om.N, B)
    eps = workloads.shifts(2900 + p, B)
    Yo, Yoe = om.apply(X), om.apply(X, eps)
    Yg = gm.apply_H(_dev(X)).cpu().numpy()
    assert _relerr(Yg, Yo, mask) <= TOL_APPLY and np.all(Yg[mask == 0] == 0)
    Yge = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert _relerr(Yge, Yoe, mask) <= TOL_APPLY and np.all(Yge[mask == 0] == 0)
    Xbad = X.copy()
    Xbad[mask == 0] = np.nan
    Yb = gm.apply_H(_dev(Xbad)).cpu().numpy()
    assert np.all(np.isfinite(Yb)) and _relerr(Yb, Yo, mask) <= TOL_APPLY
    gm.set_variant(9)  # the generic kernel on the same handle
    Y9 = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert _relerr(Y9, Yoe, mask) <= TOL_APPLY and _relerr(Yge, Y9, mask) <= 1e-12
    gm.set_variant(4)  # colour-ordered scatter through the box-cell kernel
    Y4a = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    Y4b = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert np.array_equal(Y4a, Y4b) and _relerr(Y4a, Yoe, mask) <= TOL_APPLY
    gm.set_variant(0)
    import oracle
    lo_o, hi_o, be_o = oracle.lanczos_bounds(om, workloads.normal(3900 + p, om.N), 20)
    b, a0 = hi_o + be_o, lo_o
    a = a0 + 0.1 * (b - a0)
    deg = 7
    Fo = om.filter(X, deg, a, b, a0)
    work = torch.full((2 * om.N * B,), 7.5, dtype=torch.float64, device="cuda")
    Fg = gm.cheb_filter(_dev(X).clone(), deg, a, b, a0, work).cpu().numpy()
    assert _relerr(Fg, Fo, mask) <= TOL_FILTER and np.all(Fg[mask == 0] == 0)


@pytest.mark.parametrize("p,B", [(1, 224), (2, 160), (3, 130), (4, 100), (5, 70)])
def test_box_cell_kernel_walks_several_units_per_cta(p, B):
    """More (cell, vector tile) units than resident CTAs at the orders with several CTAs per SM (8, 6, 4, 3, 1 at p = 1..5):
    every CTA of the box-cell kernel walks several units (double-buffered records, rows of the next unit copied under plane
    phase 2, owner terms).  Shifted apply <= 1e-11 and a degree-8 filter <= 1e-9 against the oracle on the twice-refined mesh."""
    import oracle
    mesh = _graded_box_mesh(2 if p <= 4 else 1)
    om, gm = _pair(mesh, p, _coulomb)
    mask = om.mask()
    X = workloads.random_block(2100 + p, om.N, B)
    eps = workloads.shifts(3100 + p, B)
    Yg = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()
    assert _relerr(Yg, om.apply(X, eps), mask) <= TOL_APPLY and np.all(Yg[mask == 0] == 0)
    lo_o, hi_o, be_o = oracle.lanczos_bounds(om, workloads.normal(4100 + p, om.N), 20)
    b, a0 = hi_o + be_o, lo_o
    a = a0 + 0.1 * (b - a0)
    Fg = gm.cheb_filter(_dev(X).clone(), 8, a, b, a0).cpu().numpy()
    assert _relerr(Fg, om.filter(X, 8, a, b, a0), mask) <= TOL_FILTER and np.all(Fg[mask == 0] == 0)


@pytest.mark.parametrize("p,B", [(3, 6), (6, 10)])
def test_consumers_on_a_box_cell_mesh(p, B):
    """The consumers of the operator on a mesh that takes the box-cell kernel: block MINRES with the preconditioner of R27
    (shifted applies with the owner terms inside the kernel), the density, and fe_apply_potential -- which borrows the GENERIC
    kernel for one call (records with zero metric) and must leave the box-cell operator as it was."""
    import oracle
    mesh = _graded_box_mesh(1)
    om, gm = _pair(mesh, p, _coulomb)
    mask = om.mask()
    free = mask.astype(bool)
    X = workloads.random_block(2200 + p, om.N, B)
    eps = workloads.shifts(3200 + p, B)
    Xo, relo, ito = oracle.minres_shifted(om, X, eps, maxit=25, tol=0.0, Minv=om.laplacian_precond())
    Xg, relg, itg = gm.minres_shifted(_dev(X), _dev(eps), maxit=25, tol=0.0, precondition=True)
    assert itg == 25 and ito == 25
    assert _relerr(Xg.cpu().numpy(), Xo, mask) <= 1e-9 and np.max(np.abs(relg - relo)) <= 1e-9
    f = 2.0 * workloads.uniform01(2201 + p, 0, B)
    rho_o = om.density(X, f).reshape(-1)
    rho_g = gm.density(_dev(X), _dev(f)).cpu().numpy()
    assert np.linalg.norm(rho_g - rho_o) <= 1e-12 * np.linalg.norm(rho_o)
    Uq = np.cos(om.quad_coords()).prod(axis=1) - 0.3
    Yg = gm.apply_potential(_dev(Uq), _dev(X)).cpu().numpy()
    assert _relerr(Yg, om.potential_apply(Uq, X * mask[:, None]), mask) <= TOL_APPLY and np.all(Yg[~free] == 0)
    Yg = gm.apply_H(_dev(X), eps=_dev(eps)).cpu().numpy()  # the box-cell operator after the borrowed call
    assert _relerr(Yg, om.apply(X, eps), mask) <= TOL_APPLY
    # the host-buffer entry point (column chunks on two streams) against the device call, and a chain of applies
    a0, a, b = -3.0, 40.0, 900.0
    Fd = gm.cheb_filter(_dev(X).clone(), 5, a, b, a0).cpu().numpy()
    Xh = np.ascontiguousarray(X.copy())
    gm.cheb_filter_host(Xh, 5, a, b, a0)
    assert _relerr(Xh, Fd, mask) <= 1e-13 and np.all(Xh[~free] == 0)
    Y1 = torch.full((om.N, B), 3.0, dtype=torch.float64, device="cuda")
    Y2 = torch.full((om.N, B), -2.0, dtype=torch.float64, device="cuda")
    gm.apply_H_chain(_dev(X), Y1, Y2, _dev(eps), y_is_clear=False)
    assert _relerr(Y1.cpu().numpy(), om.apply(X, eps), mask) <= TOL_APPLY and float(Y2.abs().max()) == 0.0
    X2 = workloads.random_block(2300 + p, om.N, B)
    gm.apply_H_chain(_dev(X2), Y2, Y1, None, y_is_clear=True)  # the target the first call cleared; clears Y1 in turn
    assert _relerr(Y2.cpu().numpy(), om.apply(X2), mask) <= TOL_APPLY and float(Y1.abs().max()) == 0.0
