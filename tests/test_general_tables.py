"""Host logic of the general-mesh path, no GPU needed: the library's numbering, hanging-node constraints, coordinates,
lumped mass and Dirichlet mask (built with integer node keys, fe_general.cpp) against the oracle's (built by geometric
matching, oracle/fe_general.py).  l2g and mask must match bit-exactly (BASELINE.json), weights and coordinates to rounding."""
import numpy as np
import pytest

import oracle
import workloads


def _meshes():
    e3 = workloads.uniform_edges(-1.5, 1.5, 3)
    e4 = workloads.uniform_edges(-2.0, 2.0, 4)
    ball = lambda r: (lambda l, lo, hi: np.linalg.norm((lo + hi) / 2) < r[l])
    wave = lambda x: x + 0.06 * np.sin(1.3 * x[:, [1, 2, 0]] + 0.4)
    shear = lambda x: x @ np.array([[1.0, 0.3, -0.2], [0.1, 0.9, 0.25], [-0.15, 0.2, 1.1]]).T
    corner = lambda l, lo, hi: bool(np.all(lo < -0.4)) if l == 0 else bool(np.all(lo < -1.2))  # refinement against the boundary
    yield "one-level", workloads.octree_mesh(e3, e3, e3, ball({0: 0.9}), 1, wave)
    yield "two-level", workloads.octree_mesh(e4, e4, e4, ball({0: 1.3, 1: 0.6}), 2, shear)
    yield "boundary", workloads.octree_mesh(e3, np.array([0.0, 0.5, 1.5]), e3, corner, 2, None)
    yield "unrefined", workloads.octree_mesh(e3, e3, np.array([0.0, 1.0]), lambda l, lo, hi: False, 0, wave)


@pytest.mark.parametrize("p", [1, 2, 3, 5])
def test_tables_match_the_oracle(p):
    import paper_2510_10529_b200 as fe
    for name, mesh in _meshes():
        om = oracle.GeneralOracleMesh(mesh, p)
        gm = fe.FEMesh.general(mesh, p, device=-1)
        assert (gm.N, gm.N_all, gm.N_free, gm.ncells, gm.nc) == (om.N, om.N_all, om.N_free, om.ncells, om.nc), name
        assert np.array_equal(gm.l2g(), om.l2g()), name
        assert np.array_equal(gm.mask(), om.mask()), name
        rp, col, val = gm.constraints()
        Cg = np.zeros((om.N_all - om.N, om.N))
        for r in range(len(rp) - 1):
            assert np.all(col[rp[r]:rp[r + 1]] < om.N)
            Cg[r, col[rp[r]:rp[r + 1]]] = val[rp[r]:rp[r + 1]]
        if om.N_all > om.N:
            assert np.max(np.abs(Cg - om.constraint_matrix())) < 1e-13, name
        scale = np.abs(om.node_coords()).max()
        assert np.max(np.abs(gm.node_coords() - om.node_coords())) < 1e-14 * scale, name
        assert np.max(np.abs(gm.quad_coords() - om.quad_coords())) < 1e-14 * scale, name
        assert np.max(np.abs(gm.mass() / om.mass() - 1.0)) < 1e-12, name
        gm.close()


def test_bad_leaf_lists_are_rejected():
    import paper_2510_10529_b200 as fe
    e = workloads.uniform_edges(0.0, 2.0, 2)
    mesh = workloads.octree_mesh(e, e, e, lambda l, lo, hi: l == 0 and bool(np.all(lo < 0.5)), 1)
    cells, verts = mesh.cells.copy(), mesh.verts.copy()
    with pytest.raises(fe.FEError):  # a leaf listed twice
        fe.fe_mesh_create_general(2, 2, 2, np.vstack([cells, cells[:1]]), np.concatenate([verts, verts[:1]]), 2, -1)
    with pytest.raises(fe.FEError):  # a leaf outside the root grid
        bad = cells.copy(); bad[-1, 1] = 9
        fe.fe_mesh_create_general(2, 2, 2, bad, verts, 2, -1)
    with pytest.raises(fe.FEError):  # 2:1 balance violated: a level-2 leaf next to a level-0 leaf
        c2 = np.array([[0, 1, 0, 0], [2, 3, 0, 0]], dtype=np.int32)
        fe.fe_mesh_create_general(2, 1, 1, c2, np.zeros((2, 8, 3)) + np.arange(8)[None, :, None], 2, -1)
    with pytest.raises(fe.FEError):
        fe.fe_mesh_create_general(2, 2, 2, cells, verts, 9, -1)
