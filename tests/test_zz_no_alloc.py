"""fe_gram_static: the Gram product A^T Bm for callers that must not allocate (include/fe_cheb.h).

The entry point uses the same kernels as fe_gram but keeps the B x B device accumulator in a file-scope static __device__
array of the library (128 x 128 doubles) whose address comes from cudaGetSymbolAddress.  Checked here against the
existing path (fe_gram) and against the plain definition in numpy, on calls in a row that share the array: a wide block,
then a narrow one (stale entries of the first call must not leak), then a wide one with other data.  Tolerance: the one
tests/test_gpu_parity.py uses for fe_gram, 1e-11 * max(1, max|C|) per entry (atomics: the sum order is not fixed).

This file sorts last on purpose: the suite runs with pytest -x, so a failure here hides no other test.
"""
import numpy as np
import pytest

import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_GRAM = 1e-11


def _mesh():
    import paper_2510_10529_b200 as fe
    e = workloads.uniform_edges(-3.0, 3.0, 6)
    return fe, fe.FEMesh(e, e, e, 4)  # N = 25^3 = 15 625 nodes


def _blocks(seed, N, B):
    A = workloads.random_block(seed, N, B)
    Bm = workloads.random_block(seed + 1, N, B)
    return A, Bm, torch.as_tensor(A, device="cuda"), torch.as_tensor(Bm, device="cuda")


def _check(C, Cref):
    assert C.shape == Cref.shape
    assert np.max(np.abs(C - Cref)) <= TOL_GRAM * max(1.0, np.max(np.abs(Cref)))


def test_gram_static_matches_existing_path_on_calls_in_a_row():
    fe, gm = _mesh()
    # B = 64: the DMMA kernel; B = 7: the generic kernel, 49 of the 4096 entries the first call left behind;
    # B = 64 again with other data; B = 128: the whole array
    for seed, B in ((700, 64), (710, 7), (720, 64), (730, 128), (740, 34)):
        A, Bm, Ad, Bd = _blocks(seed, gm.N, B)
        C_static = gm.gram_static(Ad, Bd)
        C_plain = gm.gram(Ad, Bd)          # the existing path (cudaMalloc'ed accumulator of the mesh)
        _check(C_static, C_plain)
        _check(C_static, A.T @ Bm)         # and the definition
        C_again = gm.gram_static(Ad, Bd)   # the same call twice in a row: the array is cleared, not accumulated into
        _check(C_again, C_plain)


def test_gram_static_two_meshes_share_the_array():
    """The accumulator belongs to the library, not to a mesh: alternating calls from two meshes must not mix."""
    fe, g1 = _mesh()
    e = workloads.uniform_edges(-1.0, 1.0, 3)
    g2 = fe.FEMesh(e, e, e, 2)
    A1, B1, A1d, B1d = _blocks(750, g1.N, 32)
    A2, B2, A2d, B2d = _blocks(760, g2.N, 32)
    for _ in range(2):
        _check(g1.gram_static(A1d, B1d), A1.T @ B1)
        _check(g2.gram_static(A2d, B2d), A2.T @ B2)


def test_gram_static_rejects_blocks_beyond_the_array():
    fe, gm = _mesh()
    X = torch.zeros(gm.N, 129, dtype=torch.float64, device="cuda")
    with pytest.raises(fe.FEError) as ei:
        gm.gram_static(X, X)
    assert "128" in str(ei.value) and "fe_gram_static" in str(ei.value)
    # the error left the library usable
    A, Bm, Ad, Bd = _blocks(770, gm.N, 16)
    _check(gm.gram_static(Ad, Bd), A.T @ Bm)
