"""ctypes binding of include/fe_cheb.h: argument marshalling only (torch tensors -> raw device pointers, the
current torch stream -> cudaStream_t).  Function names are those of the C ABI; FEMesh is a small convenience
wrapper that owns a handle.  torch is used for device memory and streams, nothing else."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libfecheb.so")
_lib = None

EXPORTS = (
    "fe_mesh_create", "fe_mesh_destroy", "fe_num_nodes", "fe_num_free", "fe_num_cells", "fe_nodes_per_cell",
    "fe_quad_per_cell", "fe_get_l2g", "fe_get_node_coords", "fe_get_quad_coords", "fe_get_mass",
    "fe_get_dirichlet_mask", "fe_set_potential", "fe_apply_H", "cheb_filter", "cheb_filter_host", "fe_rayleigh_ritz", "fe_minres_shifted", "fe_add_subspace", "fe_gram", "fe_gram_static", "fe_density", "fe_lanczos_bounds", "fe_apply_potential",
    "fe_set_variant", "fe_diag_peak", "fe_ritz_residuals", "fe_chfsi", "fe_mesh_create_general", "fe_apply_H_chain",
    "fe_num_all_nodes", "fe_num_constraint_entries", "fe_get_constraints",
    "fe_launch_count", "fe_last_error",
)


class FEError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("fe_cheb error %d: %s" % (code, msg))
        self.code = code


def library_path():
    return _SO


def load_library():
    """Load libfecheb.so (built in-tree by build.py / __graft_entry__.build()).  Fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise FEError(-3, "CUDA extension %s is missing: run `python -m paper_2510_10529_b200.build` "
                          "(there is no CPU fallback)" % _SO)
    L = C.CDLL(_SO)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    L.fe_mesh_create.restype = C.c_int
    L.fe_mesh_create.argtypes = [dp, C.c_int, dp, C.c_int, dp, C.c_int, C.c_int, C.c_int, C.POINTER(vp)]
    L.fe_mesh_destroy.restype, L.fe_mesh_destroy.argtypes = C.c_int, [vp]
    L.fe_mesh_create_general.restype = C.c_int
    L.fe_mesh_create_general.argtypes = [C.c_int, C.c_int, C.c_int, vp, C.c_int64, vp, C.c_int, C.c_int, C.POINTER(vp)]
    L.fe_get_constraints.restype, L.fe_get_constraints.argtypes = C.c_int, [vp, vp, vp, vp]
    for name in ("fe_num_nodes", "fe_num_free", "fe_num_cells", "fe_launch_count", "fe_num_all_nodes",
                 "fe_num_constraint_entries"):
        getattr(L, name).restype, getattr(L, name).argtypes = C.c_int64, [vp]
    for name in ("fe_nodes_per_cell", "fe_quad_per_cell"):
        getattr(L, name).restype, getattr(L, name).argtypes = C.c_int, [vp]
    for name in ("fe_get_l2g", "fe_get_node_coords", "fe_get_quad_coords", "fe_get_mass", "fe_get_dirichlet_mask"):
        getattr(L, name).restype, getattr(L, name).argtypes = C.c_int, [vp, vp]
    L.fe_set_potential.restype, L.fe_set_potential.argtypes = C.c_int, [vp, vp, C.c_int, vp]
    L.fe_apply_H.restype, L.fe_apply_H.argtypes = C.c_int, [vp, vp, vp, C.c_int, vp, vp]
    L.fe_apply_H_chain.restype, L.fe_apply_H_chain.argtypes = C.c_int, [vp, vp, vp, vp, C.c_int, vp, C.c_int, vp]
    L.cheb_filter.restype = C.c_int
    L.cheb_filter.argtypes = [vp, vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, vp, vp]
    L.cheb_filter_host.restype = C.c_int
    L.cheb_filter_host.argtypes = [vp, vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
    L.fe_rayleigh_ritz.restype, L.fe_rayleigh_ritz.argtypes = C.c_int, [vp, vp, C.c_int, vp, vp, vp]
    L.fe_minres_shifted.restype = C.c_int
    L.fe_minres_shifted.argtypes = [vp, vp, vp, C.c_int, vp, C.c_int, C.c_double, C.c_int, vp, vp, vp, vp]
    L.fe_density.restype, L.fe_density.argtypes = C.c_int, [vp, vp, C.c_int, vp, vp, vp]
    L.fe_lanczos_bounds.restype, L.fe_lanczos_bounds.argtypes = C.c_int, [vp, vp, C.c_int, vp, vp, vp]
    L.fe_apply_potential.restype, L.fe_apply_potential.argtypes = C.c_int, [vp, vp, vp, vp, C.c_int, vp]
    L.fe_gram.restype, L.fe_gram.argtypes = C.c_int, [vp, vp, vp, C.c_int, vp, vp]
    L.fe_gram_static.restype, L.fe_gram_static.argtypes = C.c_int, [vp, vp, vp, C.c_int, vp, vp]
    L.fe_add_subspace.restype, L.fe_add_subspace.argtypes = C.c_int, [vp, vp, vp, vp, C.c_int, vp]
    L.fe_set_variant.restype, L.fe_set_variant.argtypes = C.c_int, [vp, C.c_int]
    L.fe_ritz_residuals.restype, L.fe_ritz_residuals.argtypes = C.c_int, [vp, vp, vp, C.c_int, vp, vp, vp]
    L.fe_chfsi.restype = C.c_int
    L.fe_chfsi.argtypes = [vp, vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                           vp, vp, vp, vp, vp]
    L.fe_diag_peak.restype, L.fe_diag_peak.argtypes = C.c_int, [C.c_int, C.c_int, C.c_double, dp]
    L.fe_last_error.restype, L.fe_last_error.argtypes = C.c_char_p, []
    _lib = L
    return L


def fe_last_error():
    return load_library().fe_last_error().decode()


def _check(rc):
    if rc != 0:
        raise FEError(rc, fe_last_error())


def _edges(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _stream(stream):
    if stream is not None:
        return C.c_void_p(int(stream))
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev_ptr(t, name, numel=None):
    """Raw device pointer of a contiguous float64 CUDA tensor."""
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise FEError(-1, "%s must be a contiguous float64 CUDA tensor" % name)
    if numel is not None and t.numel() != numel:
        raise FEError(-1, "%s has %d elements, expected %d" % (name, t.numel(), numel))
    return C.c_void_p(t.data_ptr())


# ---- the C ABI, same names ---------------------------------------------------------------------------------------
def fe_mesh_create(xe, ye, ze, p, cuda_device=0):
    L = load_library()
    (xa, xp), (ya, yp), (za, zp) = _edges(xe), _edges(ye), _edges(ze)
    h = C.c_void_p()
    _check(L.fe_mesh_create(xp, len(xa) - 1, yp, len(ya) - 1, zp, len(za) - 1, int(p), int(cuda_device), C.byref(h)))
    return h


def fe_mesh_create_general(cx, cy, cz, cells, verts, p, cuda_device=0):
    """cells: (ncells, 4) int32 rows (level, ix, iy, iz); verts: (ncells, 8, 3) float64 corners.  cuda_device=-1: tables only."""
    L = load_library()
    cells = np.ascontiguousarray(cells, dtype=np.int32)
    verts = np.ascontiguousarray(verts, dtype=np.float64)
    if cells.ndim != 2 or cells.shape[1] != 4 or verts.shape != (len(cells), 8, 3):
        raise FEError(-1, "cells must be (ncells, 4) and verts (ncells, 8, 3)")
    h = C.c_void_p()
    _check(L.fe_mesh_create_general(int(cx), int(cy), int(cz), C.c_void_p(cells.ctypes.data), len(cells),
                                    C.c_void_p(verts.ctypes.data), int(p), int(cuda_device), C.byref(h)))
    return h


def fe_num_all_nodes(h):
    return load_library().fe_num_all_nodes(h)


def fe_num_constraint_entries(h):
    return load_library().fe_num_constraint_entries(h)


def fe_get_constraints(h):
    """(row_ptr, col, val) of the hanging-node rows h = N..N_all-1."""
    nh = fe_num_all_nodes(h) - fe_num_nodes(h)
    nnz = fe_num_constraint_entries(h)
    rp, col, val = np.zeros(nh + 1, dtype=np.int64), np.zeros(nnz, dtype=np.int32), np.zeros(nnz, dtype=np.float64)
    _check(load_library().fe_get_constraints(h, C.c_void_p(rp.ctypes.data), C.c_void_p(col.ctypes.data),
                                             C.c_void_p(val.ctypes.data)))
    return rp, col, val


def fe_mesh_destroy(h):
    _check(load_library().fe_mesh_destroy(h))


def fe_num_nodes(h):
    return load_library().fe_num_nodes(h)


def fe_num_free(h):
    return load_library().fe_num_free(h)


def fe_num_cells(h):
    return load_library().fe_num_cells(h)


def fe_nodes_per_cell(h):
    return load_library().fe_nodes_per_cell(h)


def fe_quad_per_cell(h):
    return load_library().fe_quad_per_cell(h)


def fe_launch_count(h):
    return load_library().fe_launch_count(h)


def _fill(h, fn, shape, dtype):
    out = np.empty(shape, dtype=dtype)
    _check(getattr(load_library(), fn)(h, C.c_void_p(out.ctypes.data)))
    return out


def fe_get_l2g(h):
    return _fill(h, "fe_get_l2g", (fe_num_cells(h), fe_nodes_per_cell(h)), np.int32)


def fe_get_node_coords(h):
    return _fill(h, "fe_get_node_coords", (fe_num_all_nodes(h), 3), np.float64)


def fe_get_quad_coords(h):
    return _fill(h, "fe_get_quad_coords", (fe_num_cells(h) * fe_quad_per_cell(h), 3), np.float64)


def fe_get_mass(h):
    return _fill(h, "fe_get_mass", (fe_num_nodes(h),), np.float64)


def fe_get_dirichlet_mask(h):
    return _fill(h, "fe_get_dirichlet_mask", (fe_num_nodes(h),), np.uint8)


def fe_set_potential(h, Vq_dev, copy=1, stream=None):
    n = fe_num_cells(h) * fe_quad_per_cell(h)
    _check(load_library().fe_set_potential(h, _dev_ptr(Vq_dev, "Vq", n), int(copy), _stream(stream)))


def fe_apply_H(h, X, Y, eps=None, stream=None):
    if X.dim() != 2 or X.shape[0] != fe_num_nodes(h):
        raise FEError(-1, "X must be N x B")
    B = X.shape[1]
    ep = _dev_ptr(eps, "eps", B) if eps is not None else None
    _check(load_library().fe_apply_H(h, _dev_ptr(X, "X"), _dev_ptr(Y, "Y", X.numel()), B, ep, _stream(stream)))
    return Y


def fe_apply_H_chain(h, X, Y, Ynext=None, eps=None, y_is_clear=False, stream=None):
    if X.dim() != 2 or X.shape[0] != fe_num_nodes(h):
        raise FEError(-1, "X must be N x B")
    B = X.shape[1]
    ep = _dev_ptr(eps, "eps", B) if eps is not None else None
    yn = _dev_ptr(Ynext, "Ynext", X.numel()) if Ynext is not None else None
    _check(load_library().fe_apply_H_chain(h, _dev_ptr(X, "X"), _dev_ptr(Y, "Y", X.numel()), yn, B, ep,
                                           int(bool(y_is_clear)), _stream(stream)))
    return Y


def cheb_filter(h, X, m, a, b, a0, work, stream=None):
    if X.dim() != 2 or X.shape[0] != fe_num_nodes(h):
        raise FEError(-1, "X must be N x B")
    B = X.shape[1]
    _check(load_library().cheb_filter(h, _dev_ptr(X, "X"), B, int(m), float(a), float(b), float(a0),
                                      _dev_ptr(work, "work", 2 * X.numel()), _stream(stream)))
    return X


def cheb_filter_host(h, X_host, m, a, b, a0):
    """X_host: contiguous float64 CPU tensor or numpy array N x B (pinned memory overlaps best); filtered in place."""
    import numpy as np
    if isinstance(X_host, np.ndarray):
        if X_host.dtype != np.float64 or not X_host.flags["C_CONTIGUOUS"] or X_host.ndim != 2:
            raise FEError(-1, "X_host must be a C-contiguous float64 N x B array")
        ptr, shape = X_host.ctypes.data_as(C.c_void_p), X_host.shape
    else:
        import torch
        if X_host.is_cuda or X_host.dtype != torch.float64 or not X_host.is_contiguous() or X_host.dim() != 2:
            raise FEError(-1, "X_host must be a contiguous float64 CPU tensor N x B")
        ptr, shape = C.c_void_p(X_host.data_ptr()), tuple(X_host.shape)
    if shape[0] != fe_num_nodes(h):
        raise FEError(-1, "X_host must be N x B")
    _check(load_library().cheb_filter_host(h, ptr, int(shape[1]), int(m), float(a), float(b), float(a0)))
    return X_host


def fe_rayleigh_ritz(h, Y, work, stream=None):
    """Y (device, N x B) <- Ritz vectors in span(Y); returns the B Ritz values (numpy, ascending)."""
    import numpy as np
    if Y.dim() != 2 or Y.shape[0] != fe_num_nodes(h):
        raise FEError(-1, "Y must be N x B")
    B = Y.shape[1]
    theta = np.empty(B, dtype=np.float64)
    _check(load_library().fe_rayleigh_ritz(h, _dev_ptr(Y, "Y"), B, theta.ctypes.data_as(C.c_void_p),
                                           _dev_ptr(work, "work", Y.numel()), _stream(stream)))
    return theta


def fe_minres_shifted(h, G, X, eps, maxit, tol, precondition, work, stream=None):
    """Returns (relres (numpy, B), iterations)."""
    import numpy as np
    if G.dim() != 2 or G.shape[0] != fe_num_nodes(h):
        raise FEError(-1, "G must be N x B")
    B = G.shape[1]
    relres = np.empty(B, dtype=np.float64)
    iters = C.c_int(0)
    ep = _dev_ptr(eps, "eps", B) if eps is not None else None
    _check(load_library().fe_minres_shifted(h, _dev_ptr(G, "G"), _dev_ptr(X, "X", G.numel()), B, ep, int(maxit),
                                            float(tol), int(bool(precondition)), relres.ctypes.data_as(C.c_void_p),
                                            C.byref(iters), _dev_ptr(work, "work", 6 * G.numel()), _stream(stream)))
    return relres, iters.value


def fe_density(h, X, f, rho, stream=None):
    B = X.shape[1]
    n = fe_num_cells(h) * fe_quad_per_cell(h)
    _check(load_library().fe_density(h, _dev_ptr(X, "X"), B, _dev_ptr(f, "f", B), _dev_ptr(rho, "rho", n),
                                     _stream(stream)))
    return rho


def fe_lanczos_bounds(h, v0, k=20, stream=None):
    """(theta_min, theta_max, beta_k) after k Lanczos steps from the device vector v0 (N)."""
    import numpy as np
    import torch
    N = fe_num_nodes(h)
    out = np.empty(3, dtype=np.float64)
    work = torch.empty(3 * N, dtype=torch.float64, device=v0.device)
    _check(load_library().fe_lanczos_bounds(h, _dev_ptr(v0, "v0", N), int(k), out.ctypes.data_as(C.c_void_p),
                                            _dev_ptr(work, "work"), _stream(stream)))
    return float(out[0]), float(out[1]), float(out[2])


def fe_apply_potential(h, Uq, X, Y, stream=None):
    n = fe_num_cells(h) * fe_quad_per_cell(h)
    _check(load_library().fe_apply_potential(h, _dev_ptr(Uq, "Uq", n), _dev_ptr(X, "X"), _dev_ptr(Y, "Y", X.numel()),
                                             X.shape[1], _stream(stream)))
    return Y


def fe_gram(h, A, Bm, stream=None):
    """A^T Bm as a numpy B x B array."""
    import numpy as np
    B = A.shape[1]
    out = np.empty((B, B), dtype=np.float64)
    _check(load_library().fe_gram(h, _dev_ptr(A, "A"), _dev_ptr(Bm, "Bm", A.numel()), B,
                                  out.ctypes.data_as(C.c_void_p), _stream(stream)))
    return out


def fe_gram_static(h, A, Bm, stream=None):
    """A^T Bm as a numpy B x B array; the library allocates nothing in this call (static device accumulator, B <= 128)."""
    import numpy as np
    B = A.shape[1]
    out = np.empty((B, B), dtype=np.float64)
    _check(load_library().fe_gram_static(h, _dev_ptr(A, "A"), _dev_ptr(Bm, "Bm", A.numel()), B,
                                         out.ctypes.data_as(C.c_void_p), _stream(stream)))
    return out


def fe_add_subspace(h, Psi, D, P, stream=None):
    import numpy as np
    B = Psi.shape[1]
    Dh = np.ascontiguousarray(D, dtype=np.float64)
    if Dh.shape != (B, B):
        raise FEError(-1, "D must be B x B")
    _check(load_library().fe_add_subspace(h, _dev_ptr(Psi, "Psi"), Dh.ctypes.data_as(C.c_void_p),
                                          _dev_ptr(P, "P", Psi.numel()), B, _stream(stream)))
    return P


def fe_ritz_residuals(h, X, theta, work, stream=None):
    """|| H~ x_j - theta_j x_j ||_2 per column (numpy, B)."""
    B = X.shape[1]
    th = np.ascontiguousarray(theta, dtype=np.float64)
    if th.shape != (B,):
        raise FEError(-1, "theta must have B entries")
    res = np.empty(B, dtype=np.float64)
    _check(load_library().fe_ritz_residuals(h, _dev_ptr(X, "X"), th.ctypes.data_as(C.c_void_p), B,
                                            res.ctypes.data_as(C.c_void_p), _dev_ptr(work, "work", X.numel()),
                                            _stream(stream)))
    return res


def fe_chfsi(h, X, deg, a, b, a0, t_eig, n_gate, max_cycles, work, stream=None):
    """Returns (theta, residual norms, cycles); X holds the Ritz vectors."""
    B = X.shape[1]
    theta, res = np.empty(B, dtype=np.float64), np.empty(B, dtype=np.float64)
    cycles = C.c_int(0)
    _check(load_library().fe_chfsi(h, _dev_ptr(X, "X"), B, int(deg), float(a), float(b), float(a0), float(t_eig),
                                   int(n_gate), int(max_cycles), theta.ctypes.data_as(C.c_void_p),
                                   res.ctypes.data_as(C.c_void_p), C.byref(cycles),
                                   _dev_ptr(work, "work", 2 * X.numel()), _stream(stream)))
    return theta, res, cycles.value


def fe_diag_peak(kind, min_seconds=0.3, cuda_device=0):
    """Measured ceiling of the device: kind 0 DFMA / 1 DMMA in TFLOP/s, 2 stream / 3 bulk reduce-add / 4 red.add in GB/s."""
    out = C.c_double(0.0)
    _check(load_library().fe_diag_peak(int(cuda_device), int(kind), float(min_seconds), C.byref(out)))
    return out.value


def fe_set_variant(h, variant):
    _check(load_library().fe_set_variant(h, int(variant)))


# ---- convenience wrapper -----------------------------------------------------------------------------------------
class FEMesh:
    """Owns an fe_mesh handle.  All array arguments are torch CUDA float64 tensors; results stay on the device."""

    def __init__(self, xe, ye, ze, p, device=0, _handle=None):
        self.device = int(device)
        self.h = _handle if _handle is not None else fe_mesh_create(xe, ye, ze, p, self.device)
        self.p = int(p)
        self.N, self.N_free, self.ncells = fe_num_nodes(self.h), fe_num_free(self.h), fe_num_cells(self.h)
        self.nc, self.nq3 = fe_nodes_per_cell(self.h), fe_quad_per_cell(self.h)

    @classmethod
    def general(cls, mesh, p, device=0):
        """General hexahedral mesh with hanging nodes from a leaf description with attributes cx, cy, cz, cells, verts
        (fe_mesh_create_general); device=-1 builds the tables only."""
        h = fe_mesh_create_general(mesh.cx, mesh.cy, mesh.cz, mesh.cells, mesh.verts, p, device)
        return cls(None, None, None, p, device, _handle=h)

    @property
    def N_all(self):
        return fe_num_all_nodes(self.h)

    def constraints(self):
        return fe_get_constraints(self.h)

    def close(self):
        if getattr(self, "h", None):
            fe_mesh_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    l2g = lambda self: fe_get_l2g(self.h)  # noqa: E731
    node_coords = lambda self: fe_get_node_coords(self.h)  # noqa: E731
    quad_coords = lambda self: fe_get_quad_coords(self.h)  # noqa: E731
    mass = lambda self: fe_get_mass(self.h)  # noqa: E731
    mask = lambda self: fe_get_dirichlet_mask(self.h)  # noqa: E731

    def set_potential(self, Vq, stream=None):
        import torch
        if not isinstance(Vq, torch.Tensor):
            Vq = torch.as_tensor(np.ascontiguousarray(Vq, dtype=np.float64), device="cuda:%d" % self.device)
        fe_set_potential(self.h, Vq.reshape(-1), 1, stream)

    def apply_H(self, X, Y=None, eps=None, stream=None):
        import torch
        if Y is None:
            Y = torch.empty_like(X)
        return fe_apply_H(self.h, X, Y, eps, stream)

    def apply_H_chain(self, X, Y, Ynext=None, eps=None, y_is_clear=False, stream=None):
        return fe_apply_H_chain(self.h, X, Y, Ynext, eps, y_is_clear, stream)

    def cheb_filter(self, X, m, a, b, a0, work=None, stream=None):
        import torch
        if work is None:
            work = torch.empty(2 * X.numel(), dtype=torch.float64, device=X.device)
        return cheb_filter(self.h, X, m, a, b, a0, work, stream)

    def cheb_filter_host(self, X_host, m, a, b, a0):
        return cheb_filter_host(self.h, X_host, m, a, b, a0)

    def rayleigh_ritz(self, Y, work=None, stream=None):
        import torch
        if work is None:
            work = torch.empty(Y.numel(), dtype=torch.float64, device=Y.device)
        return fe_rayleigh_ritz(self.h, Y, work, stream)

    def minres_shifted(self, G, eps=None, maxit=200, tol=1e-10, precondition=True, stream=None):
        import torch
        X = torch.empty_like(G)
        work = torch.empty(6 * G.numel(), dtype=torch.float64, device=G.device)
        relres, iters = fe_minres_shifted(self.h, G, X, eps, maxit, tol, precondition, work, stream)
        return X, relres, iters

    def density(self, X, f, stream=None):
        import torch
        rho = torch.empty(self.ncells * self.nq3, dtype=torch.float64, device=X.device)
        return fe_density(self.h, X, f, rho, stream)

    def ritz_residuals(self, X, theta, work=None, stream=None):
        import torch
        if work is None:
            work = torch.empty(X.numel(), dtype=torch.float64, device=X.device)
        return fe_ritz_residuals(self.h, X, theta, work, stream)

    def chfsi(self, X, deg, a, b, a0, t_eig, n_gate, max_cycles=50, work=None, stream=None):
        import torch
        if work is None:
            work = torch.empty(2 * X.numel(), dtype=torch.float64, device=X.device)
        return fe_chfsi(self.h, X, deg, a, b, a0, t_eig, n_gate, max_cycles, work, stream)

    def lanczos_bounds(self, v0, k=20, stream=None):
        return fe_lanczos_bounds(self.h, v0, k, stream)

    def apply_potential(self, Uq, X, Y=None, stream=None):
        import torch
        if Y is None:
            Y = torch.empty_like(X)
        return fe_apply_potential(self.h, Uq, X, Y, stream)

    def gram(self, A, Bm, stream=None):
        return fe_gram(self.h, A, Bm, stream)

    def gram_static(self, A, Bm, stream=None):
        return fe_gram_static(self.h, A, Bm, stream)

    def add_subspace(self, Psi, D, P, stream=None):
        return fe_add_subspace(self.h, Psi, D, P, stream)

    def set_variant(self, v):
        fe_set_variant(self.h, v)

    @property
    def launches(self):
        return fe_launch_count(self.h)
