"""ORACLE (TEST INFRASTRUCTURE) for general hexahedral meshes with hanging nodes (PAPER.md l.151,
l.273, Fig. 6: the adaptively refined meshes every result of the paper runs on).

Plain definition, step by step, on top of oracle/fe_oracle.c:
  1. every leaf cell is the trilinear image of [-1,1]^3 (its 8 corners come with the mesh description, workloads.OctreeMesh);
  2. nodes are identified GEOMETRICALLY: two local nodes are the same global node when they sit at the same point of the
     root lattice (logical coordinates, compared after rounding) and belong to cells of the same level;
  3. a node of a cell that lies on the closure of a COARSER leaf hangs: its value is the coarse cell's polynomial at that
     point, u_h = sum_k c_k u_k with c_k the coarse cell's Lagrange basis (Eq. 12) evaluated there; chains (a master that
     hangs itself) are substituted until only unconstrained nodes remain;
  4. cell matrices by explicit quadrature with the Jacobian at every Gauss point (orc_general_cell_matrix, Eq. 17);
  5. H_all = sum_e P_e^T H_e P_e over ALL nodes, H_c = C^T H_all C with C = [I; C_hanging] (the constrained problem lives on
     the unconstrained nodes), lumped mass M_c = diag(C^T m_all) with m_all the GLL-quadrature nodal masses (l.185; row sum
     of C^T M C because the rows of C sum to one) -- readings R23-R25 of DESIGN.md;
  6. H~ = S H_c S, S = mask / sqrt(M_c) (Eq. 19), apply and filter exactly as on the tensor-product meshes.
Numbering rule (R23): cells in the order of the description, local nodes a = ax + n (ay + n az); unconstrained nodes get
ids 0..N-1 in order of first appearance, hanging nodes N..N_all-1 in order of first appearance.
scipy.sparse serves as the sparse-matrix primitive (products and sums of explicitly listed entries).
"""
import ctypes as C

import numpy as np
import scipy.sparse as sp

from . import fe_oracle as fo


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class GeneralOracleMesh:
    def __init__(self, mesh, p):
        L = fo._load()
        L.orc_general_cell_matrix.restype = None
        L.orc_general_cell_matrix.argtypes = [C.c_int] + [C.POINTER(C.c_double)] * 2 + [C.c_double] * 2 + [C.POINTER(C.c_double)]
        L.orc_general_map.restype = None
        L.orc_general_map.argtypes = [C.POINTER(C.c_double)] * 2 + [C.c_int] + [C.POINTER(C.c_double)] * 2
        self._L = L
        self.p, self.n = int(p), int(p) + 1
        self.nc = self.nq3 = self.n ** 3
        self.cells = np.asarray(mesh.cells, dtype=np.int64)
        self.verts = np.ascontiguousarray(mesh.verts, dtype=np.float64)
        self.root = (mesh.cx, mesh.cy, mesh.cz)
        self.ncells = len(self.cells)
        self.gll_x, self.gll_w = fo.gll(self.p)
        self.gl_x, self.gl_w = fo.gauss(self.n)
        self._number_nodes()
        self.He = None
        self.Ht = None

    # ---- steps 2 and 3: node identification, hanging nodes, constraint rows -----------------------------------------------
    def _logical(self, e):
        """Logical coordinates (root-lattice units) of the n^3 nodes of cell e, local order a = ax + n (ay + n az)."""
        l, ix, iy, iz = self.cells[e]
        h = 1.0 / (1 << l)
        t = 0.5 * (self.gll_x + 1.0)
        t[-1] = 1.0
        ax = (np.array([ix, iy, iz])[:, None] + t[None, :]) * h  # [axis, local index]
        U = np.empty((self.n, self.n, self.n, 3))
        U[..., 0] = ax[0][None, None, :]
        U[..., 1] = ax[1][None, :, None]
        U[..., 2] = ax[2][:, None, None]
        return U.reshape(-1, 3)

    def _number_nodes(self):
        n, nc = self.n, self.nc
        lev = self.cells[:, 0]
        lo = self.cells[:, 1:4] / (1 << lev)[:, None].astype(np.float64)
        hi = (self.cells[:, 1:4] + 1) / (1 << lev)[:, None].astype(np.float64)
        key_of = {}
        slots = []   # per distinct node: (level, logical xyz, coarse cell it hangs on or -1)
        l2slot = np.empty((self.ncells, nc), dtype=np.int64)
        for e in range(self.ncells):
            U = self._logical(e)
            l = int(lev[e])
            coarser = np.flatnonzero(lev < l)
            if len(coarser):  # only coarser leaves whose closed box meets this cell's can contain one of its nodes
                coarser = coarser[np.all((hi[coarser] >= lo[e] - 1e-12) & (lo[coarser] <= hi[e] + 1e-12), axis=1)]
            keys = np.round(U * 2.0 ** 32).astype(np.int64).tolist()  # rounded logical coordinates of the cell's nodes
            for a in range(nc):
                u = U[a]
                key = (l, keys[a][0], keys[a][1], keys[a][2])
                s = key_of.get(key)
                if s is None:
                    parent = -1
                    if len(coarser):
                        inside = np.all((u >= lo[coarser] - 1e-12) & (u <= hi[coarser] + 1e-12), axis=1)
                        if inside.any():
                            parent = int(coarser[np.flatnonzero(inside)[0]])
                    s = len(slots)
                    key_of[key] = s
                    slots.append((l, u.copy(), parent))
                l2slot[e, a] = s
        is_hang = np.array([s[2] >= 0 for s in slots])
        ids = np.empty(len(slots), dtype=np.int64)
        self.N = int((~is_hang).sum())
        self.N_all = len(slots)
        ids[~is_hang] = np.arange(self.N)
        ids[is_hang] = self.N + np.arange(self.N_all - self.N)
        self._l2g = ids[l2slot].astype(np.int32)
        self._logical_of_id = np.empty((self.N_all, 3))
        self._logical_of_id[ids] = np.array([s[1] for s in slots])
        # constraint rows: hanging id -> {id: weight} with the coarse cell's 3-D Lagrange basis at the node's position
        rows = {}
        for s, (l, u, parent) in enumerate(slots):
            if parent < 0:
                continue
            pl, px, py, pz = self.cells[parent]
            xi = 2.0 * (u * (1 << pl) - np.array([px, py, pz])) - 1.0
            xi = np.clip(xi, -1.0, 1.0)
            w1 = [[fo.lagrange(self.gll_x, b, xi[d]) for b in range(n)] for d in range(3)]
            row = {}
            for bz in range(n):
                for by in range(n):
                    for bx in range(n):
                        w = w1[0][bx] * w1[1][by] * w1[2][bz]
                        if abs(w) > 1e-14:
                            g = int(self._l2g[parent, bx + n * (by + n * bz)])
                            row[g] = row.get(g, 0.0) + w
            rows[int(ids[s])] = row
        changed = True
        while changed:  # substitute masters that hang themselves (multi-level interfaces)
            changed = False
            for h, row in rows.items():
                for g in [g for g in row if g >= self.N]:
                    w = row.pop(g)
                    for g2, w2 in rows[g].items():
                        row[g2] = row.get(g2, 0.0) + w * w2
                    changed = True
        self.constraints = rows
        r, c, v = [], [], []
        for h, row in rows.items():
            for g, w in row.items():
                r.append(h), c.append(g), v.append(w)
        eye = sp.identity(self.N, format="csr")
        Ch = sp.csr_matrix((v, (np.array(r, dtype=np.int64) - self.N, c)), shape=(self.N_all - self.N, self.N))
        self.Cfull = sp.vstack([eye, Ch]).tocsr()  # N_all x N
        cx, cy, cz = self.root
        U = self._logical_of_id[:self.N]
        bnd = ((np.abs(U[:, 0]) < 1e-12) | (np.abs(U[:, 0] - cx) < 1e-12) | (np.abs(U[:, 1]) < 1e-12)
               | (np.abs(U[:, 1] - cy) < 1e-12) | (np.abs(U[:, 2]) < 1e-12) | (np.abs(U[:, 2] - cz) < 1e-12))
        self._mask = (~bnd).astype(np.uint8)
        self.N_free = int(self._mask.sum())
        # lumped GLL masses of all nodes and physical coordinates, cell by cell
        xi = np.array([[self.gll_x[ax], self.gll_x[ay], self.gll_x[az]] for az in range(n) for ay in range(n) for ax in range(n)])
        wg = np.array([self.gll_w[ax] * self.gll_w[ay] * self.gll_w[az] for az in range(n) for ay in range(n) for ax in range(n)])
        m_all = np.zeros(self.N_all)
        xyz = np.zeros((self.N_all, 3))
        pos, det = np.empty((nc, 3)), np.empty(nc)
        for e in range(self.ncells):
            self._L.orc_general_map(_d(self.verts[e]), _d(xi), nc, _d(pos), _d(det))
            np.add.at(m_all, self._l2g[e], wg * det)
            xyz[self._l2g[e]] = pos
        self._m_all = m_all
        self._xyz = xyz
        self._mass = self.Cfull.T @ m_all

    # ---- tables -------------------------------------------------------------------------------------------------------------
    def l2g(self):
        return self._l2g.copy()

    def constraint_matrix(self):
        """Dense (N_all - N) x N matrix of the hanging rows."""
        return self.Cfull[self.N:].toarray()

    def node_coords(self):
        return self._xyz.copy()

    def quad_coords(self):
        n = self.n
        xi = np.array([[self.gl_x[qx], self.gl_x[qy], self.gl_x[qz]] for qz in range(n) for qy in range(n) for qx in range(n)])
        out = np.empty((self.ncells, self.nq3, 3))
        det = np.empty(self.nq3)
        for e in range(self.ncells):
            self._L.orc_general_map(_d(self.verts[e]), _d(xi), self.nq3, _d(out[e]), _d(det))
        return out.reshape(-1, 3)

    def mass(self):
        return self._mass.copy()

    def mask(self):
        return self._mask.copy()

    # ---- operator -------------------------------------------------------------------------------------------------------------
    def cell_matrix(self, e, Vq_cell=None, kin=0.5, pot=1.0):
        He = np.empty((self.nc, self.nc))
        v = np.ascontiguousarray(Vq_cell, dtype=np.float64) if Vq_cell is not None else None
        self._L.orc_general_cell_matrix(self.p, _d(self.verts[e]), _d(v) if v is not None else None, float(kin), float(pot), _d(He))
        return He

    def set_potential(self, Vq, kin=0.5):
        Vq = np.ascontiguousarray(Vq, dtype=np.float64).reshape(self.ncells, self.nq3)
        r, c, v = [], [], []
        for e in range(self.ncells):
            He = self.cell_matrix(e, Vq[e], kin=kin)
            g = self._l2g[e].astype(np.int64)
            r.append(np.repeat(g, self.nc)), c.append(np.tile(g, self.nc)), v.append(He.reshape(-1))
        H_all = sp.csr_matrix((np.concatenate(v), (np.concatenate(r), np.concatenate(c))), shape=(self.N_all, self.N_all))
        self.H_all = H_all
        self.Hc = (self.Cfull.T @ H_all @ self.Cfull).tocsr()
        s = np.zeros(self.N)
        free = self._mask.astype(bool)
        s[free] = 1.0 / np.sqrt(self._mass[free])
        S = sp.diags(s)
        self.Ht = (S @ self.Hc @ S).tocsr()

    def density(self, X, f):
        """rho[e, q] = sum_j f_j psi_j(x_q)^2 at the Gauss points of every cell (Eq. 4, l.73-77), psi = M_c^{-1/2} psi~
        on the unconstrained nodes (zero Dirichlet rows), hanging values through the constraints, psi_j(x_q) written out
        with the Lagrange basis of Eq. 12."""
        X = np.ascontiguousarray(X, dtype=np.float64)
        n = self.n
        L1 = np.array([[fo.lagrange(self.gll_x, a, self.gl_x[q]) for a in range(n)] for q in range(n)])  # L1[q, a]
        free = self._mask.astype(bool)
        s = np.zeros(self.N)
        s[free] = 1.0 / np.sqrt(self._mass[free])
        psi_all = self.Cfull @ (X * s[:, None])
        fw = np.ascontiguousarray(f, dtype=np.float64)
        rho = np.zeros((self.ncells, n ** 3))
        for e in range(self.ncells):
            loc = psi_all[self._l2g[e]].reshape(n, n, n, -1)  # [az, ay, ax, j]
            val = np.einsum("ra,sb,tc,cbaj->rstj", L1, L1, L1, loc)  # [qx, qy, qz, j]
            rho[e] = np.einsum("rstj,j->rst", val ** 2, fw).transpose(2, 1, 0).reshape(-1)  # q = qx + n (qy + n qz)
        return rho

    def potential_apply(self, Uq, X):
        """M_c^{-1/2} C^T M_U C M_c^{-1/2} X with (M_U)_ab = int N_a U N_b entry by entry from the cell matrices with the
        kinetic part switched off: the integral of the adjoint right-hand side (Eq. 18, l.174-177) on a constrained mesh."""
        Uq = np.ascontiguousarray(Uq, dtype=np.float64).reshape(self.ncells, self.nq3)
        X = np.ascontiguousarray(X, dtype=np.float64)
        free = self._mask.astype(bool)
        s = np.zeros(self.N)
        s[free] = 1.0 / np.sqrt(self._mass[free])
        x_all = self.Cfull @ (X * s[:, None])
        y_all = np.zeros_like(x_all)
        for e in range(self.ncells):
            g = self._l2g[e]
            y_all[g] += self.cell_matrix(e, Uq[e], kin=0.0, pot=1.0) @ x_all[g]
        return (self.Cfull.T @ y_all) * s[:, None]

    def laplacian_precond(self):
        """MINRES preconditioner on a constrained mesh (reading R27): M_c,ii / d_i on free rows, 0 on Dirichlet
        rows, with d_i = kd_i + sum_h C_hi^2 kd_h and kd the diagonal of the assembled kinetic matrix 1/2 K over ALL nodes,
        taken entry by entry from the cell matrices with the potential switched off."""
        kd = np.zeros(self.N_all)
        for e in range(self.ncells):
            np.add.at(kd, self._l2g[e], np.diag(self.cell_matrix(e, None, kin=0.5, pot=0.0)))
        Ch = self.Cfull[self.N:]
        d = kd[:self.N] + (Ch.multiply(Ch)).T @ kd[self.N:]
        free = self._mask.astype(bool)
        out = np.zeros(self.N)
        out[free] = self._mass[free] / d[free]
        return out

    def apply(self, X, eps=None, nthreads=1):
        X = np.ascontiguousarray(X, dtype=np.float64)
        free = self._mask.astype(bool)
        Xm = X * free[:, None]
        Y = self.Ht @ Xm
        if eps is not None:
            Y = Y - Xm * np.asarray(eps, dtype=np.float64)[None, :]
        Y[~free] = 0.0
        return Y

    def apply_rows(self, X, rows, Vq, eps=None):
        """Selected rows of H~ X - X diag(eps) straight from the definition, without assembling anything (meshes whose cell
        matrices are out of reach): row i of C^T H_all C collects, for node i and every hanging node that depends on it
        (weight C_hi), the rows of the cell matrices of the cells that contain that node, applied to x_all = C (s . X).
        Cell matrices are computed on demand by explicit quadrature and cached."""
        X = np.ascontiguousarray(X, dtype=np.float64)
        Vq = np.ascontiguousarray(Vq, dtype=np.float64).reshape(self.ncells, self.nq3)
        free = self._mask.astype(bool)
        s = np.zeros(self.N)
        s[free] = 1.0 / np.sqrt(self._mass[free])
        x_all = self.Cfull @ (X * s[:, None])
        Ccsc = self.Cfull.tocsc()
        flat = self._l2g.reshape(-1).astype(np.int64)
        order = np.argsort(flat, kind="stable")
        starts = np.searchsorted(flat[order], np.arange(self.N_all + 1))
        cache = {}
        out = np.zeros((len(rows), X.shape[1]))
        for r, i in enumerate(rows):
            if not free[i]:
                continue
            acc = np.zeros(X.shape[1])
            for a, w in zip(Ccsc.indices[Ccsc.indptr[i]:Ccsc.indptr[i + 1]], Ccsc.data[Ccsc.indptr[i]:Ccsc.indptr[i + 1]]):
                for pos in order[starts[a]:starts[a + 1]]:
                    e, la = divmod(int(pos), self.nc)
                    if e not in cache:
                        cache[e] = self.cell_matrix(e, Vq[e])
                    acc += w * (cache[e][la] @ x_all[self._l2g[e]])
            out[r] = s[i] * acc
            if eps is not None:
                out[r] -= np.asarray(eps, dtype=np.float64) * X[i]
        return out

    def filter(self, X, m, a, b, a0, nthreads=1):
        """Scaled three-term recurrence of reading R7 (l.208-210), serial."""
        if not (a0 < a < b) or m < 1:
            raise ValueError("need a0 < a < b and m >= 1")
        free = self._mask.astype(bool)
        e, c = (b - a) / 2.0, (b + a) / 2.0
        s1 = e / (a0 - c)
        s = s1
        Ykm = np.ascontiguousarray(X, dtype=np.float64) * free[:, None]
        Yk = (s1 / e) * (self.apply(Ykm) - c * Ykm)
        for _ in range(1, m):
            sn = 1.0 / (2.0 / s1 - s)
            Yk, Ykm = (2.0 * sn / e) * (self.apply(Yk) - c * Yk) - s * sn * Ykm, Yk
            s = sn
        return Yk
