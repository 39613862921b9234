"""Seeded synthetic inputs for the five BASELINE.json workloads (readings R11-R13, R18, R19 in DESIGN.md).

This module serves BOTH the CUDA product's harness (bench.py, tests) and the CPU oracle's harness and holds
none of the method's arithmetic: it only defines mesh edges, atoms, potentials evaluated at coordinates the
caller supplies, random blocks and shifts.  Random numbers are counter based (splitmix64 -> uniform (0,1] ->
Box-Muller), so any element can be regenerated on its own; blocks are generated ONCE and the same array is
handed to both paths.

The workloads are stand-ins shaped like the paper's GPU benchmarks (p=6 meshes with 2.6 M
and 7.2 M basis functions, 40 / 100 electrons); no item of any external data set is reproduced.
"""
import math

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed, start, count):
    """Outputs start .. start+count-1 of the splitmix64 stream of `seed` (counter based, uint64)."""
    with np.errstate(over="ignore"):
        i = np.arange(start + 1, start + count + 1, dtype=np.uint64)
        z = np.uint64(seed) + i * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def uniform01(seed, start, count):
    """Uniform on (0, 1]: ((z >> 11) + 1) * 2^-53."""
    z = splitmix64(seed, start, count)
    return ((z >> np.uint64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)


def normal(seed, count, start=0):
    """N(0,1) numbers start..start+count-1: number 2k / 2k+1 = r cos(t) / r sin(t), r = sqrt(-2 ln u_{2k}),
    t = 2 pi u_{2k+1}."""
    k0, k1 = start // 2, (start + count + 1) // 2
    out = np.empty(2 * (k1 - k0))
    chunk = 1 << 22
    for k in range(k0, k1, chunk):
        kk = min(k1, k + chunk)
        u = uniform01(seed, 2 * k, 2 * (kk - k))
        r = np.sqrt(-2.0 * np.log(u[0::2]))
        t = (2.0 * math.pi) * u[1::2]
        out[2 * (k - k0):2 * (kk - k0):2] = r * np.cos(t)
        out[2 * (k - k0) + 1:2 * (kk - k0):2] = r * np.sin(t)
    return out[start - 2 * k0:start - 2 * k0 + count]


def random_block(seed, N, B, mask=None):
    """X (N x B, node-major, vector fastest), all rows N(0,1), then boundary rows zeroed (R13)."""
    X = normal(seed, N * B).reshape(N, B)
    if mask is not None:
        X[np.asarray(mask) == 0] = 0.0
    return X


def uniform_edges(lo, hi, cells):
    return lo + (hi - lo) * np.arange(cells + 1, dtype=np.float64) / cells


def graded_edges(half_width=15.0, cells_per_side=20, h0=0.2, ratio=1.15, hmax=1.5):
    """Reading R11: symmetric about 0, h_k = s*min(hmax, h0*ratio^k) outward, s scales the sum to half_width."""
    h = np.minimum(hmax, h0 * ratio ** np.arange(cells_per_side, dtype=np.float64))
    h *= half_width / h.sum()
    pos = np.concatenate([[0.0], np.cumsum(h)])
    pos[-1] = half_width
    return np.concatenate([-pos[:0:-1], pos])


def atoms(seed, count, zmax):
    """Reading R12: positions uniform in [-5,5]^3, Z uniform integer in {1..zmax}."""
    u = uniform01(seed, 0, 4 * count).reshape(count, 4)
    R = -5.0 + 10.0 * u[:, :3]
    Z = np.minimum(zmax, 1 + np.floor(u[:, 3] * zmax)).astype(np.float64)
    return R, Z


def harmonic(xyz):
    """V = 1/2 |r|^2 (config 1)."""
    return 0.5 * np.einsum("ij,ij->i", xyz, xyz)


def soft_coulomb(xyz, R, Z, soft2=0.25):
    """V(r) = -sum_a Z_a / sqrt(|r-R_a|^2 + 0.25) (configs 2-5)."""
    V = np.zeros(len(xyz))
    for Ra, Za in zip(np.atleast_2d(R), np.atleast_1d(Z)):
        d = xyz - Ra
        V -= Za / np.sqrt(np.einsum("ij,ij->i", d, d) + soft2)
    return V


def shifts(seed, B, lo=-2.0, hi=0.0):
    """eps sorted ascending, uniform in [lo, hi] (R18)."""
    return np.sort(lo + (hi - lo) * uniform01(seed, 0, B))


class Workload:
    """One BASELINE.json config: mesh edges, order, block width, filter degree, potential recipe, seeds."""

    def __init__(self, index, name, edges, p, B, m, potential, x_seed, atom_seed=None, n_atoms=0, zmax=0,
                 eps_seed=None, n_applies=1):
        self.index, self.name = index, name
        self.xe, self.ye, self.ze = edges
        self.p, self.B, self.m = p, B, m
        self.potential, self.x_seed = potential, x_seed
        self.atom_seed, self.n_atoms, self.zmax = atom_seed, n_atoms, zmax
        self.eps_seed, self.n_applies = eps_seed, n_applies

    @property
    def cells(self):
        return (len(self.xe) - 1, len(self.ye) - 1, len(self.ze) - 1)

    @property
    def nodes_per_axis(self):
        return tuple(c * self.p + 1 for c in self.cells)

    @property
    def N(self):
        nx, ny, nz = self.nodes_per_axis
        return nx * ny * nz

    @property
    def N_free(self):
        nx, ny, nz = self.nodes_per_axis
        return (nx - 2) * (ny - 2) * (nz - 2)

    @property
    def ncells(self):
        cx, cy, cz = self.cells
        return cx * cy * cz

    def atom_list(self):
        if self.potential == "single":
            return np.zeros((1, 3)), np.array([4.0])
        return atoms(self.atom_seed, self.n_atoms, self.zmax)

    def V(self, quad_xyz):
        """Potential at the quadrature points the caller supplies (cells*n_q^3 x 3)."""
        if self.potential == "harmonic":
            return harmonic(quad_xyz)
        R, Z = self.atom_list()
        return soft_coulomb(quad_xyz, R, Z)

    def X(self, mask=None, seed=None, B=None):
        return random_block(self.x_seed if seed is None else seed, self.N, self.B if B is None else B, mask)

    def eps(self):
        return shifts(self.eps_seed, self.B) if self.eps_seed is not None else None

    def describe(self):
        cx, cy, cz = self.cells
        return "cfg%d %s: %dx%dx%d cells p=%d N=%d B=%d m=%d" % (self.index, self.name, cx, cy, cz, self.p,
                                                                   self.N, self.B, self.m)


def config(i):
    """BASELINE.json configs 1..5."""
    if i == 1:
        e = uniform_edges(-6.0, 6.0, 4)
        return Workload(1, "tiny-harmonic", (e, e, e), 2, 8, 10, "harmonic", x_seed=0)
    if i == 2:
        e = uniform_edges(-10.0, 10.0, 16)
        return Workload(2, "single-atom-well", (e, e, e), 4, 64, 20, "single", x_seed=1)
    if i == 3:
        e = uniform_edges(-12.0, 12.0, 24)
        return Workload(3, "small-molecule", (e, e, e), 6, 64, 30, "atoms", x_seed=2, atom_seed=1003, n_atoms=10,
                        zmax=8)
    if i == 4:
        e = graded_edges()
        return Workload(4, "graded-100e-molecule", (e, e, e), 6, 128, 40, "atoms", x_seed=3, atom_seed=1004,
                        n_atoms=20, zmax=9)
    if i == 5:
        e = uniform_edges(-10.0, 10.0, 16)
        return Workload(5, "adjoint-shifted-apply", (e, e, e), 4, 64, 0, "single", x_seed=4, eps_seed=2005,
                        n_applies=200)
    raise ValueError("config index 1..5")


def reduced(i, cells):
    """Same recipe as config i (order, cell size, potential) on a centred sub-box of cells^3 cells: the bounded
    sample the CPU baseline times, and the small parity meshes of the tests."""
    w = config(i)

    def centre(e):
        c = len(e) - 1
        k = min(cells, c)
        lo = (c - k) // 2
        return np.array(e[lo:lo + k + 1])

    w.xe, w.ye, w.ze = centre(w.xe), centre(w.ye), centre(w.ze)
    w.name += "-sub%d" % cells
    return w


# ---- general hexahedral meshes with hanging nodes (Fig. 6) -----------------------
class OctreeMesh:
    """Description of an adaptively refined hexahedral mesh, the INPUT both the library and the oracle build from (no
    method arithmetic here: only which cells exist and where their corners are).

    cells : (ncells, 4) int32 rows (level, ix, iy, iz): the leaf with index (ix, iy, iz) on the level-`level` lattice of
            2^level (cx, cy, cz) cells.  Leaves are listed root by root (root e = ex + cx (ey + cy ez)), the children of a
            refined cell depth first in the order child = hx + 2 (hy + 2 hz).  Levels of leaves whose closures touch
            differ by at most one (2:1 balance over faces, edges and corners).
    verts : (ncells, 8, 3) float64 corner coordinates, corner v = vx + 2 (vy + 2 vz); the cell is the trilinear image of
            the reference cube.  Corners shared by cells coincide, and a corner that hangs on a coarser neighbour's edge or
            face lies on that neighbour's (bi)linear edge / face."""

    def __init__(self, cx, cy, cz, cells, verts, maxlevel):
        self.cx, self.cy, self.cz = int(cx), int(cy), int(cz)
        self.cells = np.ascontiguousarray(cells, dtype=np.int32)
        self.verts = np.ascontiguousarray(verts, dtype=np.float64)
        self.maxlevel = int(maxlevel)

    @property
    def ncells(self):
        return len(self.cells)


def octree_mesh(xe, ye, ze, refine, maxlevel, deform=None):
    """Refine the tensor-product root grid (edges xe, ye, ze): a leaf of level < maxlevel is split into 8 when
    refine(level, lo, hi) is true (lo, hi = corners of its undeformed box), then cells are split further until the 2:1
    balance holds.  deform(xyz) -> xyz moves the lattice points (identity if None); points that hang on a coarser cell are
    then put back onto that cell's trilinear image, coarse levels first, so that the mesh has no cracks."""
    xe, ye, ze = (np.asarray(e, dtype=np.float64) for e in (xe, ye, ze))
    cx, cy, cz = len(xe) - 1, len(ye) - 1, len(ze) - 1
    L = int(maxlevel)

    def box(level, ix, iy, iz):
        def ax(e, i):
            r, k = divmod(i, 1 << level)
            return e[r] + (e[r + 1] - e[r]) * k / (1 << level) if r < len(e) - 1 else e[-1]
        lo = np.array([ax(xe, ix), ax(ye, iy), ax(ze, iz)])
        hi = np.array([ax(xe, ix + 1), ax(ye, iy + 1), ax(ze, iz + 1)])
        return lo, hi

    leaves = {(0, ix, iy, iz) for iz in range(cz) for iy in range(cy) for ix in range(cx)}

    def split(c):
        l, ix, iy, iz = c
        leaves.discard(c)
        for hz in range(2):
            for hy in range(2):
                for hx in range(2):
                    leaves.add((l + 1, 2 * ix + hx, 2 * iy + hy, 2 * iz + hz))

    for level in range(L):
        for c in sorted(leaves):
            if c[0] == level and refine(level, *box(*c)):
                split(c)

    def containing_leaf(l, ix, iy, iz):
        while l >= 0:
            if (l, ix, iy, iz) in leaves:
                return (l, ix, iy, iz)
            l, ix, iy, iz = l - 1, ix >> 1, iy >> 1, iz >> 1
        return None

    changed = True
    while changed:  # 2:1 balance over the 26-neighbourhood
        changed = False
        for c in sorted(leaves, key=lambda t: -t[0]):
            l, ix, iy, iz = c
            if c not in leaves or l < 2:
                continue
            for dz in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dx in (-1, 0, 1):
                        jx, jy, jz = ix + dx, iy + dy, iz + dz
                        if not (0 <= jx < cx << l and 0 <= jy < cy << l and 0 <= jz < cz << l):
                            continue
                        nb = containing_leaf(l, jx, jy, jz)
                        if nb is not None and nb[0] < l - 1:
                            split(nb)
                            changed = True

    def order_key(c):  # root by root, children depth first
        l, ix, iy, iz = c
        rx, ry, rz = ix >> l, iy >> l, iz >> l
        path = []
        for k in range(l - 1, -1, -1):
            path.append(((ix >> k) & 1) + 2 * (((iy >> k) & 1) + 2 * ((iz >> k) & 1)))
        return (rx + cx * (ry + cy * rz), path)

    cells = sorted(leaves, key=order_key)
    # lattice points of the finest level, deformed, then hanging points put back onto the coarser cell's trilinear image
    Vx, Vy, Vz = (cx << L) + 1, (cy << L) + 1, (cz << L) + 1

    def axis_pts(e, c):
        out = np.empty((c << L) + 1)
        for r in range(c):
            out[r << L:((r + 1) << L) + 1] = e[r] + (e[r + 1] - e[r]) * np.arange((1 << L) + 1) / (1 << L)
        out[-1] = e[-1]
        return out

    X, Y, Z = np.meshgrid(axis_pts(xe, cx), axis_pts(ye, cy), axis_pts(ze, cz), indexing="ij")
    P = np.stack([X, Y, Z], axis=-1)  # [vx, vy, vz, 3]
    if deform is not None:
        P = np.asarray(deform(P.reshape(-1, 3)), dtype=np.float64).reshape(Vx, Vy, Vz, 3)
    for level in range(L):  # coarse first; cells of the finest level have no interior lattice points
        s = 1 << (L - level)
        t = np.arange(s + 1) / s
        for (l, ix, iy, iz) in cells:
            if l != level:
                continue
            x0, y0, z0 = ix * s, iy * s, iz * s
            C = P[x0:x0 + s + 1:s, y0:y0 + s + 1:s, z0:z0 + s + 1:s].copy()  # [2,2,2,3] corners
            wx = np.stack([1 - t, t])  # [2, s+1]
            P[x0:x0 + s + 1, y0:y0 + s + 1, z0:z0 + s + 1] = np.einsum("ai,bj,ck,abcd->ijkd", wx, wx, wx, C)
    verts = np.empty((len(cells), 8, 3))
    for e, (l, ix, iy, iz) in enumerate(cells):
        s = 1 << (L - l)
        for v in range(8):
            verts[e, v] = P[(ix + (v & 1)) * s, (iy + ((v >> 1) & 1)) * s, (iz + (v >> 2)) * s]
    return OctreeMesh(cx, cy, cz, np.array(cells, dtype=np.int32).reshape(-1, 4), verts, L)


def adaptive_molecule(roots=12, half=12.0, levels=2, radii=(3.0, 1.5), atom_seed=1003, n_atoms=10, zmax=8):
    """NEXT-3 workload: the atoms of config 3 on an adaptively refined mesh -- a roots^3 root grid on [-half, half]^3,
    refined `levels` times where a cell centre is within radii[level] of an atom (cell size half/roots*2 -> /4 near the
    nuclei), the shape of the paper's meshes (l.273, Fig. 6).  Returns (OctreeMesh, V) with V(quad_xyz) the soft-Coulomb
    wells of R12."""
    e = uniform_edges(-half, half, roots)
    R, Z = atoms(atom_seed, n_atoms, zmax)

    def refine(level, lo, hi):
        c = 0.5 * (lo + hi)
        return bool((np.linalg.norm(R - c, axis=1) < radii[level]).any())

    mesh = octree_mesh(e, e, e, refine, levels)
    return mesh, (lambda q: soft_coulomb(q, R, Z))
