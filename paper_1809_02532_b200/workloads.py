"""Seeded synthetic inputs (meshes and states) for the two-fluid assembly path.

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It holds
none of the method's arithmetic (no gradients, fluxes, sources, Jacobians): it only
lays out triangles and samples the analytic initial fields of the paper's two
workloads at the cell centroids.

Recipes (BASELINE.json configs; PAPER.md L410-433 wave,
L551-559 GEM):

* wave  — circularly polarised wave on the periodic unit square
* gem   — GEM Harris-sheet reconnection set-up on [-12.8,12.8]x[-6.4,6.4]

State layout: AoS ``[ncells][18]`` float64, variable order
``Bx By Bz Ex Ey Ez Psi Phi rho_i rho_e ui(3) ue(3) T_i T_e``.
"""
from __future__ import annotations

import dataclasses
import numpy as np

NEQ = 18
# variable indices
IB, IE, IPSI, IPHI, IRHOI, IRHOE, IUI, IUE, ITI, ITE = 0, 3, 6, 7, 8, 9, 10, 13, 16, 17


@dataclasses.dataclass
class MeshInput:
    """What ``tfa_mesh_create`` / ``tfa_mesh_create_poly`` consume: nodes, counter-clockwise cells, per-cell corner
    coordinates.  Triangle meshes: ``cell_nodes [nc][3]``, ``cell_xy [nc][3][2]``, ``cell_ptr`` None.  Mixed
    triangle / quadrilateral meshes: ``cell_ptr [nc+1]`` and flat ``cell_nodes [cell_ptr[nc]]``,
    ``cell_xy [cell_ptr[nc]][2]``."""

    node_xy: np.ndarray      # [nn][2] f64 (periodic images identified: one entry per topological node)
    cell_nodes: np.ndarray   # i32, counter-clockwise
    cell_xy: np.ndarray      # f64, each cell's own (unwrapped) corner coordinates
    name: str = ""
    cell_ptr: np.ndarray | None = None

    @property
    def n_cells(self) -> int:
        return int(self.cell_nodes.shape[0]) if self.cell_ptr is None else int(self.cell_ptr.shape[0] - 1)

    @property
    def n_nodes(self) -> int:
        return int(self.node_xy.shape[0])

    def centroids(self) -> np.ndarray:
        """Where the initial states are sampled (S23): the area centroid of each cell (for a triangle, the mean
        of its corners)."""
        if self.cell_ptr is None:
            return self.cell_xy.mean(axis=1)
        cp = self.cell_ptr
        out = np.empty((self.n_cells, 2))
        for nv in np.unique(np.diff(cp)):
            idx = np.nonzero(np.diff(cp) == nv)[0]
            X = self.cell_xy[cp[idx][:, None] + np.arange(nv)[None, :]]      # [n][nv][2]
            if nv == 3:
                out[idx] = X.mean(axis=1)
                continue
            r = X - X[:, :1]
            a, b = r[:, 1:-1], r[:, 2:]
            cr = a[..., 0] * b[..., 1] - a[..., 1] * b[..., 0]               # twice the fan triangles' areas
            out[idx] = X[:, 0] + (cr[..., None] * (a + b)).sum(axis=1) / (3.0 * cr.sum(axis=1)[:, None])
        return out

    def permuted(self, perm_new_to_old: np.ndarray) -> "MeshInput":
        p = np.asarray(perm_new_to_old)
        if self.cell_ptr is None:
            return MeshInput(self.node_xy, np.ascontiguousarray(self.cell_nodes[p]),
                             np.ascontiguousarray(self.cell_xy[p]), self.name + "+perm")
        cnt = np.diff(self.cell_ptr)[p]
        cp = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
        src = np.repeat(self.cell_ptr[:-1][p], cnt) + (np.arange(cp[-1]) - np.repeat(cp[:-1], cnt))
        return MeshInput(self.node_xy, np.ascontiguousarray(self.cell_nodes[src]),
                         np.ascontiguousarray(self.cell_xy[src]), self.name + "+perm", cp)

    def rotated(self, theta: float, origin=(0.0, 0.0)) -> "MeshInput":
        c, s = np.cos(theta), np.sin(theta)
        R = np.array([[c, -s], [s, c]])
        o = np.asarray(origin, dtype=np.float64)
        return MeshInput(np.ascontiguousarray((self.node_xy - o) @ R.T + o),
                         self.cell_nodes.copy(),
                         np.ascontiguousarray((self.cell_xy - o) @ R.T + o), self.name + "+rot",
                         None if self.cell_ptr is None else self.cell_ptr.copy())


def quad_mesh(nx: int, ny: int, x0=0.0, x1=1.0, y0=0.0, y1=1.0, periodic_x=True, periodic_y=True,
              jitter: float = 0.0, seed: int = 0, tri_every: int = 0) -> MeshInput:
    """nx x ny quadrilaterals (the paper's Cartesian meshes, L433 "2N x N cells", L559 "512x512 elements").

    ``jitter`` moves every topological node by ``jitter*h*U(-1,1)`` per axis (hull nodes of a non-periodic
    direction stay on the hull), which makes the quadrilaterals general convex ones.  ``tri_every`` = k > 0 splits
    every cell with (i + j) % k == 0 by its (i,j)->(i+1,j+1) diagonal into two triangles: a mixed mesh.  Periodic
    directions identify nodes topologically; ``cell_xy`` keeps the unwrapped coordinates (S9).
    """
    nxn = nx if periodic_x else nx + 1
    nyn = ny if periodic_y else ny + 1
    hx, hy = (x1 - x0) / nx, (y1 - y0) / ny
    jj, ii = np.meshgrid(np.arange(nyn), np.arange(nxn), indexing="ij")
    shift = np.zeros((nyn, nxn, 2))
    if jitter > 0:
        rng = np.random.default_rng(seed)
        shift = rng.uniform(-1.0, 1.0, size=(nyn, nxn, 2)) * np.array([hx, hy]) * jitter
        if not periodic_x:
            shift[:, 0, 0] = shift[:, -1, 0] = 0.0
        if not periodic_y:
            shift[0, :, 1] = shift[-1, :, 1] = 0.0
    node_xy = (np.stack([x0 + ii * hx, y0 + jj * hy], axis=-1) + shift).reshape(-1, 2).astype(np.float64)
    j, i = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    i, j = i.reshape(-1), j.reshape(-1)

    def nid(a, b):
        return (b % nyn) * nxn + (a % nxn)

    def xy(a, b):    # unwrapped lattice position + the shift of the topological node
        return np.stack([x0 + a * hx, y0 + b * hy], axis=-1) + shift[b % nyn, a % nxn]

    corners = [(i, j), (i + 1, j), (i + 1, j + 1), (i, j + 1)]
    qn = np.stack([nid(a, b) for a, b in corners], axis=-1).astype(np.int32)     # [n][4]
    qx = np.stack([xy(a, b) for a, b in corners], axis=1)                         # [n][4][2]
    if tri_every <= 0:
        cp = (4 * np.arange(nx * ny + 1)).astype(np.int32)
        return MeshInput(node_xy, np.ascontiguousarray(qn.reshape(-1)), np.ascontiguousarray(qx.reshape(-1, 2)),
                         f"quad{nx}x{ny}", cp)
    split = (i + j) % tri_every == 0
    nodes, coords, counts = [], [], []
    for c in range(nx * ny):
        if split[c]:
            for tri in ((0, 1, 2), (0, 2, 3)):
                nodes.extend(qn[c, list(tri)]); coords.extend(qx[c, list(tri)]); counts.append(3)
        else:
            nodes.extend(qn[c]); coords.extend(qx[c]); counts.append(4)
    cp = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    return MeshInput(node_xy, np.asarray(nodes, dtype=np.int32), np.asarray(coords, dtype=np.float64),
                     f"mixed{nx}x{ny}", cp)


def split_quad_mesh(nx: int, ny: int, x0=0.0, x1=1.0, y0=0.0, y1=1.0,
                    periodic_x=True, periodic_y=True) -> MeshInput:
    """nx x ny quads, each split by the (i,j)->(i+1,j+1) diagonal into two CCW triangles.

    Periodic directions identify the node columns/rows topologically; ``cell_xy`` keeps the
    unwrapped coordinates so no minimum-image arithmetic is ever needed.
    Cell id = 2*(j*nx+i)+t, t=0 lower-right triangle, t=1 upper-left triangle.
    """
    nxn = nx if periodic_x else nx + 1
    nyn = ny if periodic_y else ny + 1
    hx, hy = (x1 - x0) / nx, (y1 - y0) / ny
    jj, ii = np.meshgrid(np.arange(nyn), np.arange(nxn), indexing="ij")
    node_xy = np.stack([x0 + ii * hx, y0 + jj * hy], axis=-1).reshape(-1, 2).astype(np.float64)

    j, i = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    i = i.reshape(-1)
    j = j.reshape(-1)

    def nid(a, b):
        return (b % nyn) * nxn + (a % nxn)

    n00, n10, n11, n01 = nid(i, j), nid(i + 1, j), nid(i + 1, j + 1), nid(i, j + 1)
    cells = np.empty((nx * ny, 2, 3), dtype=np.int32)
    cells[:, 0, :] = np.stack([n00, n10, n11], axis=-1)
    cells[:, 1, :] = np.stack([n00, n11, n01], axis=-1)

    def xy(a, b):
        return np.stack([x0 + a * hx, y0 + b * hy], axis=-1)

    c00, c10, c11, c01 = xy(i, j), xy(i + 1, j), xy(i + 1, j + 1), xy(i, j + 1)
    cxy = np.empty((nx * ny, 2, 3, 2), dtype=np.float64)
    cxy[:, 0] = np.stack([c00, c10, c11], axis=1)
    cxy[:, 1] = np.stack([c00, c11, c01], axis=1)
    return MeshInput(node_xy, cells.reshape(-1, 3), cxy.reshape(-1, 3, 2),
                     f"splitquad{nx}x{ny}")


def delaunay_mesh(npx: int, npy: int, x0: float, x1: float, y0: float, y1: float,
                  jitter: float, seed: int, shuffle_cells: bool = False) -> MeshInput:
    """Delaunay triangulation of an npx x npy lattice whose interior points are jittered.

    Interior points move by ``jitter*h*U(-1,1)`` per axis; the outer ring stays on the lattice so
    the hull has no slivers.  Gives exactly 2*(npx-1)*(npy-1) CCW triangles.  With
    ``shuffle_cells`` the cells are randomly permuted (same seed stream) — BASELINE config 4 run A.
    """
    from scipy.spatial import Delaunay  # library step of the *generator*, not of the method

    rng = np.random.default_rng(seed)
    hx, hy = (x1 - x0) / (npx - 1), (y1 - y0) / (npy - 1)
    jj, ii = np.meshgrid(np.arange(npy), np.arange(npx), indexing="ij")
    pts = np.stack([x0 + ii * hx, y0 + jj * hy], axis=-1).astype(np.float64)
    jit = rng.uniform(-1.0, 1.0, size=pts.shape) * np.array([hx, hy]) * jitter
    interior = np.zeros((npy, npx), dtype=bool)
    interior[1:-1, 1:-1] = True
    pts = pts + jit * interior[..., None]
    pts = pts.reshape(-1, 2)
    tri = Delaunay(pts).simplices.astype(np.int32)
    a, b, c = pts[tri[:, 0]], pts[tri[:, 1]], pts[tri[:, 2]]
    area2 = (b[:, 0] - a[:, 0]) * (c[:, 1] - a[:, 1]) - (b[:, 1] - a[:, 1]) * (c[:, 0] - a[:, 0])
    flip = area2 < 0
    tri[flip, 1], tri[flip, 2] = tri[flip, 2].copy(), tri[flip, 1].copy()
    # canonical cell order before the optional shuffle: by centroid lattice position (row-major)
    cen = pts[tri].mean(axis=1)
    order = np.lexsort((cen[:, 0], cen[:, 1]))
    tri = tri[order]
    if shuffle_cells:
        tri = tri[rng.permutation(tri.shape[0])]
    tri = np.ascontiguousarray(tri)
    return MeshInput(np.ascontiguousarray(pts), tri, np.ascontiguousarray(pts[tri]),
                     f"delaunay{npx}x{npy}s{seed}")


# ----------------------------------------------------------------------------------------------
# physical set-ups
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class Physics:
    gamma_gas: float = 5.0 / 3.0
    mass_ratio: float = 25.0
    c: float = 20.0
    gamma_psi: float = 1.0
    chi_phi: float = 1.0
    rusanov_alpha: float = 1.0


def fan_mesh(n: int, radius: float = 1.0, seed: int = 0, jitter: float = 0.2) -> MeshInput:
    """``n`` triangles around one hub node (a closed fan, all rim faces on the boundary): every cell meets every
    other cell at the hub, so each vertex-neighbour stencil has n - 1 entries -- the long-stencil case of step a2.
    Rim radii and angles are jittered so that the least-squares systems are generic."""
    if n < 3:
        raise ValueError("a closed fan needs at least 3 triangles")
    rng = np.random.default_rng(seed)
    ang = 2.0 * np.pi * (np.arange(n) + rng.uniform(-jitter, jitter, n)) / n
    rad = radius * (1.0 + rng.uniform(-jitter, jitter, n))
    node_xy = np.zeros((n + 1, 2))
    node_xy[1:, 0] = rad * np.cos(ang)
    node_xy[1:, 1] = rad * np.sin(ang)
    k = np.arange(n)
    cell_nodes = np.stack([np.zeros(n, dtype=np.int64), 1 + k, 1 + (k + 1) % n], axis=1).astype(np.int32)
    return MeshInput(node_xy, cell_nodes, np.ascontiguousarray(node_xy[cell_nodes]), f"fan{n}")


def wave_state(centroids: np.ndarray, seed: int | None, noise: float = 1e-3,
               mass_ratio: float = 25.0) -> np.ndarray:
    """Circularly polarised wave (BASELINE config 1-2; Eq. 16-17 for the shape)."""
    x = centroids[:, 0]
    n = centroids.shape[0]
    P = np.zeros((n, NEQ), dtype=np.float64)
    cs, sn = np.cos(2 * np.pi * x), np.sin(2 * np.pi * x)
    P[:, IB + 0] = 1.0
    P[:, IB + 1] = 0.1 * cs
    P[:, IB + 2] = 0.1 * sn
    for iu in (IUI, IUE):
        P[:, iu + 1] = -0.1 * cs
        P[:, iu + 2] = -0.1 * sn
    # E = -u x B with u = (0, uy, uz), B = (1, By, Bz)
    uy, uz = P[:, IUI + 1], P[:, IUI + 2]
    Bx, By, Bz = P[:, IB + 0], P[:, IB + 1], P[:, IB + 2]
    P[:, IE + 0] = -(uy * Bz - uz * By)
    P[:, IE + 1] = -(uz * Bx)
    P[:, IE + 2] = -(-uy * Bx)
    P[:, IRHOI] = 1.0
    P[:, IRHOE] = 1.0 / mass_ratio
    P[:, ITI] = 0.5   # p_i = rho_i * (1/m_i) * T_i = 0.5 with m_i = 1
    P[:, ITE] = 0.5   # p_e = rho_e * (1/m_e) * T_e = 0.5 with m_e = 1/mass_ratio
    if seed is not None and noise > 0:
        rng = np.random.default_rng(seed)
        P += rng.uniform(-noise, noise, size=P.shape)
    return P


def gem_state(centroids: np.ndarray, mass_ratio: float = 25.0, lam: float = 0.5,
              Lx: float = 25.6, Ly: float = 12.8, psi0: float = 0.1) -> np.ndarray:
    """GEM Harris sheet (BASELINE config 3-5; Birn et al. set-up)."""
    x, y = centroids[:, 0], centroids[:, 1]
    n = centroids.shape[0]
    P = np.zeros((n, NEQ), dtype=np.float64)
    sech2 = 1.0 / np.cosh(y / lam) ** 2
    dens = sech2 + 0.2
    kx, ky = 2 * np.pi / Lx, np.pi / Ly
    # psi = psi0 cos(kx x) cos(ky y); Bx = tanh(y/lam) - dpsi/dy ; By = dpsi/dx
    P[:, IB + 0] = np.tanh(y / lam) + psi0 * ky * np.cos(kx * x) * np.sin(ky * y)
    P[:, IB + 1] = -psi0 * kx * np.sin(kx * x) * np.cos(ky * y)
    P[:, IRHOI] = dens
    P[:, IRHOE] = dens / mass_ratio
    P[:, ITI] = 5.0 / 12.0
    P[:, ITE] = 1.0 / 12.0
    Jz = -sech2 / lam
    P[:, IUE + 2] = Jz / (-1.0 * dens)   # electrons carry the current: u_ez = J_z/(q_e n_e)
    return P


def gem_double_state(centroids: np.ndarray, mass_ratio: float = 25.0, lam: float = 0.5,
                     Lx: float = 25.6, Ly: float = 25.6, psi0: float = 0.1) -> np.ndarray:
    """Double current sheet on the periodic square [-Lx/2, Lx/2] x [-Ly/2, Ly/2] ("a square, where
    a double current sheet is simulated ... periodic boundary conditions in all sides"): two Harris sheets of
    opposite current at y = -+Ly/4, each the set-up of gem_state, each seeded with an X point at x = 0."""
    x, y = centroids[:, 0], centroids[:, 1]
    n = centroids.shape[0]
    P = np.zeros((n, NEQ), dtype=np.float64)
    ya, yb = (y + 0.25 * Ly) / lam, (y - 0.25 * Ly) / lam
    sa, sb = 1.0 / np.cosh(ya) ** 2, 1.0 / np.cosh(yb) ** 2
    dens = sa + sb + 0.2
    kx, ky = 2 * np.pi / Lx, 2 * np.pi / Ly
    # psi = psi0 cos(kx x) sin(ky y) (+-1 on the two sheets); Bx = Bx0 - dpsi/dy, By = dpsi/dx
    P[:, IB + 0] = np.tanh(ya) - np.tanh(yb) - 1.0 - psi0 * ky * np.cos(kx * x) * np.cos(ky * y)
    P[:, IB + 1] = -psi0 * kx * np.sin(kx * x) * np.sin(ky * y)
    P[:, IRHOI] = dens
    P[:, IRHOE] = dens / mass_ratio
    P[:, ITI] = 5.0 / 12.0
    P[:, ITE] = 1.0 / 12.0
    Jz = -(sa - sb) / lam
    P[:, IUE + 2] = Jz / (-1.0 * dens)
    return P


def perturb(state: np.ndarray, seed: int, amp: float) -> np.ndarray:
    """State perturbation between consecutive assemblies (BASELINE config 2)."""
    rng = np.random.default_rng(seed)
    return state + rng.uniform(-amp, amp, size=state.shape)


@dataclasses.dataclass
class Workload:
    name: str
    mesh: MeshInput
    state: np.ndarray
    physics: Physics
    dt: float
    n_calls: int
    reorder: str = "none"     # "none" | "rcm"
    seed: int = 0


GEM_DOMAIN = (-12.8, 12.8, -6.4, 6.4)


def make_workload(name: str, scale: float = 1.0) -> Workload:
    """BASELINE.json configs by name: c1 c2 c3 c4a (random order) c4b (RCM) c5; and the quadrilateral / mixed meshes
    of SURVEY 8(f)1: q1 (512x512 periodic quads, double current sheet), q2 (256x128 periodic quads, wave), qm
    (mixed triangles and jittered quadrilaterals, GEM).

    ``scale`` < 1 shrinks the lattice (linear factor) for tests that want the same recipe at a
    size the oracle finishes in seconds.
    """
    ph = Physics()
    if name == "c1":
        n = max(4, int(round(16 * scale)))
        m = split_quad_mesh(n, n)
        return Workload(name, m, wave_state(m.centroids(), seed=0), ph, 1e-3, 1, seed=0)
    if name == "c2":
        n = max(4, int(round(256 * scale)))
        m = split_quad_mesh(n, n)
        return Workload(name, m, wave_state(m.centroids(), seed=1), ph, 1e-3, 10, seed=1)
    if name == "c3":
        nx, ny = max(4, int(round(512 * scale))), max(4, int(round(256 * scale)))
        m = split_quad_mesh(nx, ny, *GEM_DOMAIN, periodic_x=True, periodic_y=False)
        return Workload(name, m, gem_state(m.centroids()), ph, 1e-3, 10)
    if name in ("c4a", "c4b", "c4m"):   # c4m: config 4's mesh in Z-order (not a BASELINE run; a third ordering)
        npx, npy = int(round(1000 * scale)) + 1, int(round(500 * scale)) + 1
        m = delaunay_mesh(npx, npy, *GEM_DOMAIN, jitter=0.3, seed=2, shuffle_cells=True)
        return Workload(name, m, gem_state(m.centroids()), ph, 1e-3, 10,
                        reorder={"c4a": "none", "c4b": "rcm", "c4m": "morton"}[name], seed=2)
    if name == "c5":
        npx, npy = int(round(2000 * scale)) + 1, int(round(1000 * scale)) + 1
        m = delaunay_mesh(npx, npy, *GEM_DOMAIN, jitter=0.3, seed=3, shuffle_cells=False)
        return Workload(name, m, gem_state(m.centroids()), ph, 1e-3, 3, reorder="rcm", seed=3)
    if name == "q1":   # the paper's second case on its own mesh (L559; Table 9): double current sheet, 512x512 quads
        n = max(6, int(round(512 * scale)))
        m = quad_mesh(n, n, -12.8, 12.8, -12.8, 12.8)
        return Workload(name, m, gem_double_state(m.centroids()), ph, 1e-3, 10)
    if name == "q2":   # the paper's first case on its own mesh (L433; Table 4): wave on 2N x N quads, N = 128
        n = max(4, int(round(128 * scale)))
        m = quad_mesh(2 * n, n, 0.0, 2.0, 0.0, 1.0)
        return Workload(name, m, wave_state(m.centroids(), seed=5), ph, 1e-3, 10, seed=5)
    if name == "qm":   # mixed mesh: jittered quads, every third one split into two triangles, boundaries in y
        nx, ny = max(6, int(round(768 * scale))), max(6, int(round(384 * scale)))
        m = quad_mesh(nx, ny, *GEM_DOMAIN, periodic_x=True, periodic_y=False, jitter=0.2, seed=6, tri_every=3)
        return Workload(name, m, gem_state(m.centroids()), ph, 1e-3, 10, reorder="rcm", seed=6)
    raise ValueError(f"unknown workload {name!r}")
