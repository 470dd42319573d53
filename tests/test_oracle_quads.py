"""Pins for the oracle on quadrilateral and mixed meshes and for its boundary rules.

The paper's own meshes are Cartesian quadrilaterals ("2N x N cells", L559 "512x512 elements in a
Cartesian grid") and its boundary conditions are a separate loop over the boundary faces (L260).  Each check
compares the oracle with something fixed by the paper or by mathematics and computed here by another route:
hand-worked connectivity (tests/golden/quad_2x2.txt), set arithmetic, Green's-theorem moments, numpy least
squares, central differences, the paper's exact wave solution (Eq. 15-18).
"""
import numpy as np
import pytest

from conftest import random_state
from helpers import (read_golden_sections, check_connectivity_against_brute, rcm_reference, bsr_to_dense,
                     cells_as_lists)
from test_exact_wave import exact_wave, check_convergence

RNG = np.random.default_rng(4321)


def meshes(W):
    return {
        "quads_periodic": W.quad_mesh(6, 5),
        "quads_channel": W.quad_mesh(7, 4, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False, jitter=0.25, seed=2),
        "quads_box": W.quad_mesh(6, 5, 0.0, 3.0, 0.0, 2.0, periodic_x=False, periodic_y=False, jitter=0.3, seed=3),
        "mixed_box": W.quad_mesh(7, 5, 0.0, 3.5, 0.0, 2.5, periodic_x=False, periodic_y=False, jitter=0.2, seed=4,
                                 tri_every=3),
        "mixed_periodic": W.quad_mesh(6, 6, jitter=0.15, seed=5, tri_every=2),
    }


def _sizes(m):
    return (m.n_cells, m.n_faces, m.nnzb, m.n_stencil)


# ------------------------------------------------------------------------------------------
# connectivity
# ------------------------------------------------------------------------------------------
def test_golden_quad_2x2(orc, W):
    g = read_golden_sections("quad_2x2.txt")
    mi = W.quad_mesh(2, 2, periodic_x=False, periodic_y=False)
    np.testing.assert_array_equal(mi.cell_nodes.reshape(-1, 4), np.array(g["cell_nodes"]))
    m = orc.OracleMesh.from_input(mi)
    assert m.max_faces == 4 and _sizes(m) == (4, 12, 12, 12)
    faces = np.array(g["faces"])
    np.testing.assert_array_equal(m.get("face_nodes"), faces[:, :2])
    np.testing.assert_array_equal(m.get("face_cells"), faces[:, 2:])
    np.testing.assert_array_equal(m.get("cell_faces"), np.array(g["cell_faces"]))
    np.testing.assert_array_equal(m.get("bfaces"), np.array(g["bfaces"][0]))
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    sp, si = m.get("stencil_ptr"), m.get("stencil_idx")
    for c in range(4):
        assert list(col[rp[c]:rp[c + 1]]) == g["bsr_rows"][c]
        assert list(si[sp[c]:sp[c + 1]]) == g["stencil"][c]
    m.reorder("rcm")
    np.testing.assert_array_equal(m.get("perm"), np.array(g["rcm_perm"][0]))
    np.testing.assert_array_equal(m.get("bfaces"), np.array(g["bfaces"][0]))   # face ids do not move with the cells


@pytest.mark.parametrize("kind", ["quads_periodic", "quads_channel", "quads_box", "mixed_box", "mixed_periodic"])
def test_brute_force_and_euler(orc, W, kind):
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    check_connectivity_against_brute(m.get, _sizes(m), mi.cell_nodes, mi.cell_ptr)
    nb = int((m.get("face_cells")[:, 1] < 0).sum())
    corners = int(mi.cell_ptr[-1])
    assert 2 * m.n_faces == corners + nb                  # handshake: every corner is one cell-face incidence
    assert m.nnzb == m.n_cells + corners - nb             # self + one block per interior cell-face incidence
    assert m.n_bfaces == nb and (np.diff(m.get("bfaces")) > 0).all()
    if kind == "quads_periodic":
        assert nb == 0 and m.n_faces == 2 * m.n_cells and m.nnzb == 5 * m.n_cells     # 5 blocks per row
        assert (np.diff(m.get("stencil_ptr")) == 8).all()                              # the 8 surrounding quads
    # RCM equals the independent serial reference (S11) on meshes with 2- to 4-neighbour cells
    ref = rcm_reference(m.get("bsr_rowptr"), m.get("bsr_col"))
    m.reorder("rcm")
    np.testing.assert_array_equal(m.get("perm"), ref)
    mp = mi.permuted(ref)
    check_connectivity_against_brute(m.get, _sizes(m), mp.cell_nodes, mp.cell_ptr)


def test_mesh_errors(orc, W):
    mi = W.quad_mesh(3, 3, periodic_x=False, periodic_y=False)
    bad = mi.cell_nodes.copy().reshape(-1, 4)
    badxy = mi.cell_xy.copy().reshape(-1, 4, 2)
    bad[4], badxy[4] = bad[4][::-1].copy(), badxy[4][::-1].copy()            # clockwise
    with pytest.raises(RuntimeError, match="counter-clockwise|convex"):
        orc.OracleMesh(mi.node_xy, bad.reshape(-1), badxy.reshape(-1, 2), mi.cell_ptr)
    xy = mi.cell_xy.copy().reshape(-1, 4, 2)
    xy[2, 2] = xy[2, 0] + 0.1 * (xy[2, 2] - xy[2, 0])                         # corner pulled inside: not convex
    with pytest.raises(RuntimeError, match="convex"):
        orc.OracleMesh(mi.node_xy, mi.cell_nodes, xy.reshape(-1, 2), mi.cell_ptr)
    with pytest.raises(RuntimeError):
        orc.OracleMesh.from_input(W.quad_mesh(2, 4))                          # periodic direction 2 cells wide
    cp = np.array([0, 5], dtype=np.int32)                                     # a pentagon
    with pytest.raises(RuntimeError, match="3 or 4"):
        orc.OracleMesh(np.zeros((5, 2)), np.arange(5, dtype=np.int32), None, cp)


# ------------------------------------------------------------------------------------------
# geometry
# ------------------------------------------------------------------------------------------
def test_geometry_against_greens_theorem(orc, W):
    """Area and area centroid of every cell from the boundary integrals A = 1/2 sum (x_k y_k+1 - x_k+1 y_k),
    A C_x = 1/6 sum (x_k + x_k+1)(x_k y_k+1 - x_k+1 y_k) in global coordinates (the oracle uses a triangle fan
    relative to corner 0); the two diagonal splits of a quadrilateral give the same centroid; unit outward
    normals close (sum n_k len_k = 0); areas tile the domain."""
    mi = meshes(W)["mixed_box"]
    m = orc.OracleMesh.from_input(mi)
    vol, cen = m.get("volume"), m.get("centroid")
    assert abs(vol.sum() - 3.5 * 2.5) < 1e-12
    cells = cells_as_lists(mi.cell_nodes, mi.cell_ptr)
    fnl, fc, cf = m.get("face_normal_len"), m.get("face_cells"), m.get("cell_faces")
    for c, a in enumerate(cells):
        X = mi.cell_xy[mi.cell_ptr[c]:mi.cell_ptr[c + 1]]
        x, y = X[:, 0], X[:, 1]
        x1, y1 = np.roll(x, -1), np.roll(y, -1)
        cr = x * y1 - x1 * y
        A = 0.5 * cr.sum()
        C = np.array([((x + x1) * cr).sum(), ((y + y1) * cr).sum()]) / (6 * A)
        assert abs(vol[c] - A) < 1e-13 and np.abs(cen[c] - C).max() < 1e-12
        if len(a) == 4:
            for d in (0, 1):   # split by the diagonal (d, d+2): area-weighted mean of the two triangles' centroids
                t1, t2 = X[[d, d + 1, d + 2]], X[[d + 2, (d + 3) % 4, d]]
                ar = lambda T: 0.5 * ((T[1, 0] - T[0, 0]) * (T[2, 1] - T[0, 1]) - (T[1, 1] - T[0, 1]) * (T[2, 0] - T[0, 0]))
                Cs = (ar(t1) * t1.mean(axis=0) + ar(t2) * t2.mean(axis=0)) / (ar(t1) + ar(t2))
                assert np.abs(cen[c] - Cs).max() < 1e-12
        s = np.zeros(2)
        for k in range(len(a)):
            f = cf[c, k]
            sign = 1.0 if fc[f, 0] == c else -1.0
            s += sign * fnl[f, :2] * fnl[f, 2]
            assert abs(np.hypot(*fnl[f, :2]) - 1) < 1e-14
            # outward: the normal points from the centroid towards the face midpoint
            mid = 0.5 * (X[k] + X[(k + 1) % len(a)])
            assert sign * fnl[f, :2] @ (mid - cen[c]) > 0
        assert np.abs(s).max() < 1e-13
    # rectangles: the centroid is the mean of the corners
    mr = W.quad_mesh(5, 3, 0.0, 2.0, 0.0, 1.0)
    o = orc.OracleMesh.from_input(mr)
    np.testing.assert_allclose(o.get("centroid"), mr.cell_xy.reshape(-1, 4, 2).mean(axis=1), atol=1e-15)
    np.testing.assert_allclose(o.get("volume"), 2.0 / 15.0, rtol=1e-14)


# ------------------------------------------------------------------------------------------
# reconstruction
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["quads_box", "mixed_box"])
def test_gradient_exact_for_linear_fields_and_limiter_closed_form(orc, W, kind):
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    cen = mi.centroids()
    a, gx, gy = RNG.uniform(-1, 1, 18), RNG.uniform(-1, 1, 18), RNG.uniform(-1, 1, 18)
    P = a + np.outer(cen[:, 0], gx) + np.outer(cen[:, 1], gy)
    grad, _ = orc.gradients(m, orc.default_numerics(), P)
    np.testing.assert_allclose(grad[:, :, 0], np.broadcast_to(gx, (m.n_cells, 18)), atol=1e-12)
    np.testing.assert_allclose(grad[:, :, 1], np.broadcast_to(gy, (m.n_cells, 18)), atol=1e-12)
    # Venkatakrishnan at K = 1 over the cell's 3 or 4 face midpoints, closed form on a linear field
    g = np.array([0.9, -0.6])
    lin = cen @ g
    _, phi = orc.gradients(m, orc.default_numerics(venkat_K=1.0), np.tile(lin[:, None], (1, 18)))
    sp, si, vol = m.get("stencil_ptr"), m.get("stencil_idx"), m.get("volume")
    active = 0
    for i in range(m.n_cells):
        js = si[sp[i]:sp[i + 1]]
        umax, umin = max(lin[js].max(), lin[i]), min(lin[js].min(), lin[i])
        X = mi.cell_xy[mi.cell_ptr[i]:mi.cell_ptr[i + 1]]
        eps2 = np.sqrt(vol[i]) ** 3
        exp = 1.0
        for k in range(len(X)):
            d2 = (0.5 * (X[k] + X[(k + 1) % len(X)]) - cen[i]) @ g
            d1 = (umax if d2 > 0 else umin) - lin[i]
            if d2 != 0:
                exp = min(exp, (d1 * d1 + eps2 + 2 * d1 * d2) / (d1 * d1 + 2 * d2 * d2 + d1 * d2 + eps2))
        assert abs(phi[i, 3] - exp) < 1e-11
        active += exp < 0.999
    assert active >= 4


def test_stencil_of_a_cartesian_quad_is_its_eight_neighbours_and_gradient_is_central(orc, W):
    """On a uniform Cartesian mesh the 8-cell vertex stencil with any radial weight is symmetric, so the
    least-squares gradient of a QUADRATIC field is exact too (odd error terms cancel): a check of the stencil
    geometry across the periodic seam that a linear field cannot give."""
    mi = W.quad_mesh(8, 6, 0.0, 4.0, 0.0, 3.0)
    m = orc.OracleMesh.from_input(mi)
    cen = mi.centroids()
    X, Y = cen[:, 0], cen[:, 1]
    f = np.sin(2 * np.pi * X / 4.0) * np.cos(2 * np.pi * Y / 3.0)        # periodic on the domain
    grad, _ = orc.gradients(m, orc.default_numerics(), np.tile(f[:, None], (1, 18)))
    h = 0.5
    # the weighted LS on the symmetric 3x3 stencil is the weighted mean of the axial and diagonal central differences
    F = f.reshape(6, 8)
    sh = lambda a, dj, di: np.roll(np.roll(a, -dj, axis=0), -di, axis=1)
    w_ax, w_dg = 1.0 / h ** 2, 1.0 / (2 * h ** 2)
    gx = (w_ax * h * (sh(F, 0, 1) - sh(F, 0, -1)) + w_dg * h * (sh(F, 1, 1) - sh(F, 1, -1) + sh(F, -1, 1) - sh(F, -1, -1))) \
        / (2 * w_ax * h * h + 4 * w_dg * h * h)
    np.testing.assert_allclose(grad[:, 0, 0], gx.reshape(-1), atol=1e-12)


# ------------------------------------------------------------------------------------------
# residual and Jacobian on quadrilateral / mixed meshes
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["quads_periodic", "quads_channel", "mixed_box", "mixed_periodic"])
def test_free_stream_and_telescoping(orc, W, kind):
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, term_mask=1)
    P = np.tile(random_state(RNG, 1), (m.n_cells, 1))
    rhs, scale, _ = orc.assemble(m, ph, nu, P, jacobian=False)
    assert (np.abs(rhs) <= 1e-13 * scale.max(axis=0)).all() and scale.max() > 1.0
    if "periodic" in kind:
        P = random_state(RNG, m.n_cells)
        rhs, scale, _ = orc.assemble(m, ph, nu, P, jacobian=False)
        assert (np.abs(rhs.sum(axis=0)) <= 1e-12 * scale.sum(axis=0)).all() and np.abs(rhs).max() > 1e-3


def brute_force_jacobian(orc, m, ph, nu, P, grad, phi, dt):
    n = m.n_cells
    J = np.zeros((n * 18, n * 18))
    for j in range(n):
        for k in range(18):
            h = 1e-5 * max(abs(P[j, k]), 1.0 if k != 9 else 0.04)
            Pp, Pm = P.copy(), P.copy()
            Pp[j, k] += h
            Pm[j, k] -= h
            rp = orc.residual_frozen(m, ph, nu, Pp, grad, phi, P, P, dt)
            rm = orc.residual_frozen(m, ph, nu, Pm, grad, phi, P, P, dt)
            J[:, j * 18 + k] = -((rp - rm) / (2 * h)).reshape(-1)
    return J


@pytest.mark.parametrize("kind,bc", [("quads_periodic", None), ("mixed_box", "mixed-tags")])
def test_jacobian_vs_brute_force(orc, W, kind, bc):
    """Forward-difference blocks against central differences of the frozen residual (S7, S8) on <= 64 cells with
    3- and 4-face cells; with all three boundary rules on the hull: the transmissive and wall far sides move with
    the inner state, the ghost state does not, and the brute force sees exactly that."""
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    assert m.n_cells <= 64
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    cen = mi.centroids()
    # (the noisy wave of config 1 sits at Mbar = M_inf on this mesh, where f_a has a kink: there the forward and
    # the central difference differ by 4e-5 of the row; a generic state keeps the comparison sharp)
    P = random_state(RNG, m.n_cells) if kind == "quads_periodic" else W.wave_state(cen / 3.5, seed=5)
    if bc:
        tags = (np.arange(m.n_bfaces) % 3).astype(np.int32)
        m.set_bc(tags, random_state(RNG, m.n_bfaces))
    dt = 1e-3
    grad, phi = orc.gradients(m, nu, P)
    rhs, scale, vals = orc.assemble(m, ph, nu, P, dt=dt)
    np.testing.assert_array_equal(orc.residual_frozen(m, ph, nu, P, grad, phi, P, P, dt), rhs)
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    A = bsr_to_dense(vals, rp, col)
    J = brute_force_jacobian(orc, m, ph, nu, P, grad, phi, dt)
    err = np.abs(A - J) / np.abs(J).max(axis=1, keepdims=True)
    assert err.max() < 1e-5, err.max()
    em = np.concatenate([np.arange(18 * i, 18 * i + 8) for i in range(m.n_cells)])
    assert err[em].max() < 1e-9, err[em].max()
    mask = np.kron(bsr_to_dense(np.ones_like(vals), rp, col)[::18, ::18] > 0, np.ones((18, 18))) > 0
    assert np.abs(J[~mask]).max() == 0.0
    assert int(np.diff(rp).max()) == 5                     # a quadrilateral with four neighbours: 5 blocks


def test_exact_wave_converges_at_second_order_on_the_papers_quad_meshes(orc, W):
    """The external pin of tests/test_exact_wave.py on the mesh type the paper used (2N x N Cartesian
    quadrilaterals, L433): the paper's exact circularly polarised wave (Eq. 15-18) makes the spatial residual
    converge at second order -- here pointwise, without the quad averaging the split triangles need."""
    c, mass_ratio = 20.0, 25.0
    errs = []
    for n in (8, 16, 32):
        m = W.quad_mesh(2 * n, n, 0.0, 2.0 * np.pi, 0.0, np.pi)
        P, dU, w = exact_wave(m.centroids()[:, 0], 0.3, c, mass_ratio)
        o = orc.OracleMesh.from_input(m)
        pc = orc.physics_c(W.Physics(mass_ratio=mass_ratio, c=c))
        nu = orc.default_numerics(pc, venkat_K=1e9, term_mask=3)
        rhs, _, _ = orc.assemble(o, pc, nu, P, dt=1.0, jacobian=False)
        errs.append(np.abs(rhs / o.get("volume")[:, None] - dU).max(axis=0))
    check_convergence(np.array(errs), np.abs(dU).max(axis=0), c)


# ------------------------------------------------------------------------------------------
# boundary rules (L260; S9, S24)
# ------------------------------------------------------------------------------------------
def test_wall_ghost_is_an_involution_and_closes_the_wall(orc):
    """S24: the mirror state; mirrored twice it is the state again; the face mean has B.n = 0, E_t = 0, u.n = 0;
    and the numerical flux through the wall carries no mass, no energy, no tangential or z momentum, no flux of
    Psi, of tangential B or of normal E."""
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    for th in RNG.uniform(0, 2 * np.pi, 6):
        nx, ny = np.cos(th), np.sin(th)
        P = random_state(RNG, 1)[0]
        G = orc.wall_ghost(P, nx, ny)
        np.testing.assert_allclose(orc.wall_ghost(G, nx, ny), P, atol=1e-15)
        M = 0.5 * (P + G)
        t = np.array([-ny, nx])
        assert abs(M[0] * nx + M[1] * ny) < 1e-15 and abs(M[3:5] @ t) < 1e-15 and abs(M[5]) < 1e-15
        for s in (0, 1):
            assert abs(M[10 + 3 * s] * nx + M[11 + 3 * s] * ny) < 1e-15
        np.testing.assert_array_equal(G[[8, 9, 16, 17, 2, 6, 12, 15]], P[[8, 9, 16, 17, 2, 6, 12, 15]])
        H = orc.flux_face(ph, nu, P, G, nx, ny)
        scale = np.abs(orc.phys_flux(ph, P, nx, ny)).max()
        assert max(abs(H[8]), abs(H[9]), abs(H[16]), abs(H[17])) < 1e-14 * scale      # mass, energy
        assert abs(H[6]) < 1e-14 * scale                                               # Psi row: c^2 B.n
        assert abs(H[0:2] @ t) < 1e-14 * scale and abs(H[2]) < 1e-14 * scale           # Faraday, tangential rows
        assert abs(H[3] * nx + H[4] * ny) < 1e-14 * scale                              # normal Ampere row
        for s in (0, 1):
            mom = H[10 + 3 * s:13 + 3 * s]
            assert abs(mom[:2] @ t) < 1e-14 * scale and abs(mom[2]) < 1e-14 * scale    # only pressure, along n
            assert mom[:2] @ np.array([nx, ny]) > 0


def test_ghost_rule_reproduces_an_interior_face(orc, W):
    """A ghost-state boundary that is handed the neighbour's reconstructed face state is an interior face.  With a
    linear field and the limiter off the reconstruction is exact for any stencil, so cutting a mesh in two and
    feeding the cut faces the linear field's values at their midpoints must give, in the remaining half, the rows
    of the whole mesh: residual to rounding, and the diagonal blocks to the accuracy of the differences (the
    ghost state is held fixed, exactly as the far cell's state is when the own cell is perturbed)."""
    whole = W.quad_mesh(8, 5, 0.0, 4.0, 0.0, 2.5, periodic_x=False, periodic_y=False, jitter=0.2, seed=8, tri_every=3)
    ow = orc.OracleMesh.from_input(whole)
    cen = whole.centroids()
    keep = np.nonzero(cen[:, 0] < 2.0)[0]                                   # left half (cut along a jittered line)
    cnt = np.diff(whole.cell_ptr)[keep]
    cp = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
    src = np.concatenate([np.arange(whole.cell_ptr[c], whole.cell_ptr[c + 1]) for c in keep])
    half = W.MeshInput(whole.node_xy, whole.cell_nodes[src], whole.cell_xy[src], "half", cp)
    oh = orc.OracleMesh.from_input(half)
    a, gx, gy = RNG.uniform(0.5, 1.0, 18), RNG.uniform(-0.05, 0.05, 18), RNG.uniform(-0.05, 0.05, 18)
    lin = lambda xy: a + np.outer(xy[:, 0], gx) + np.outer(xy[:, 1], gy)
    a[9] /= 25.0; gx[9] /= 25.0; gy[9] /= 25.0
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, venkat_K=1e12)
    Pw = lin(cen)
    rhs_w, sc_w, vals_w = orc.assemble(ow, ph, nu, Pw)
    # boundary faces of the half mesh: the old hull stays transmissive, the cut gets ghost states
    bf = oh.get("bfaces")
    fn = oh.get("face_nodes")[bf]
    mid = 0.5 * (whole.node_xy[fn[:, 0]] + whole.node_xy[fn[:, 1]])
    hull = (np.abs(mid[:, 0]) < 1e-12) | (np.abs(mid[:, 1]) < 1e-12) | (np.abs(mid[:, 1] - 2.5) < 1e-12)
    tags = np.where(hull, orc.BC_TRANSMISSIVE, orc.BC_GHOST).astype(np.int32)
    assert (tags == orc.BC_GHOST).sum() >= 5
    oh.set_bc(tags, lin(mid))
    rhs_h, sc_h, vals_h = orc.assemble(oh, ph, nu, Pw[keep])
    np.testing.assert_allclose(rhs_h, rhs_w[keep], rtol=0, atol=1e-12 * sc_w.max())
    rpw, colw, rph, colh = ow.get("bsr_rowptr"), ow.get("bsr_col"), oh.get("bsr_rowptr"), oh.get("bsr_col")
    for r, c in enumerate(keep):
        dw = vals_w[rpw[c] + list(colw[rpw[c]:rpw[c + 1]]).index(c)]
        dh = vals_h[rph[r] + list(colh[rph[r]:rph[r + 1]]).index(r)]
        np.testing.assert_allclose(dh, dw, rtol=0, atol=1e-7 * np.abs(dw).max())
    # not vacuous: with the transmissive rule on the cut (whose far side moves with the inner state) the residual
    # is the same on this linear field, but the diagonal blocks of the cells at the cut are different ones
    oh.set_bc(np.zeros(oh.n_bfaces, dtype=np.int32))
    _, _, vals_t = orc.assemble(oh, ph, nu, Pw[keep])
    assert np.abs(vals_t - vals_h).max() > 1e-3 * np.abs(vals_h).max()    # (the BDF2 diagonal, 3 Omega / 2 dt, sets the max)


def test_boundary_tags_survive_reordering(orc, W):
    mi = meshes(W)["mixed_box"]
    m = orc.OracleMesh.from_input(mi)
    tags = (np.arange(m.n_bfaces) % 3).astype(np.int32)
    ghost = random_state(RNG, m.n_bfaces)
    m.set_bc(tags, ghost)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    P = W.gem_state(mi.centroids()) + RNG.uniform(-1e-3, 1e-3, (m.n_cells, 18))
    rhs0, sc0, _ = orc.assemble(m, ph, nu, P, jacobian=False)
    bf0 = m.get("bfaces").copy()
    m.reorder("rcm")
    perm = m.get("perm")
    np.testing.assert_array_equal(m.get("bfaces"), bf0)
    np.testing.assert_array_equal(m.get("bc_tags"), tags)
    rhs1, _, _ = orc.assemble(m, ph, nu, P[perm], jacobian=False)
    # (not bit for bit: a face's L cell, whose corners define its normal, can change with the numbering)
    np.testing.assert_allclose(rhs1, rhs0[perm], rtol=0, atol=1e-13 * sc0.max())
    with pytest.raises(RuntimeError, match="ghost"):
        m.set_bc(tags, None)
