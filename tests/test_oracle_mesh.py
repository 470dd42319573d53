"""Pins for the oracle's connectivity, geometry, stencil, BSR pattern and RCM."""
import numpy as np
import pytest

from helpers import (read_golden_sections, check_connectivity_against_brute, rcm_reference, bandwidth)


def _sizes(m):
    return (m.n_cells, m.n_faces, m.nnzb, m.n_stencil)


def test_golden_2x2(orc, W):
    """tests/golden/mesh_2x2.txt: hand-worked faces, cell_faces, BSR rows, stencil, RCM."""
    g = read_golden_sections("mesh_2x2.txt")
    mi = W.split_quad_mesh(2, 2, periodic_x=False, periodic_y=False)
    np.testing.assert_array_equal(mi.cell_nodes, np.array(g["cell_nodes"]))
    m = orc.OracleMesh.from_input(mi)
    faces = np.array(g["faces"])
    np.testing.assert_array_equal(m.get("face_nodes"), faces[:, :2])
    np.testing.assert_array_equal(m.get("face_cells"), faces[:, 2:])
    np.testing.assert_array_equal(m.get("cell_faces"), np.array(g["cell_faces"]))
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    sp, si = m.get("stencil_ptr"), m.get("stencil_idx")
    for c in range(8):
        assert list(col[rp[c]:rp[c + 1]]) == g["bsr_rows"][c]
        assert list(si[sp[c]:sp[c + 1]]) == g["stencil"][c]
    m.reorder("rcm")
    np.testing.assert_array_equal(m.get("perm"), np.array(g["rcm_perm"][0]))


@pytest.mark.parametrize("kind", ["periodic", "channel", "delaunay"])
def test_brute_force_and_euler(orc, W, kind):
    if kind == "periodic":
        mi = W.split_quad_mesh(6, 5)
    elif kind == "channel":
        mi = W.split_quad_mesh(7, 4, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False)
    else:
        mi = W.delaunay_mesh(9, 7, *W.GEM_DOMAIN, jitter=0.3, seed=5, shuffle_cells=True)
    m = orc.OracleMesh.from_input(mi)
    check_connectivity_against_brute(m.get, _sizes(m), mi.cell_nodes)
    nc = m.n_cells
    nb = int((m.get("face_cells")[:, 1] < 0).sum())
    # Euler / handshake counts (S10): nf = (3 nc + nb)/2 ; nnzb = 4 nc - nb
    assert 2 * m.n_faces == 3 * nc + nb
    assert m.nnzb == 4 * nc - nb
    if kind == "periodic":
        assert nb == 0 and 2 * m.n_faces == 3 * nc
    if kind == "channel":
        assert nb == 2 * 7
    if kind == "delaunay":
        assert nc == 2 * 8 * 6 and nb == 2 * (8 + 6)


def test_geometry_closed_forms(orc, W):
    """Areas sum to the domain area; face normals are unit, outward, and closed per cell
    (sum_k n_k len_k = 0, the discrete Gauss identity behind free-stream preservation)."""
    mi = W.delaunay_mesh(11, 8, *W.GEM_DOMAIN, jitter=0.3, seed=1)
    m = orc.OracleMesh.from_input(mi)
    vol = m.get("volume")
    assert abs(vol.sum() - 25.6 * 12.8) < 1e-10
    np.testing.assert_allclose(m.get("centroid"), mi.centroids(), rtol=0, atol=1e-13)
    fnl, fc, cf = m.get("face_normal_len"), m.get("face_cells"), m.get("cell_faces")
    np.testing.assert_allclose(np.hypot(fnl[:, 0], fnl[:, 1]), 1.0, atol=1e-14)
    acc = np.zeros((m.n_cells, 2))
    for c in range(m.n_cells):
        for k in range(3):
            f = cf[c, k]
            s = 1.0 if fc[f, 0] == c else -1.0
            acc[c] += s * fnl[f, :2] * fnl[f, 2]
    assert np.abs(acc).max() < 1e-13
    # face length equals the distance of its two nodes; normal is perpendicular to the edge
    fn = m.get("face_nodes")
    e = mi.node_xy[fn[:, 1]] - mi.node_xy[fn[:, 0]]
    np.testing.assert_allclose(fnl[:, 2], np.hypot(e[:, 0], e[:, 1]), rtol=1e-14)
    assert np.abs((e * fnl[:, :2]).sum(axis=1)).max() < 1e-13
    # outward from L: normal points away from L's centroid
    cenL = m.get("centroid")[fc[:, 0]]
    mid = 0.5 * (mi.node_xy[fn[:, 0]] + mi.node_xy[fn[:, 1]])
    assert (((mid - cenL) * fnl[:, :2]).sum(axis=1) > 0).all()


def test_rcm_matches_serial_reference_and_reduces_bandwidth(orc, W):
    mi = W.delaunay_mesh(13, 9, *W.GEM_DOMAIN, jitter=0.3, seed=7, shuffle_cells=True)
    m = orc.OracleMesh.from_input(mi)
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    bw0 = bandwidth(rp, col)
    ref = rcm_reference(rp, col)
    m.reorder("rcm")
    perm = m.get("perm")
    np.testing.assert_array_equal(perm, ref)
    assert sorted(perm.tolist()) == list(range(m.n_cells))
    bw1 = bandwidth(m.get("bsr_rowptr"), m.get("bsr_col"))
    assert bw1 < bw0
    # the reordered mesh is the same mesh: brute force on the permuted input
    check_connectivity_against_brute(m.get, _sizes(m), mi.cell_nodes[perm])


def test_mesh_errors(orc, W):
    mi = W.split_quad_mesh(3, 3, periodic_x=False, periodic_y=False)
    bad = mi.cell_nodes.copy()
    bad[0] = bad[0][::-1]                  # clockwise
    with pytest.raises(RuntimeError):
        orc.OracleMesh(mi.node_xy, bad, None)
    with pytest.raises(RuntimeError):      # periodic direction only 2 cells wide
        orc.OracleMesh.from_input(W.split_quad_mesh(2, 4))


@pytest.mark.parametrize("n", [3, 4, 13, 40])
def test_fan_stencil_is_everyone_else(orc, W, n):
    """Closed fan of n triangles around a hub: the vertex-neighbour stencil of every cell is all other cells, the
    face neighbours are the two adjacent ones (brute force on the definition)."""
    mi = W.fan_mesh(n, seed=n)
    m = orc.OracleMesh.from_input(mi)
    assert (m.n_cells, m.n_faces, m.nnzb, m.n_stencil) == (n, 2 * n, 3 * n, n * (n - 1))
    sp, si = m.get("stencil_ptr"), m.get("stencil_idx")
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    for c in range(n):
        assert list(si[sp[c]:sp[c + 1]]) == [j for j in range(n) if j != c]
        assert list(col[rp[c]:rp[c + 1]]) == sorted({(c - 1) % n, c, (c + 1) % n})
    check_connectivity_against_brute(m.get, _sizes(m), mi.cell_nodes)
    assert (m.get("volume") > 0).all()


def test_fan_gradient_is_exact_for_linear_fields(orc, W):
    """Least squares over a 39-entry stencil reproduces a linear field's gradient; the limiter leaves it alone when
    K is huge (S12, S13)."""
    mi = W.fan_mesh(40, seed=3)
    m = orc.OracleMesh.from_input(mi)
    cen = mi.centroids()
    a = np.linspace(-1.0, 1.0, 18)
    b = np.linspace(0.5, -0.7, 18)
    P = 2.0 + a[None, :] * cen[:, :1] + b[None, :] * cen[:, 1:2]
    grad, phi = orc.gradients(m, orc.default_numerics(venkat_K=1e9), P)
    np.testing.assert_allclose(grad[:, :, 0], np.broadcast_to(a, (40, 18)), atol=1e-11)
    np.testing.assert_allclose(grad[:, :, 1], np.broadcast_to(b, (40, 18)), atol=1e-11)
    np.testing.assert_allclose(phi, 1.0, atol=1e-9)
