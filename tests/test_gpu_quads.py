"""GPU parity on quadrilateral and mixed meshes and with the three boundary rules: libtfa through
the C ABI against the CPU oracle, element by element; same tolerances as tests/test_gpu_parity.py."""
import numpy as np
import pytest

from conftest import random_state
from helpers import (RES_TOL, JAC_TOL, residual_error, jacobian_error_blocks, check_connectivity_against_brute)
from test_gpu_parity import api, dev, INT_ITEMS, sweep_every_row  # noqa: F401 (api: fixture)
from test_oracle_quads import meshes

pytestmark = pytest.mark.gpu

KINDS = ["quads_periodic", "quads_channel", "quads_box", "mixed_box", "mixed_periodic"]


def mixed_tags(m, rng):
    """All three rules on the hull, cyclically; ghost states for every boundary face (only GHOST rows are read)."""
    tags = (np.arange(m.n_bfaces) % 3).astype(np.int32)
    return tags, random_state(rng, max(m.n_bfaces, 1))[:m.n_bfaces]


# ------------------------------------------------------------------------------------------
# a1 on quadrilateral / mixed meshes
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", KINDS)
def test_connectivity_geometry_rcm_bit_exact(api, orc, W, kind):
    mi = meshes(W)[kind]
    g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
    assert (g.n_cells, g.n_faces, g.nnzb, g.n_stencil, g.max_faces, g.n_bfaces) == \
        (o.n_cells, o.n_faces, o.nnzb, o.n_stencil, o.max_faces, o.n_bfaces)
    assert g.max_faces == 4
    for item in INT_ITEMS + ["bfaces", "bc_tags"]:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)
    check_connectivity_against_brute(g.get, (g.n_cells, g.n_faces, g.nnzb, g.n_stencil), mi.cell_nodes, mi.cell_ptr)
    nbr, cf, fc = g.get("cell_nbr"), g.get("cell_faces"), g.get("face_cells")
    for c in range(g.n_cells):
        for k in range(4):
            if cf[c, k] < 0:
                assert nbr[c, k] == -1 and k == 3          # a triangle's empty fourth slot
            else:
                L, R = fc[cf[c, k]]
                assert nbr[c, k] == (R if L == c else L)
    for item in ("volume", "centroid", "face_normal_len"):
        np.testing.assert_allclose(g.get(item), o.get(item), rtol=1e-13, atol=1e-15, err_msg=item)
    g.reorder("rcm")
    o.reorder("rcm")
    for item in INT_ITEMS + ["bfaces"]:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg="rcm " + item)
    p2 = np.random.default_rng(0).permutation(g.n_cells).astype(np.int32)
    g.reorder("user", p2)
    o.reorder("user", p2)
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg="user " + item)


def test_golden_quad_mesh_on_the_gpu(api, W):
    from helpers import read_golden_sections
    gold = read_golden_sections("quad_2x2.txt")
    g = api.Mesh.from_input(W.quad_mesh(2, 2, periodic_x=False, periodic_y=False))
    faces = np.array(gold["faces"])
    np.testing.assert_array_equal(g.get("face_nodes"), faces[:, :2])
    np.testing.assert_array_equal(g.get("face_cells"), faces[:, 2:])
    np.testing.assert_array_equal(g.get("cell_faces"), np.array(gold["cell_faces"]))
    np.testing.assert_array_equal(g.get("bfaces"), np.array(gold["bfaces"][0]))
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    for c in range(4):
        assert list(col[rp[c]:rp[c + 1]]) == gold["bsr_rows"][c]
    g.reorder("rcm")
    np.testing.assert_array_equal(g.get("perm"), np.array(gold["rcm_perm"][0]))


def test_mesh_errors(api, W):
    mi = W.quad_mesh(3, 3, periodic_x=False, periodic_y=False)
    xy = mi.cell_xy.copy().reshape(-1, 4, 2)
    xy[2, 2] = xy[2, 0] + 0.1 * (xy[2, 2] - xy[2, 0])                      # not convex
    with pytest.raises(api.TfaError) as e:
        api.Mesh(mi.node_xy, mi.cell_nodes, xy.reshape(-1, 2), mi.cell_ptr)
    assert e.value.code == -2 and "convex" in str(e.value)
    cn = mi.cell_nodes.copy().reshape(-1, 4)
    cxy = mi.cell_xy.copy().reshape(-1, 4, 2)
    cn[4], cxy[4] = cn[4][::-1].copy(), cxy[4][::-1].copy()                # clockwise
    with pytest.raises(api.TfaError) as e:
        api.Mesh(mi.node_xy, cn.reshape(-1), cxy.reshape(-1, 2), mi.cell_ptr)
    assert e.value.code == -2
    with pytest.raises(api.TfaError) as e:                                  # a pentagon
        api.Mesh(np.zeros((5, 2)), np.arange(5, dtype=np.int32), None, np.array([0, 5], dtype=np.int32))
    assert e.value.code == -1
    with pytest.raises(api.TfaError):
        api.Mesh.from_input(W.quad_mesh(2, 4))                              # periodic direction 2 cells wide
    g = api.Mesh.from_input(mi)
    with pytest.raises(api.TfaError):
        g.set_bc(np.full(g.n_bfaces, 7, dtype=np.int32))                    # unknown tag
    # a ghost-tagged mesh needs ghost states of the right size
    g.set_bc(np.full(g.n_bfaces, api.BC_GHOST, dtype=np.int32))
    ctx = api.Context()
    P = dev(W.gem_state(mi.centroids()))
    with pytest.raises(api.TfaError) as e:
        ctx.assemble(g, P)
    assert e.value.code == -1 and "ghost" in str(e.value)
    ctx.set_ghost_states(dev(random_state(np.random.default_rng(1), g.n_bfaces + 1)))
    with pytest.raises(api.TfaError):
        ctx.assemble(g, P)
    ctx.set_ghost_states(dev(random_state(np.random.default_rng(1), g.n_bfaces)))
    ctx.assemble(g, P)
    ctx.check()
    # a single quadrilateral: 4 boundary faces, one block
    one = api.Mesh(np.array([[0.0, 0], [1, 0], [1.2, 1.1], [0, 1]]), np.arange(4, dtype=np.int32), None,
                   np.array([0, 4], dtype=np.int32))
    assert (one.n_cells, one.n_faces, one.nnzb, one.n_stencil, one.n_bfaces) == (1, 4, 1, 0, 4)
    rhs, vals = api.Context().assemble(one, dev(random_state(np.random.default_rng(0), 1)))
    assert np.isfinite(rhs.cpu().numpy()).all() and vals.shape == (1, 18, 18)


# ------------------------------------------------------------------------------------------
# a2..a7 on quadrilateral / mixed meshes, with the boundary rules
# ------------------------------------------------------------------------------------------
def compare(api, orc, mi, P, Pn=None, Pnm1=None, dt=1e-3, bc_seed=None, numerics_kw=None, reorder=None):
    numerics_kw = numerics_kw or {}
    g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
    ctx = api.Context(numerics=api.default_numerics(**numerics_kw))
    if bc_seed is not None and g.n_bfaces:
        tags, ghost = mixed_tags(g, np.random.default_rng(bc_seed))
        g.set_bc(tags)
        o.set_bc(tags, ghost)
        ctx.set_ghost_states(dev(ghost))
    if reorder:
        g.reorder(reorder)
        o.reorder(reorder)
        perm = g.get("perm")
        np.testing.assert_array_equal(perm, o.get("perm"))
        np.testing.assert_array_equal(g.get("bc_tags"), o.get("bc_tags"))
        P, Pn, Pnm1 = P[perm], None if Pn is None else Pn[perm], None if Pnm1 is None else Pnm1[perm]
    ph_o = orc.physics_c()
    nu_o = orc.default_numerics(ph_o, **numerics_kw)
    d = lambda x: None if x is None else dev(x)
    rhs, vals = ctx.assemble(g, dev(P), d(Pn), d(Pnm1), dt)
    rhs_r, _ = ctx.assemble(g, dev(P), d(Pn), d(Pnm1), dt, jacobian=False)      # the residual-only kernel
    ctx.check()
    rhs_o, sc_o, vals_o = orc.assemble(o, ph_o, nu_o, P, Pn, Pnm1, dt)
    rp = g.get("bsr_rowptr")
    er = residual_error(rhs.cpu().numpy(), rhs_o, sc_o)
    err = residual_error(rhs_r.cpu().numpy(), rhs_o, sc_o)
    ej = jacobian_error_blocks(vals.cpu().numpy(), vals_o, rp)
    return er, err, ej, (g, rhs.cpu().numpy(), vals.cpu().numpy(), rhs_o, vals_o)


@pytest.mark.parametrize("kind,bc", [(k, False) for k in KINDS] + [(k, True) for k in KINDS if "periodic" not in k])
def test_assembly_parity_small(api, orc, W, kind, bc):
    mi = meshes(W)[kind]
    cen = mi.centroids()
    if kind == "quads_periodic":
        P = W.wave_state(cen, seed=0)
    else:
        P = W.gem_state(cen) + np.random.default_rng(1).uniform(-1e-3, 1e-3, (mi.n_cells, 18))
    er, err, ej, (g, rhs, vals, rhs_o, vals_o) = compare(api, orc, mi, P, W.perturb(P, 11, 1e-4), W.perturb(P, 12, 1e-4),
                                                       bc_seed=7 if bc else None)
    assert er < RES_TOL and err < RES_TOL and ej < JAC_TOL, (er, err, ej)
    if kind == "quads_periodic":
        assert g.nnzb == 5 * g.n_cells
        # structural zeros of the off-diagonal blocks are exact zeros
        grp = np.array([0] * 8 + [1, 2] + [1] * 3 + [2] * 3 + [1, 2])
        coupled = grp[:, None] == grp[None, :]
        rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
        offd = np.repeat(np.arange(g.n_cells), np.diff(rp)) != col
        assert (vals[offd][:, ~coupled] == 0.0).all() and (vals_o[offd][:, ~coupled] == 0.0).all()


@pytest.mark.parametrize("mask", [1, 2, 4, 3])
def test_term_masks_and_constants_on_a_mixed_mesh_with_boundaries(api, orc, W, mask):
    mi = meshes(W)["mixed_box"]
    P = random_state(np.random.default_rng(mask), mi.n_cells, vel=1.2)        # sub- and supersonic faces
    kw = dict(term_mask=mask, venkat_K=0.5, lsq_weight_power=1.0, ausm_Kp=0.3, ausm_Ku=0.6, fd_delta=1e-5)
    er, err, ej, _ = compare(api, orc, mi, P, W.perturb(P, 1, 1e-3), W.perturb(P, 2, 1e-3), dt=2e-3, bc_seed=3,
                             numerics_kw=kw, reorder="rcm")
    assert er < RES_TOL and err < RES_TOL and ej < JAC_TOL, (er, err, ej)


def test_gradients_parity(api, orc, W):
    for kind in ("quads_channel", "mixed_box"):
        mi = meshes(W)[kind]
        g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
        P = random_state(np.random.default_rng(5), g.n_cells)
        for K, p in ((1.0, 2.0), (0.3, 1.0)):
            ctx = api.Context(numerics=api.default_numerics(venkat_K=K, lsq_weight_power=p))
            grad, phi = ctx.gradients(g, dev(P))
            go, po = orc.gradients(o, orc.default_numerics(venkat_K=K, lsq_weight_power=p), P)
            np.testing.assert_allclose(grad.cpu().numpy(), go, rtol=0, atol=1e-12 * np.abs(go).max())
            np.testing.assert_allclose(phi.cpu().numpy(), po, rtol=0, atol=1e-11)


def test_determinism_nan_canary_and_boundary_tag_changes(api, W):
    """Bit-identical reruns with every entry written, on a mixed mesh with boundary rules; changing the tags of an
    existing mesh takes effect at the next assembly and going back restores the first result bit for bit."""
    import torch
    mi = meshes(W)["mixed_box"]
    g = api.Mesh.from_input(mi)
    g.reorder("rcm")
    rng = np.random.default_rng(2)
    tags, ghost = mixed_tags(g, rng)
    ctx = api.Context()
    ctx.set_ghost_states(dev(ghost))
    P = dev((W.gem_state(mi.centroids()) + rng.uniform(-1e-3, 1e-3, (mi.n_cells, 18)))[g.get("perm")])

    def run(fill):
        rhs = torch.full((g.n_cells, 18), fill, dtype=torch.float64, device="cuda")
        vals = torch.full((g.nnzb, 18, 18), fill, dtype=torch.float64, device="cuda")
        ctx.assemble(g, P, rhs=rhs, vals=vals)
        ctx.check()
        return rhs, vals
    g.set_bc(tags)
    r1, v1 = run(float("nan"))
    r2, v2 = run(7.0)
    assert torch.equal(r1, r2) and torch.equal(v1, v2) and bool(torch.isfinite(v1).all())
    g.set_bc(np.zeros(g.n_bfaces, dtype=np.int32))
    r3, v3 = run(0.0)
    assert not torch.equal(r1, r3)
    g.set_bc(tags)
    r4, v4 = run(1.0)
    assert torch.equal(r1, r4) and torch.equal(v1, v4)


def test_walls_close_the_box_on_the_gpu(api, W):
    """GPU-side invariant, no oracle: in a box whose whole hull is a conducting wall nothing flows out, so the
    domain sums of the mass and energy rows of the convective residual vanish (interior faces telescope, wall
    faces carry no mass or energy), while with the transmissive rule they do not."""
    mi = W.quad_mesh(9, 7, 0.0, 3.0, 0.0, 2.0, periodic_x=False, periodic_y=False, jitter=0.25, seed=9, tri_every=4)
    g = api.Mesh.from_input(mi)
    ctx = api.Context(numerics=api.default_numerics(term_mask=1))
    P = dev(random_state(np.random.default_rng(3), g.n_cells))
    g.set_bc(np.full(g.n_bfaces, api.BC_WALL, dtype=np.int32))
    for jac in (False, True):
        rhs, _ = ctx.assemble(g, P, jacobian=jac)
        tot, mag = rhs.sum(dim=0).abs().cpu().numpy(), rhs.abs().sum(dim=0).cpu().numpy()
        assert (tot[[8, 9, 16, 17]] <= 1e-12 * mag[[8, 9, 16, 17]]).all(), (tot, mag)
        assert tot[10] > 1e-6 * mag[10]                       # momentum does feel the wall's pressure
    g.set_bc(np.zeros(g.n_bfaces, dtype=np.int32))
    rhs, _ = ctx.assemble(g, P, jacobian=False)
    tot, mag = rhs.sum(dim=0).abs().cpu().numpy(), rhs.abs().sum(dim=0).cpu().numpy()
    assert (tot[[8, 9]] > 1e-6 * mag[[8, 9]]).all()
    ctx.check()


def test_ghost_rule_reproduces_an_interior_face_on_the_gpu(api, W):
    """The cut-mesh pin of tests/test_oracle_quads.py on the CUDA path itself (no oracle): a linear field, limiter
    off; the left half of a mixed mesh with the cut faces fed the field's midpoint values as ghost states gives the
    rows the whole mesh gives."""
    whole = W.quad_mesh(8, 5, 0.0, 4.0, 0.0, 2.5, periodic_x=False, periodic_y=False, jitter=0.2, seed=8, tri_every=3)
    cen = whole.centroids()
    keep = np.nonzero(cen[:, 0] < 2.0)[0]
    cnt = np.diff(whole.cell_ptr)[keep]
    cp = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
    src = np.concatenate([np.arange(whole.cell_ptr[c], whole.cell_ptr[c + 1]) for c in keep])
    half = W.MeshInput(whole.node_xy, whole.cell_nodes[src], whole.cell_xy[src], "half", cp)
    rng = np.random.default_rng(4)
    a, gx, gy = rng.uniform(0.5, 1.0, 18), rng.uniform(-0.05, 0.05, 18), rng.uniform(-0.05, 0.05, 18)
    a[9] /= 25.0; gx[9] /= 25.0; gy[9] /= 25.0
    lin = lambda xy: a + np.outer(xy[:, 0], gx) + np.outer(xy[:, 1], gy)
    gw, gh = api.Mesh.from_input(whole), api.Mesh.from_input(half)
    ctx = api.Context(numerics=api.default_numerics(venkat_K=1e12))
    Pw = lin(cen)
    rhs_w, vals_w = ctx.assemble(gw, dev(Pw))
    bf = gh.get("bfaces")
    fn = gh.get("face_nodes")[bf]
    mid = 0.5 * (whole.node_xy[fn[:, 0]] + whole.node_xy[fn[:, 1]])
    hull = (np.abs(mid[:, 0]) < 1e-12) | (np.abs(mid[:, 1]) < 1e-12) | (np.abs(mid[:, 1] - 2.5) < 1e-12)
    gh.set_bc(np.where(hull, api.BC_TRANSMISSIVE, api.BC_GHOST).astype(np.int32))
    ctx.set_ghost_states(dev(lin(mid)))
    rhs_h, vals_h = ctx.assemble(gh, dev(Pw[keep]))
    ctx.check()
    rhs_w, rhs_h = rhs_w.cpu().numpy(), rhs_h.cpu().numpy()
    assert np.abs(rhs_h - rhs_w[keep]).max() < 1e-12 * np.abs(vals_w.cpu().numpy()).max() * np.abs(Pw).max()
    rpw, colw, rph, colh = gw.get("bsr_rowptr"), gw.get("bsr_col"), gh.get("bsr_rowptr"), gh.get("bsr_col")
    vw, vh = vals_w.cpu().numpy(), vals_h.cpu().numpy()
    for r, c in enumerate(keep):
        dw = vw[rpw[c] + list(colw[rpw[c]:rpw[c + 1]]).index(c)]
        dh = vh[rph[r] + list(colh[rph[r]:rph[r + 1]]).index(r)]
        assert np.abs(dh - dw).max() < 1e-7 * np.abs(dw).max()


def wall_y(g, o):
    """GEM channel: conducting walls on the y boundaries (the GEM challenge's own set-up)."""
    return np.full(g.n_bfaces, 2, dtype=np.int32), None


@pytest.mark.parametrize("name,bc", [("q1", None), ("q2", None), ("qm", wall_y)])
def test_full_size_every_row_quads(api, orc, W, name, bc):
    """The paper's own meshes at full size -- q1: 512 x 512 periodic quadrilaterals, double current sheet (L559,
    Table 9); q2: 256 x 128 periodic quadrilaterals, wave (L433, Table 4) -- and qm: 294 912 jittered
    quadrilaterals with every third one split into triangles, RCM order, conducting walls in y.  Every row."""
    w = W.make_workload(name)
    er, e3, ej = sweep_every_row(api, orc, W, w, bc=bc, flux_noise=0.0 if name == "q2" else 1e-3)
    assert er < RES_TOL and ej < JAC_TOL, (name, er, ej)
    assert e3.max() < RES_TOL, (name, e3)      # flux + source at their own scale (see test_full_size_every_row)


def test_linear_solve_kernels_on_a_quad_mesh(api, orc, W):
    """tfa_bsr_spmv, tfa_block_jacobi, tfa_gmres and the matrix-free operator on 5-block rows (and 3- to 5-block
    rows of a mixed mesh with boundary rules): against scipy on the assembled matrix."""
    import scipy.sparse as sp
    import scipy.sparse.linalg as spl
    import torch
    for kind, bc in (("quads_periodic", False), ("mixed_box", True)):
        mi = meshes(W)[kind]
        g = api.Mesh.from_input(mi)
        ctx = api.Context()
        rng = np.random.default_rng(6)
        if bc:
            tags, ghost = mixed_tags(g, rng)
            g.set_bc(tags)
            ctx.set_ghost_states(dev(ghost))
        P = W.wave_state(mi.centroids() / 3.5, seed=2)
        Pd = dev(P)
        rhs, vals = ctx.assemble(g, Pd, dt=0.05)
        rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
        A = sp.bsr_matrix((vals.cpu().numpy(), col, rp), shape=(18 * g.n_cells,) * 2).tocsr()
        x = rng.normal(size=18 * g.n_cells)
        y = api.bsr_spmv(g, vals, dev(x)).cpu().numpy()
        np.testing.assert_allclose(y, A @ x, rtol=0, atol=1e-13 * (abs(A) @ np.abs(x)).max())
        dinv = ctx.block_jacobi(g, vals)
        ctx.check()
        D = dinv.cpu().numpy()
        for i in range(0, g.n_cells, 5):
            blk = vals[rp[i] + list(col[rp[i]:rp[i + 1]]).index(i)].cpu().numpy()
            np.testing.assert_allclose(D[i] @ blk, np.eye(18), atol=1e-9)
        b = rhs.reshape(-1).contiguous()
        xs, its, rel = ctx.gmres(g, vals, b, dinv=dinv, restart=30, max_iters=200, rtol=1e-10)
        ref = spl.spsolve(A.tocsc(), b.cpu().numpy())
        assert rel <= 1e-10 and np.abs(xs.cpu().numpy() - ref).max() < 1e-6 * np.abs(ref).max()
        # matrix-free operator (limiter recomputed): close to the assembled one on this smooth state
        v = dev(rng.normal(size=(g.n_cells, 18)))
        jv = ctx.jvp(g, Pd, v, dt=0.05, eps=1e-7).cpu().numpy().reshape(-1)
        av = A @ v.cpu().numpy().reshape(-1)
        assert np.abs(jv - av).max() < 0.2 * np.abs(av).max()
        xj, itj, relj = ctx.gmres_jfnk(g, Pd, b, dt=0.05, dinv=dinv, restart=30, max_iters=200, rtol=1e-6)
        assert relj <= 1e-6
        ctx.check()
        torch.cuda.synchronize()
