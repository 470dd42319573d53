"""GPU parity tests: libtfa (through the C ABI binding) against the CPU oracle, element by element.

Tolerances are north_star's, read as in DESIGN.md (S18): residual 1e-12 of the per-variable
sum-of-|terms| scale; Jacobian 1e-8 of the row-maximum magnitude; connectivity bit-exact.
"""
import numpy as np
import pytest

from conftest import random_state, rot18
from helpers import (RES_TOL, JAC_TOL, residual_error, jacobian_error_rows, jacobian_error_blocks,
                     jacobian_error_padded, bsr_to_rows, check_connectivity_against_brute)

pytestmark = pytest.mark.gpu

INT_ITEMS = ["face_nodes", "face_cells", "cell_faces", "stencil_ptr", "stencil_idx", "bsr_rowptr", "bsr_col", "perm"]


@pytest.fixture(scope="module")
def api():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_1809_02532_b200 import build, api
    build.build()
    return api


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def small_meshes(W):
    return {
        "c1": W.make_workload("c1").mesh,
        "periodic7x5": W.split_quad_mesh(7, 5),
        "channel": W.split_quad_mesh(9, 6, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False),
        "box": W.split_quad_mesh(5, 4, periodic_x=False, periodic_y=False),
        "delaunay": W.delaunay_mesh(23, 17, *W.GEM_DOMAIN, jitter=0.3, seed=4, shuffle_cells=True),
    }


# ------------------------------------------------------------------------------------------
# a1: connectivity, geometry, reordering
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["c1", "periodic7x5", "channel", "box", "delaunay"])
def test_connectivity_bit_exact(api, orc, W, name):
    mi = small_meshes(W)[name]
    g = api.Mesh.from_input(mi)
    o = orc.OracleMesh.from_input(mi)
    assert (g.n_cells, g.n_faces, g.nnzb, g.n_stencil) == (o.n_cells, o.n_faces, o.nnzb, o.n_stencil)
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)
    check_connectivity_against_brute(g.get, (g.n_cells, g.n_faces, g.nnzb, g.n_stencil), mi.cell_nodes)
    # neighbour table is consistent with the face table
    nbr, cf, fc = g.get("cell_nbr"), g.get("cell_faces"), g.get("face_cells")
    for c in range(0, g.n_cells, 5):
        for k in range(3):
            L, R = fc[cf[c, k]]
            assert nbr[c, k] == (R if L == c else L)
    for item in ("volume", "centroid", "face_normal_len"):
        np.testing.assert_allclose(g.get(item), o.get(item), rtol=1e-14, atol=1e-15, err_msg=item)
    assert g.device_ptr("bsr_col") != 0 and g.device_ptr("bsr_rowptr") != 0


@pytest.mark.parametrize("name", ["c1", "channel", "delaunay"])
def test_rcm_bit_exact(api, orc, W, name):
    mi = small_meshes(W)[name]
    g = api.Mesh.from_input(mi)
    o = orc.OracleMesh.from_input(mi)
    g.reorder("rcm")
    o.reorder("rcm")
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)
    perm = g.get("perm")
    assert sorted(perm.tolist()) == list(range(g.n_cells))
    # a second, user-given permutation composes with the first
    rng = np.random.default_rng(0)
    p2 = rng.permutation(g.n_cells).astype(np.int32)
    g.reorder("user", p2)
    o.reorder("user", p2)
    np.testing.assert_array_equal(g.get("perm"), perm[p2])
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)


def test_rcm_disconnected_components(api, orc, W):
    """Two meshes glued into one node/cell list: RCM restarts at the min-(degree, id) unvisited cell."""
    a = W.split_quad_mesh(4, 3, periodic_x=False, periodic_y=False)
    b = W.delaunay_mesh(6, 5, *W.GEM_DOMAIN, jitter=0.3, seed=9)
    nodes = np.concatenate([a.node_xy, b.node_xy + 100.0])
    cells = np.concatenate([a.cell_nodes, b.cell_nodes + a.n_nodes]).astype(np.int32)
    rng = np.random.default_rng(3)
    cells = cells[rng.permutation(len(cells))]
    g = api.Mesh(nodes, cells)
    o = orc.OracleMesh(nodes, cells)
    g.reorder("rcm")
    o.reorder("rcm")
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)


@pytest.mark.parametrize("name", ["c1", "delaunay"])
def test_morton_order(api, orc, W, name):
    """tfa_mesh_reorder kind 3 (Z-order through the centroids, include/tfa.h).  The curve is the library's own choice, so
    what is checked is what is unique: the permutation is a bijection that sorts the cells by the interleaved 16-bit
    centroid coordinates written out here with numpy (ties by cell id), and every table after it equals the
    oracle's after the same permutation given as a user one.  Patches of 32 consecutive cells are compact: they
    touch fewer distinct stencil rows than in RCM order."""
    mi = small_meshes(W)[name]
    g = api.Mesh.from_input(mi)
    cen = g.get("centroid")
    g.reorder("morton")
    perm = g.get("perm")
    assert sorted(perm.tolist()) == list(range(g.n_cells))
    lo, hi = cen.min(axis=0), cen.max(axis=0)
    q = np.clip(np.floor((cen - lo) * (65535.0 / (hi - lo))), 0, 65535).astype(np.uint64)
    code = np.zeros(g.n_cells, dtype=np.uint64)
    for b in range(16):
        code |= ((q[:, 0] >> np.uint64(b)) & np.uint64(1)) << np.uint64(2 * b)
        code |= ((q[:, 1] >> np.uint64(b)) & np.uint64(1)) << np.uint64(2 * b + 1)
    np.testing.assert_array_equal(perm, np.lexsort((np.arange(g.n_cells), code)))
    o = orc.OracleMesh.from_input(mi)
    o.reorder("user", perm.astype(np.int32))
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)

    def rows_per_patch(mesh):
        sp, sc = mesh.get("stencil_ptr"), mesh.get("stencil_idx")
        return np.mean([len(np.unique(sc[sp[a]:sp[min(a + 32, mesh.n_cells)]]))
                        for a in range(0, mesh.n_cells, 32)])
    r = api.Mesh.from_input(mi)
    r.reorder("rcm")
    assert rows_per_patch(g) < rows_per_patch(r)


def test_mesh_errors_and_degenerate_sizes(api, W):
    mi = W.split_quad_mesh(3, 3, periodic_x=False, periodic_y=False)
    bad = mi.cell_nodes.copy()
    bad[4] = bad[4][::-1]
    with pytest.raises(api.TfaError) as e:
        api.Mesh(mi.node_xy, bad)
    assert e.value.code == -2 and "counter-clockwise" in str(e.value)
    with pytest.raises(api.TfaError) as e:
        api.Mesh.from_input(W.split_quad_mesh(2, 4))       # periodic direction 2 cells wide
    assert e.value.code == -2
    dup = np.concatenate([mi.cell_nodes, mi.cell_nodes[:1]])   # a node pair shared by 3 cells
    with pytest.raises(api.TfaError):
        api.Mesh(mi.node_xy, dup)
    g = api.Mesh.from_input(mi)
    with pytest.raises(api.TfaError) as e:
        g.reorder("user", np.zeros(g.n_cells, dtype=np.int32))
    assert e.value.code == -1
    # empty mesh and single triangle
    e0 = api.Mesh(np.zeros((0, 2)), np.zeros((0, 3), dtype=np.int32))
    assert (e0.n_cells, e0.n_faces, e0.nnzb) == (0, 0, 0)
    one = api.Mesh(np.array([[0.0, 0], [1, 0], [0, 1]]), np.array([[0, 1, 2]], dtype=np.int32))
    assert (one.n_cells, one.n_faces, one.nnzb, one.n_stencil) == (1, 3, 1, 0)
    ctx = api.Context()
    import torch
    P = dev(random_state(np.random.default_rng(0), 1))
    rhs, vals = ctx.assemble(one, P)
    torch.cuda.synchronize()
    assert np.isfinite(rhs.cpu().numpy()).all() and vals.shape == (1, 18, 18)
    rhs0, vals0 = ctx.assemble(e0, dev(np.zeros((0, 18))))
    assert rhs0.shape == (0, 18)


# ------------------------------------------------------------------------------------------
# a2: gradient + limiter
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["c1", "channel", "delaunay"])
@pytest.mark.parametrize("K,p", [(1.0, 2.0), (0.3, 1.0)])
def test_gradients_parity(api, orc, W, name, K, p):
    mi = small_meshes(W)[name]
    g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
    rng = np.random.default_rng(5)
    P = random_state(rng, g.n_cells)
    ctx = api.Context(numerics=api.default_numerics(venkat_K=K, lsq_weight_power=p))
    grad, phi = ctx.gradients(g, dev(P))
    go, po = orc.gradients(o, orc.default_numerics(venkat_K=K, lsq_weight_power=p), P)
    h = np.sqrt(o.get("volume")).min()
    np.testing.assert_allclose(grad.cpu().numpy(), go, rtol=0, atol=1e-12 * np.abs(go).max())
    np.testing.assert_allclose(phi.cpu().numpy(), po, rtol=0, atol=1e-11)
    assert h > 0


@pytest.mark.parametrize("n", [3, 4, 13, 40, 75])
def test_long_stencils_fan(api, orc, W, n):
    """Closed fans: every stencil has n - 1 entries (2, 3, 12, 39, 74): the stencil walk's batches of eight, its
    batch of four and its tail entries in every combination; connectivity, gradients and assembly."""
    mi = W.fan_mesh(n, seed=n)
    g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
    for item in INT_ITEMS:
        np.testing.assert_array_equal(g.get(item), o.get(item), err_msg=item)
    assert g.n_stencil == n * (n - 1)
    P = random_state(np.random.default_rng(n), n)
    ctx = api.Context()
    grad, phi = ctx.gradients(g, dev(P))
    go, po = orc.gradients(o, orc.default_numerics(), P)
    np.testing.assert_allclose(grad.cpu().numpy(), go, rtol=0, atol=1e-12 * np.abs(go).max())
    np.testing.assert_allclose(phi.cpu().numpy(), po, rtol=0, atol=1e-11)
    Pg = W.gem_state(mi.centroids()) + np.random.default_rng(1).uniform(-1e-3, 1e-3, (n, 18))
    er, ej, _ = compare_assembly(api, orc, mi, Pg, W.perturb(Pg, 11, 1e-4), W.perturb(Pg, 12, 1e-4))
    assert er < RES_TOL, er
    assert ej < JAC_TOL, ej


# ------------------------------------------------------------------------------------------
# a3..a7: residual + Jacobian
# ------------------------------------------------------------------------------------------
def compare_assembly(api, orc, mi, P, Pn=None, Pnm1=None, dt=1e-3, physics=None, numerics_kw=None,
                     reorder=None, rows=None):
    numerics_kw = numerics_kw or {}
    g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
    if reorder:
        g.reorder(reorder)
        o.reorder(reorder)
        perm = g.get("perm")
        np.testing.assert_array_equal(perm, o.get("perm"))
        P = P[perm]
        Pn = None if Pn is None else Pn[perm]
        Pnm1 = None if Pnm1 is None else Pnm1[perm]
    ph_g = api.default_physics(physics)
    ctx = api.Context(ph_g, api.default_numerics(ph_g, **numerics_kw))
    ph_o = orc.physics_c(physics)
    nu_o = orc.default_numerics(ph_o, **numerics_kw)
    rhs, vals = ctx.assemble(g, dev(P), None if Pn is None else dev(Pn), None if Pnm1 is None else dev(Pnm1), dt)
    ctx.check()
    rhs, vals = rhs.cpu().numpy(), vals.cpu().numpy()
    rhs_o, scale_o, vals_o = orc.assemble(o, ph_o, nu_o, P, Pn, Pnm1, dt, rows=rows)
    rp = g.get("bsr_rowptr")
    if rows is None:
        er = residual_error(rhs, rhs_o, scale_o)
        ej = jacobian_error_rows(bsr_to_rows(vals, rp), bsr_to_rows(vals_o, rp))
    else:
        # per-variable scale from the sampled rows
        er = residual_error(rhs[rows], rhs_o, scale_o)
        ej = jacobian_error_rows(bsr_to_rows(vals, rp, rows), vals_o)
    return er, ej, (rhs, vals, rhs_o, vals_o)


@pytest.mark.parametrize("name", ["c1", "periodic7x5", "channel", "box", "delaunay"])
def test_assembly_parity_small(api, orc, W, name):
    mi = small_meshes(W)[name]
    cen = mi.centroids()
    if name in ("c1", "periodic7x5"):
        P = W.wave_state(cen, seed=0)
    else:
        P = W.gem_state(cen) + np.random.default_rng(1).uniform(-1e-3, 1e-3, (mi.n_cells, 18))
    Pn = W.perturb(P, 11, 1e-4)
    Pnm1 = W.perturb(P, 12, 1e-4)
    er, ej, _ = compare_assembly(api, orc, mi, P, Pn, Pnm1)
    assert er < RES_TOL, er
    assert ej < JAC_TOL, ej


def test_config1_exact_recipe(api, orc, W):
    """BASELINE config 1: 512 cells, seed 0, P^n = P^{n-1} = P, dt = 1e-3, one assembly."""
    w = W.make_workload("c1")
    assert w.mesh.n_cells == 512
    er, ej, (rhs, vals, rhs_o, vals_o) = compare_assembly(api, orc, w.mesh, w.state, dt=w.dt, physics=w.physics)
    assert er < RES_TOL, er
    assert ej < JAC_TOL, ej
    # structural zeros of the off-diagonal blocks are exact zeros on the GPU as well
    grp = np.array([0] * 8 + [1, 2] + [1] * 3 + [2] * 3 + [1, 2])
    coupled = grp[:, None] == grp[None, :]
    g = api.Mesh.from_input(w.mesh)
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    rows = np.repeat(np.arange(g.n_cells), np.diff(rp))
    offd = rows != col
    assert (vals[offd][:, ~coupled] == 0.0).all() and (vals_o[offd][:, ~coupled] == 0.0).all()


@pytest.mark.parametrize("mask", [1, 2, 4, 3, 5, 6])
def test_term_masks(api, orc, W, mask):
    mi = small_meshes(W)["delaunay"]
    P = W.gem_state(mi.centroids()) + np.random.default_rng(2).uniform(-1e-3, 1e-3, (mi.n_cells, 18))
    er, ej, _ = compare_assembly(api, orc, mi, P, W.perturb(P, 1, 1e-3), W.perturb(P, 2, 1e-3),
                                 numerics_kw=dict(term_mask=mask))
    assert er < RES_TOL and ej < JAC_TOL, (er, ej)


def test_other_constants(api, orc, W):
    """Non-default physics and numerics reach the kernels (cleaning speeds, alpha, AUSM constants, delta)."""
    mi = small_meshes(W)["channel"]
    P = W.gem_state(mi.centroids()) + np.random.default_rng(3).uniform(-1e-2, 1e-2, (mi.n_cells, 18))
    ph = W.Physics(gamma_gas=1.4, mass_ratio=100.0, c=10.0, gamma_psi=1.3, chi_phi=0.7, rusanov_alpha=0.4)
    P[:, 9] = P[:, 8] / 100.0
    kw = dict(fd_delta=1e-5, venkat_K=0.5, lsq_weight_power=1.0, ausm_Kp=0.3, ausm_Ku=0.6, ausm_sigma=0.9,
              ausm_beta=0.1, ausm_Minf=[0.2, 0.05])
    er, ej, _ = compare_assembly(api, orc, mi, P, dt=2e-3, physics=ph, numerics_kw=kw)
    assert er < RES_TOL and ej < JAC_TOL, (er, ej)


def test_supersonic_and_upwind_branches(api, orc, W):
    """States with |M| > 1 and both flow directions exercise the other branches of the AUSM splits."""
    mi = small_meshes(W)["periodic7x5"]
    rng = np.random.default_rng(6)
    P = random_state(rng, mi.n_cells, vel=2.5)
    er, ej, _ = compare_assembly(api, orc, mi, P)
    assert er < RES_TOL and ej < JAC_TOL, (er, ej)


def test_reordered_assembly(api, orc, W):
    mi = small_meshes(W)["delaunay"]
    P = W.gem_state(mi.centroids()) + np.random.default_rng(4).uniform(-1e-3, 1e-3, (mi.n_cells, 18))
    er, ej, _ = compare_assembly(api, orc, mi, P, reorder="rcm")
    assert er < RES_TOL and ej < JAC_TOL, (er, ej)


def test_run_to_run_determinism_and_no_memset_needed(api, orc, W):
    """S21: two assemblies of the same input are bit-identical, whatever the output held before."""
    import torch
    mi = small_meshes(W)["delaunay"]
    g = api.Mesh.from_input(mi)
    ctx = api.Context()
    P = dev(W.gem_state(mi.centroids()))
    rhs1 = torch.full((g.n_cells, 18), float("nan"), dtype=torch.float64, device="cuda")
    vals1 = torch.full((g.nnzb, 18, 18), float("nan"), dtype=torch.float64, device="cuda")
    ctx.assemble(g, P, rhs=rhs1, vals=vals1)
    rhs2 = torch.full((g.n_cells, 18), 7.0, dtype=torch.float64, device="cuda")
    vals2 = torch.full((g.nnzb, 18, 18), 7.0, dtype=torch.float64, device="cuda")
    ctx.assemble(g, P, rhs=rhs2, vals=vals2)
    torch.cuda.synchronize()
    assert torch.equal(rhs1, rhs2) and torch.equal(vals1, vals2)
    assert torch.isfinite(vals1).all()
    # the residual-only call (its own kernel: no staging, no perturbed lanes) is deterministic as well and
    # meets the residual tolerance against the oracle; the two kernels' residuals agree to rounding
    rhs3, none = ctx.assemble(g, P, jacobian=False)
    rhs4, _ = ctx.assemble(g, P, jacobian=False)
    assert none is None and torch.equal(rhs3, rhs4)
    o = orc.OracleMesh.from_input(mi)
    ph_o = orc.physics_c()
    rhs_o, sc_o, _ = orc.assemble(o, ph_o, orc.default_numerics(ph_o), W.gem_state(mi.centroids()), jacobian=False)
    assert residual_error(rhs3.cpu().numpy(), rhs_o, sc_o) < RES_TOL
    assert residual_error(rhs3.cpu().numpy(), rhs1.cpu().numpy(), sc_o) < 1e-14
    assert ctx.launches_per_assemble == 2


def test_context_workspace_follows_the_mesh_not_its_address(api, orc, W):
    """One context used on mesh A, A destroyed, then on a larger mesh B (which the allocator may well place at A's
    address): the per-mesh workspace (least-squares coefficients, face-state buffer) must be rebuilt for B."""
    ctx = api.Context()
    for trial in range(4):                           # several rounds make an address reuse near certain
        a = W.split_quad_mesh(4 + trial, 4)
        ga = api.Mesh.from_input(a)
        ctx.assemble(ga, dev(W.wave_state(a.centroids(), seed=1)))
        ctx.check()
        ga.close()
        del ga
        b = W.delaunay_mesh(23, 17, *W.GEM_DOMAIN, jitter=0.3, seed=4 + trial, shuffle_cells=True)
        gb, ob = api.Mesh.from_input(b), orc.OracleMesh.from_input(b)
        P = W.gem_state(b.centroids()) + np.random.default_rng(trial).uniform(-1e-3, 1e-3, (b.n_cells, 18))
        rhs, vals = ctx.assemble(gb, dev(P))
        ctx.check()
        ph_o = orc.physics_c()
        rhs_o, sc_o, vals_o = orc.assemble(ob, ph_o, orc.default_numerics(ph_o), P)
        assert residual_error(rhs.cpu().numpy(), rhs_o, sc_o) < RES_TOL
        assert jacobian_error_blocks(vals.cpu().numpy(), vals_o, gb.get("bsr_rowptr")) < JAC_TOL
        gb.close()


def test_host_entry_point_matches_device_entry_point(api, W):
    import torch
    mi = small_meshes(W)["channel"]
    g = api.Mesh.from_input(mi)
    ctx = api.Context()
    P = W.gem_state(mi.centroids())
    Pn = W.perturb(P, 1, 1e-3)
    rhs_d, vals_d = ctx.assemble(g, dev(P), dev(Pn), dev(Pn), 1e-3)
    rhs_h = torch.empty((g.n_cells, 18), dtype=torch.float64).pin_memory()
    vals_h = torch.empty((g.nnzb, 18, 18), dtype=torch.float64).pin_memory()
    ctx.assemble_host(g, P, Pn, Pn, 1e-3, rhs_h, vals_h)
    assert torch.equal(rhs_h, rhs_d.cpu()) and torch.equal(vals_h, vals_d.cpu())


def test_nonphysical_state_is_reported(api, W):
    mi = small_meshes(W)["box"]
    g = api.Mesh.from_input(mi)
    ctx = api.Context()
    P = W.gem_state(mi.centroids())
    P[3, 16] = -1.0
    ctx.assemble(g, dev(P))
    with pytest.raises(api.TfaError) as e:
        ctx.check()
    assert e.value.code == -5
    ctx.assemble(g, dev(W.gem_state(mi.centroids())))
    ctx.check()     # the flag was cleared


def test_config2_first_and_last_of_ten_calls(api, orc, W):
    """BASELINE config 2 at its full size (256x256 quads split = 131 072 cells): 10 consecutive assemblies with
    the state perturbed by 1e-6 between calls; every row of the 1st and of the 10th call against the oracle."""
    w = W.make_workload("c2")
    assert w.mesh.n_cells == 131072
    g, o = api.Mesh.from_input(w.mesh), orc.OracleMesh.from_input(w.mesh)
    ctx = api.Context(w.physics)
    ph_o = orc.physics_c(w.physics)
    nu_o = orc.default_numerics(ph_o)
    rp = g.get("bsr_rowptr")
    P_prev2 = P_prev = P = w.state
    for call in range(10):
        rhs, vals = ctx.assemble(g, dev(P), dev(P_prev), dev(P_prev2), w.dt)
        if call in (0, 9):
            rhs_o, sc_o, vals_o = orc.assemble(o, ph_o, nu_o, P, P_prev, P_prev2, w.dt)
            er = residual_error(rhs.cpu().numpy(), rhs_o, sc_o)
            ej = jacobian_error_blocks(vals.cpu().numpy(), vals_o, rp)
            assert er < RES_TOL and ej < JAC_TOL, (call, er, ej)
        P_prev2, P_prev, P = P_prev, P, W.perturb(P, 100 + call, 1e-6)
    ctx.check()


SWEEP_CHUNK = 100_000


def sweep_every_row(api, orc, W, w, bc=None, flux_noise=0.0):
    """Assemble workload `w` on the GPU in the launch configuration bench.py times (device buffers, RCM where the
    workload says so) and compare EVERY row of rhs and of the BSR Jacobian with the oracle, swept in chunks of
    100 000 consecutive rows (oracle row-subset mode; the GPU's value array is sliced per chunk), so that every
    persistent CTA, both stages of the input pipeline and the tail tile are covered.  The pattern is compared
    bit-exactly over the whole mesh; every entry of the value array must have been written (NaN canary).
    bc(g, o) -> (tags, ghost) sets boundary rules on both sides.  A second, residual-only pass compares flux +
    source alone (term_mask = 3 on both sides) against their own scale, on the state plus U(-flux_noise,
    flux_noise).  Returns (er, er_flux_source_per_variable, ej)."""
    import torch
    g, o = api.Mesh.from_input(w.mesh), orc.OracleMesh.from_input(w.mesh)
    if w.reorder == "rcm":
        g.reorder("rcm")
        o.reorder("rcm")
    perm = g.get("perm")
    assert np.array_equal(perm, o.get("perm"))
    P = np.ascontiguousarray(w.state[perm])
    nc = g.n_cells
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    assert np.array_equal(rp, o.get("bsr_rowptr")) and np.array_equal(col, o.get("bsr_col"))
    ctx = api.Context(w.physics)
    ctx3 = api.Context(w.physics, api.default_numerics(ctx.physics, term_mask=3))
    if bc is not None:
        tags, ghost = bc(g, o)
        g.set_bc(tags)
        o.set_bc(tags, ghost)
        gd = None if ghost is None else dev(ghost)
        ctx.set_ghost_states(gd)
        ctx3.set_ghost_states(gd)
    Pd = dev(P)
    rhs = torch.full((nc, 18), float("nan"), dtype=torch.float64, device="cuda")
    vals = torch.full((g.nnzb, 18, 18), float("nan"), dtype=torch.float64, device="cuda")
    ctx.assemble(g, Pd, dt=w.dt, rhs=rhs, vals=vals)
    ctx.check()
    assert not bool(torch.isnan(vals).any()), "an entry of the BSR value array was not written"
    assert not bool(torch.isnan(rhs).any())
    # flux + source only, through the residual-only kernel, for the second residual bar
    P3 = P + np.random.default_rng(31).uniform(-flux_noise, flux_noise, P.shape) if flux_noise > 0 else P
    rhs3, _ = ctx3.assemble(g, dev(P3), dt=w.dt, jacobian=False)
    ctx3.check()
    rhs_h, rhs3_h = rhs.cpu().numpy(), rhs3.cpu().numpy()
    ph_o = orc.physics_c(w.physics)
    nu_o, nu3_o = orc.default_numerics(ph_o), orc.default_numerics(ph_o, term_mask=3)
    num = np.zeros(18); den = np.zeros(18); num3 = np.zeros(18); den3 = np.zeros(18)
    ej = 0.0
    for r0 in range(0, nc, SWEEP_CHUNK):
        r1 = min(nc, r0 + SWEEP_CHUNK)
        rows = np.arange(r0, r1, dtype=np.int32)
        rhs_o, sc_o, vals_o = orc.assemble(o, ph_o, nu_o, P, dt=w.dt, rows=rows)
        got = vals[int(rp[r0]):int(rp[r1])].cpu().numpy()
        ej = max(ej, jacobian_error_padded(got, vals_o, rp[r0:r1 + 1] - rp[r0]))
        num = np.maximum(num, np.abs(rhs_h[r0:r1] - rhs_o).max(axis=0))
        den = np.maximum(den, sc_o.max(axis=0))
        rhs3_o, sc3_o, _ = orc.assemble(o, ph_o, nu3_o, P3, dt=w.dt, rows=rows, jacobian=False)
        num3 = np.maximum(num3, np.abs(rhs3_h[r0:r1] - rhs3_o).max(axis=0))
        den3 = np.maximum(den3, sc3_o.max(axis=0))
    er = float((num / np.where(den > 0, den, 1.0)).max())
    e3 = num3 / np.where(den3 > 0, den3, 1.0)
    return er, e3, ej


@pytest.mark.parametrize("name", ["c2", "c3", "c4a", "c4b", "c5"])
def test_full_size_every_row(api, orc, W, name):
    """BASELINE configs 2-5 at their full sizes: every row against the oracle (sweep_every_row).  The residual is
    held to 1e-12 of the full sum-of-|terms| scale (S18), and -- with the BDF2 term masked out of both sides,
    term_mask = 3 -- to 1e-12 of the flux + source scale alone, which in these configurations (P^n = P^{n-1} = P)
    is up to 1e3 times smaller for the density and energy rows.

    The second bar is taken on the state plus U(-1e-3, 1e-3) (the noise config 2 carries anyway).  On the exactly
    smooth GEM state whole rows of the flux are differences of two nearly equal reconstructed face states and
    nothing else: the B_x, B_y rows (E_z = Psi = 0 leaves only the Rusanov dissipation c (B_R - B_L)) and the mass /
    energy rows (u_s.n = 0 leaves only the pressure-diffusion term ~ p_R - p_L).  The jump is O(h^2) of the state,
    so the rounding of the reconstruction (2^-53 |P|, different on the two sides: own-frame lanes against the
    oracle's L/R frame) is amplified by |P| / |P_R - P_L| = 1e4..1e7 relative to such a row's own scale (measured
    6e-12 on c3, 4e-11 on c5, 1e-9 on the Cartesian q1): the conditioning of those rows, not an error of either
    side, and already bounded by the first bar, which is 1e-11 of the un-cancelled flux magnitude c |P| Sigma."""
    er, e3, ej = sweep_every_row(api, orc, W, W.make_workload(name), flux_noise=0.0 if name == "c2" else 1e-3)
    assert er < RES_TOL and ej < JAC_TOL, (name, er, ej)
    assert e3.max() < RES_TOL, (name, e3)


def test_flux_sqrt_and_reciprocal_error_bound(api):
    """The Newton-refined square root and reciprocal of the AUSM flux kernel against the
    correctly rounded numpy results over 12 decades: within 1 ulp (the claim the Jacobian tolerance
    budget in DESIGN.md section 7 rests on)."""
    import torch
    rng = np.random.default_rng(5)
    x = np.concatenate([10.0 ** rng.uniform(-6, 6, 200000), [1.0, 4.0, 0.25, 2.0, 3.0, 1e-6, 1e6]])
    s, r = api.probe_math(torch.from_numpy(x).cuda())
    s, r = s.cpu().numpy(), r.cpu().numpy()
    es = np.abs(s - np.sqrt(x)) / np.spacing(np.sqrt(x))
    er = np.abs(r - 1.0 / x) / np.spacing(1.0 / x)
    assert es.max() <= 1.0 and er.max() <= 1.0, (es.max(), er.max())


def test_gpu_invariants_free_stream_and_telescoping(api, W):
    """north_star's first two oracle invariants, checked on the CUDA path itself (no oracle involved):
    a uniform state gives a zero convective residual on any mesh, boundary cells included (free-stream
    preservation, L85 consistency); on a periodic mesh the face fluxes telescope to a zero domain sum per
    equation.  Each cell evaluates its faces in its own outward frame, so the two sides of a
    face agree to rounding, not bit for bit: the sums are zero to rounding of the largest term."""
    import torch
    rng = np.random.default_rng(11)
    ctx = api.Context()
    nu = api.default_numerics(ctx.physics)
    nu.term_mask = 1                                   # convective fluxes only
    ctx.set_numerics(nu)
    # free stream: one random physical state everywhere, on a mesh with boundaries and on a Delaunay mesh
    for mi in (W.split_quad_mesh(9, 6, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False),
               W.delaunay_mesh(23, 17, *W.GEM_DOMAIN, jitter=0.3, seed=4, shuffle_cells=True)):
        g = api.Mesh.from_input(mi)
        P1 = random_state(rng, 1)
        P = np.repeat(P1, g.n_cells, axis=0)
        rhs, vals = ctx.assemble(g, dev(P))
        ctx.check()
        # scale of one face term: |F(U).n| Sigma <= c^2 |U| h
        scale = 400.0 * np.abs(P1).max() * np.sqrt(g.get("volume").max())
        assert float(rhs.abs().max()) <= 1e-12 * scale
    # telescoping: noisy wave on the periodic mesh of config 1
    w = W.make_workload("c1")
    g = api.Mesh.from_input(w.mesh)
    rhs, _ = ctx.assemble(g, dev(w.state), jacobian=False)
    rhs2, _ = ctx.assemble(g, dev(w.state))
    ctx.check()
    for r in (rhs, rhs2):
        tot = r.sum(dim=0).abs().cpu().numpy()
        mag = r.abs().sum(dim=0).cpu().numpy()
        assert (tot <= 1e-12 * np.maximum(mag, 1e-300) + 1e-13).all(), (tot, mag)


@pytest.mark.parametrize("theta,K", [(0.7, 1e9), (np.pi / 2, 1.0)])
def test_gpu_rotation_covariance_of_the_wave(api, W, theta, K):
    """north_star's fourth invariant (S19) on the CUDA path itself: rotate the mesh and the in-plane vector
    components; the rhs rows rotate with them, the Jacobian blocks are conjugated (up to the forward-difference
    truncation, the step sizes depending on the components).  Arbitrary angle with the limiter off, 90 degrees
    with it on."""
    mi = W.split_quad_mesh(6, 6)
    ctx = api.Context()
    nu = api.default_numerics(ctx.physics)
    nu.venkat_K = K
    ctx.set_numerics(nu)
    P = W.wave_state(mi.centroids(), seed=3)
    Q = rot18(theta)
    g0, g1 = api.Mesh.from_input(mi), api.Mesh.from_input(mi.rotated(theta))
    assert np.array_equal(g0.get("face_cells"), g1.get("face_cells"))
    rhs0, v0 = ctx.assemble(g0, dev(P))
    rhs1, v1 = ctx.assemble(g1, dev(P @ Q.T))
    ctx.check()
    rhs0, v0, rhs1, v1 = (t.cpu().numpy() for t in (rhs0, v0, rhs1, v1))
    # scale of the residual's terms: time term Omega 3U/(2 dt) dominates at dt = 1e-3
    scale = np.abs(v0).max() * np.abs(P).max()
    assert np.abs(rhs1 - rhs0 @ Q.T).max() < 1e-11 * scale
    J0rot = np.einsum("ab,nbc,dc->nad", Q, v0, Q)
    assert np.abs(v1 - J0rot).max() < 2e-5 * np.abs(v0).max()
