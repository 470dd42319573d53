"""The packed Jacobian (second option; include/tfa.h): 114 structural non-zeros per off-diagonal block.

CPU: the oracle-side packer (oracle/pack.py, numpy only) against hand-placed entries and its own inverse.  GPU:
tfa_assemble_packed against the oracle's packed Jacobian and, bit for bit, against tfa_assemble's BSR output; the
linear-solve entry points on the packed form against those on the BSR form.
"""
import numpy as np
import pytest

from conftest import random_state
from helpers import RES_TOL, JAC_TOL, residual_error, jacobian_error_blocks


def test_packer_layout_and_round_trip(orc, W):
    from oracle import pack
    assert pack.PACKED_BLOCK == 114
    mi = W.delaunay_mesh(7, 5, *W.GEM_DOMAIN, jitter=0.3, seed=11, shuffle_cells=True)
    o = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    P = W.gem_state(mi.centroids()) + np.random.default_rng(0).uniform(-1e-3, 1e-3, (o.n_cells, 18))
    _, _, vals = orc.assemble(o, ph, orc.default_numerics(ph), P)
    rp, col = o.get("bsr_rowptr"), o.get("bsr_col")
    diag, offd = pack.pack_bsr(vals, rp, col)
    assert diag.shape == (o.n_cells, 18, 18) and offd.shape == (o.nnzb - o.n_cells, 114)
    np.testing.assert_array_equal(pack.unpack_bsr(diag, offd, rp, col), vals)
    # hand-placed entries of the first off-diagonal block of row 5 (slot = rowptr[5] - 5 if the diagonal comes later)
    b = rp[5] if col[rp[5]] != 5 else rp[5] + 1
    slot = b - 5 - (1 if col[rp[5]] == 5 else 0)
    blk = vals[b]
    assert offd[slot, 8 * 3 + 6] == blk[3, 6]                   # fields: row E_x, column Psi
    assert offd[slot, 64 + 5 * 2 + 4] == blk[11, 16]            # ions: row momentum-y (11), column T_i (16)
    assert offd[slot, 64 + 25 + 5 * 0 + 3] == blk[9, 15]        # electrons: row mass (9), column u_e,z (15)
    assert offd[slot, 64 + 25 + 5 * 4 + 0] == blk[17, 9]        # electrons: row energy (17), column rho_e (9)
    bad = vals.copy()
    bad[b, 0, 8] = 1.0                                           # a field row must not see rho_i in an off-diagonal block
    with pytest.raises(AssertionError):
        pack.pack_bsr(bad, rp, col)


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


def cases(W):
    return {
        "triangles": (W.delaunay_mesh(23, 17, *W.GEM_DOMAIN, jitter=0.3, seed=4, shuffle_cells=True), False),
        "quads": (W.quad_mesh(9, 7), False),
        "mixed_bc": (W.quad_mesh(9, 6, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False, jitter=0.2, seed=4, tri_every=3), True),
    }


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["triangles", "quads", "mixed_bc"])
def test_packed_assembly_parity_and_solve(api, orc, W, case):
    import torch
    from oracle import pack
    mi, bc = cases(W)[case]
    g, o = api.Mesh.from_input(mi), orc.OracleMesh.from_input(mi)
    g.reorder("rcm")
    o.reorder("rcm")
    ctx = api.Context()
    rng = np.random.default_rng(2)
    if bc:
        tags = (np.arange(g.n_bfaces) % 3).astype(np.int32)
        ghost = random_state(rng, g.n_bfaces)
        g.set_bc(tags)
        o.set_bc(tags, ghost)
        ctx.set_ghost_states(dev(ghost))
    perm = g.get("perm")
    P = (W.gem_state(mi.centroids()) + rng.uniform(-1e-3, 1e-3, (g.n_cells, 18)))[perm]
    Pn = W.perturb(P, 3, 1e-4)
    nan = float("nan")
    diag = torch.full((g.n_cells, 18, 18), nan, dtype=torch.float64, device="cuda")
    offd = torch.full((g.nnzb - g.n_cells, 114), nan, dtype=torch.float64, device="cuda")
    rhs_p, _, _ = ctx.assemble_packed(g, dev(P), dev(Pn), dev(Pn), 0.02, diag=diag, offd=offd)
    rhs_b, vals_b = ctx.assemble(g, dev(P), dev(Pn), dev(Pn), 0.02)
    ctx.check()
    assert not bool(torch.isnan(diag).any()) and not bool(torch.isnan(offd).any())      # every entry written
    # same arithmetic: bit-identical to the BSR assembly, entry for entry
    assert torch.equal(rhs_p, rhs_b)
    assert torch.equal(api.packed_to_bsr(g, diag, offd), vals_b)
    # against the oracle, packed by the oracle-side packer
    ph_o = orc.physics_c()
    rhs_o, sc_o, vals_o = orc.assemble(o, ph_o, orc.default_numerics(ph_o), P, Pn, Pn, 0.02)
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    d_o, f_o = pack.pack_bsr(vals_o, rp, col)
    assert residual_error(rhs_p.cpu().numpy(), rhs_o, sc_o) < RES_TOL
    got = pack.unpack_bsr(diag.cpu().numpy(), offd.cpu().numpy(), rp, col)
    assert jacobian_error_blocks(got, vals_o, rp) < JAC_TOL
    rowmax = np.abs(vals_o).max()
    assert np.abs(diag.cpu().numpy() - d_o).max() < 1e-7 * rowmax and np.abs(offd.cpu().numpy() - f_o).max() < 1e-7 * rowmax
    # linear-solve entry points: packed against BSR
    x = dev(rng.normal(size=18 * g.n_cells))
    y_p, y_b = api.packed_spmv(g, diag, offd, x), api.bsr_spmv(g, vals_b, x)
    scale = float(api.bsr_spmv(g, vals_b.abs(), x.abs()).max())
    assert float((y_p - y_b).abs().max()) <= 1e-14 * scale
    dinv_p, dinv_b = ctx.block_jacobi_packed(g, diag), ctx.block_jacobi(g, vals_b)
    assert torch.equal(dinv_p, dinv_b)
    b = rhs_b.reshape(-1).contiguous()
    xp, itp, relp = ctx.gmres_packed(g, diag, offd, b, dinv=dinv_p, restart=30, max_iters=200, rtol=1e-10)
    xb, itb, relb = ctx.gmres(g, vals_b, b, dinv=dinv_b, restart=30, max_iters=200, rtol=1e-10)
    assert relp <= 1e-10 and abs(itp - itb) <= 1
    assert float((xp - xb).abs().max()) <= 1e-7 * float(xb.abs().max())
    # mixed precision (tfa_gmres_packed_f32): Krylov cycles on FP32 copies, restarts and the reported residual in
    # FP64 -- the same tolerance is reached, and the residual it reports is the true FP64 one
    d32, o32 = api.packed_to_f32(g, diag, offd)
    assert o32.shape[1] == 116 and float(o32[:, 114:].abs().max()) == 0.0
    assert torch.equal(d32, diag.to(torch.float32)) and torch.equal(o32[:, :114], offd.to(torch.float32))
    dinv32 = api.to_f32(dinv_p)
    for tol in (1e-6, 1e-10):
        xm, itm, relm = ctx.gmres_packed_f32(g, diag, offd, d32, o32, b, dinv32=dinv32, restart=30, max_iters=200, rtol=tol)
        true_rel = float((b - api.bsr_spmv(g, vals_b, xm)).norm() / b.norm())
        assert relm <= tol and abs(true_rel - relm) <= 1e-3 * relm + 1e-15, (tol, relm, true_rel)
        x64, it64, _ = ctx.gmres_packed(g, diag, offd, b, dinv=dinv_p, restart=30, max_iters=200, rtol=tol)
        assert itm <= it64 + max(3, it64 // 5), (tol, itm, it64)
    assert float((xm - xb).abs().max()) <= 1e-7 * float(xb.abs().max())
    xu, itu, relu = ctx.gmres_packed_f32(g, diag, offd, d32, o32, b, restart=30, max_iters=600, rtol=1e-6)   # no preconditioner
    assert relu <= 1e-6
    ctx.check()


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [None, (1, 1), (3, 3)])
def test_mixed_precision_solve_on_tiny_meshes(api, W, shape):
    """tfa_gmres_packed_f32 at the sizes where its layout rules bite: one cell (no off-diagonal block at all, n = 18
    is not a multiple of four: the FP32 basis has a padded stride and a two-entry tail), two and eighteen cells;
    restart lengths 1 and 30.  The check is the direct dense solution."""
    import torch
    if shape is None:
        g = api.Mesh(np.array([[0.0, 0], [1, 0], [0, 1]]), np.array([[0, 1, 2]], dtype=np.int32))
        cen = np.array([[1 / 3, 1 / 3]])
    else:
        mi = W.split_quad_mesh(*shape, periodic_x=False, periodic_y=False)
        g = api.Mesh.from_input(mi)
        cen = mi.centroids()
    P = dev(W.wave_state(cen, seed=2))
    ctx = api.Context(W.Physics())
    rhs, diag, offd = ctx.assemble_packed(g, P, dt=0.05)
    ctx.check()
    A = api.packed_to_bsr(g, diag, offd).cpu().numpy()
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    n = 18 * g.n_cells
    D = np.zeros((n, n))
    for i in range(g.n_cells):
        for bk in range(rp[i], rp[i + 1]):
            D[18 * i:18 * i + 18, 18 * col[bk]:18 * col[bk] + 18] = A[bk]
    b = rhs.reshape(-1).contiguous()
    xd = np.linalg.solve(D, b.cpu().numpy())
    d32, o32 = api.packed_to_f32(g, diag, offd)
    dinv32 = api.to_f32(ctx.block_jacobi_packed(g, diag))
    x, it, rel = ctx.gmres_packed_f32(g, diag, offd, d32, o32, b, dinv32=dinv32, restart=30, max_iters=600, rtol=1e-11)
    assert rel <= 1e-11, (it, rel)
    assert np.abs(x.cpu().numpy() - xd).max() <= 1e-11 * np.linalg.cond(D) * np.abs(xd).max()
    # GMRES(1) may stagnate on a non-symmetric system (it minimises along one direction per cycle): what must hold
    # is that the shortest restart runs (workspace layout), never increases the residual, and agrees with the FP64
    # GMRES(1) on the same system
    x1, it1, rel1 = ctx.gmres_packed_f32(g, diag, offd, d32, o32, b, dinv32=dinv32, restart=1, max_iters=40, rtol=1e-11)
    x2, it2, rel2 = ctx.gmres_packed(g, diag, offd, b, dinv=ctx.block_jacobi_packed(g, diag), restart=1, max_iters=40,
                                     rtol=1e-11)
    if rel2 <= 1e-11:    # FP64 converged (one cell: the preconditioner is the inverse): the mixed solve needs at most
        assert rel1 <= 1e-11 and it1 <= 2 * it2 + 1, (it1, it2, rel1, rel2)      # one refinement cycle more per cycle
    else:
        assert rel1 <= 1.0 and it1 == it2 and abs(rel1 - rel2) <= 1e-5 * rel2, (it1, it2, rel1, rel2)
    ctx.check()


@pytest.mark.gpu
def test_packed_assembly_full_size_config4(api, orc, W):
    """BASELINE config 4 (1M cells, RCM): the packed output expanded on the device equals the BSR output bit for
    bit (which test_full_size_every_row compares with the oracle row by row); 5.33 GB instead of 10.36 GB."""
    import torch
    w = W.make_workload("c4b")
    g = api.Mesh.from_input(w.mesh)
    g.reorder("rcm")
    P = dev(w.state[g.get("perm")])
    ctx = api.Context(w.physics)
    rhs_p, diag, offd = ctx.assemble_packed(g, P, dt=w.dt)
    rhs_b, vals_b = ctx.assemble(g, P, dt=w.dt)
    ctx.check()
    assert torch.equal(rhs_p, rhs_b)
    vals_x = api.packed_to_bsr(g, diag, offd)
    assert torch.equal(vals_x, vals_b)
    assert diag.numel() * 8 + offd.numel() * 8 == 1_000_000 * 2592 + 2_997_000 * 912
