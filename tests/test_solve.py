"""Linear-solve step: oracle pins (-m "not gpu") and GPU parity (-m gpu)."""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spl


def random_bsr(rng, n, extra=2, diag_boost=6.0):
    """Random 18x18-block matrix: diagonal blocks plus `extra` off-diagonal blocks per row, columns ascending."""
    rowptr, col = [0], []
    for i in range(n):
        others = rng.choice([j for j in range(n) if j != i], size=min(extra, n - 1), replace=False)
        cols = sorted(set([i] + [int(j) for j in others]))
        col += cols
        rowptr.append(len(col))
    rowptr, col = np.array(rowptr, dtype=np.int32), np.array(col, dtype=np.int32)
    vals = rng.normal(size=(len(col), 18, 18))
    for i in range(n):
        b = rowptr[i] + int(np.nonzero(col[rowptr[i]:rowptr[i + 1]] == i)[0][0])
        vals[b] += diag_boost * np.sqrt(18 * (extra + 1)) * np.eye(18)
    return vals, rowptr, col


# ---------------------------------------------------------------------------------------------------
# oracle pins
# ---------------------------------------------------------------------------------------------------
def test_oracle_gmres_equals_the_direct_solution():
    from oracle import solve
    rng = np.random.default_rng(1)
    vals, rp, col = random_bsr(rng, 12)
    A = solve.bsr_matrix(vals, rp, col)
    b = rng.normal(size=A.shape[0])
    xd = spl.spsolve(A.tocsc(), b)
    for dinv in (None, solve.block_jacobi(vals, rp, col)):
        x, it, rel, est = solve.gmres(A, b, dinv=dinv, restart=20, max_iters=400, rtol=1e-12)
        assert rel <= 1e-12 and np.abs(x - xd).max() <= 1e-9 * np.abs(xd).max()
        # the recurrence's last estimate agrees with the true residual
        assert abs(est[-1] - rel) <= 1e-3 * rel + 1e-14


def test_oracle_full_gmres_terminates_in_n_steps():
    """Without restart GMRES is exact after at most n steps (n = 36 here)."""
    from oracle import solve
    rng = np.random.default_rng(2)
    vals, rp, col = random_bsr(rng, 2, extra=1, diag_boost=0.3)     # not diagonally dominant
    A = solve.bsr_matrix(vals, rp, col)
    b = rng.normal(size=36)
    x, it, rel, est = solve.gmres(A, b, restart=36, max_iters=36, rtol=1e-13)
    assert it <= 36 and rel <= 1e-10
    assert np.abs(A @ x - b).max() <= 1e-9 * np.abs(b).max()


def test_oracle_block_jacobi_makes_identity_on_block_diagonal_matrices():
    from oracle import solve
    rng = np.random.default_rng(3)
    vals, rp, col = random_bsr(rng, 6, extra=0)
    dinv = solve.block_jacobi(vals, rp, col)
    A = solve.bsr_matrix(vals, rp, col)
    v = rng.normal(size=A.shape[0])
    assert np.abs(A @ solve.apply_block_diag(dinv, v) - v).max() <= 1e-12 * np.abs(v).max()
    x, it, rel, _ = solve.gmres(A, v, dinv=dinv, restart=5, max_iters=5, rtol=1e-12)
    assert it == 1 and rel <= 1e-12                    # exact preconditioner: one iteration


# ---------------------------------------------------------------------------------------------------
# GPU parity
# ---------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def system(W):
    """A real system: BDF2 Jacobian and rhs of the noisy wave (config-1 recipe) on 24 x 12 split quads."""
    import torch
    from paper_1809_02532_b200 import api, build
    build.build()
    m = W.split_quad_mesh(24, 12)
    g = api.Mesh.from_input(m)
    g.reorder("rcm")
    P = np.ascontiguousarray(W.wave_state(m.centroids(), seed=3)[g.get("perm")])
    ctx = api.Context(W.Physics())
    rhs, vals = ctx.assemble(g, torch.from_numpy(P).cuda(), dt=1e-2)
    ctx.check()
    return api, ctx, g, rhs, vals


@pytest.mark.gpu
def test_spmv_parity(system):
    import torch
    from oracle import solve
    api, ctx, g, rhs, vals = system
    rng = np.random.default_rng(4)
    x = rng.normal(size=18 * g.n_cells)
    y = api.bsr_spmv(g, vals, torch.from_numpy(x).cuda()).cpu().numpy()
    A = solve.bsr_matrix(vals.cpu().numpy(), g.get("bsr_rowptr"), g.get("bsr_col"))
    ref = A @ x
    scale = abs(A) @ np.abs(x)                        # sum of |terms| per row
    assert (np.abs(y - ref) <= 1e-14 * scale * 80).all()


@pytest.mark.gpu
def test_block_jacobi_parity_and_singular_block(system):
    import torch
    from oracle import solve
    api, ctx, g, rhs, vals = system
    dinv = ctx.block_jacobi(g, vals).cpu().numpy()
    ctx.check()
    ref = solve.block_jacobi(vals.cpu().numpy(), g.get("bsr_rowptr"), g.get("bsr_col"))
    err = np.abs(dinv - ref).max(axis=(1, 2)) / np.abs(ref).max(axis=(1, 2))
    assert err.max() <= 1e-10, err.max()
    bad = vals.clone()
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    b = rp[5] + int(np.nonzero(col[rp[5]:rp[6]] == 5)[0][0])
    bad[b] = 0.0
    ctx.block_jacobi(g, bad)
    with pytest.raises(api.TfaError) as e:
        ctx.check()
    assert e.value.code == -6
    ctx.check()


@pytest.mark.gpu
def test_block_jacobi_needs_its_pivoting(system):
    """Diagonal blocks the assembled Jacobian never produces: dense random blocks with a zero diagonal,
    signed permutation matrices, rows of very different scale.  Every pivot step moves (implicitly) a row, so
    the permutation bookkeeping of the kernel is exercised; A A^-1 = I is the check, numpy's inverse the oracle."""
    import torch
    api, ctx, g, rhs, vals = system
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    n = g.n_cells
    diag = np.array([rp[i] + int(np.nonzero(col[rp[i]:rp[i + 1]] == i)[0][0]) for i in range(n)])
    rng = np.random.default_rng(7)
    blocks = rng.standard_normal((n, 18, 18))
    blocks[:, np.arange(18), np.arange(18)] = 0.0                       # no usable diagonal pivot
    for i in range(0, n, 3):                                            # signed, scaled permutations
        blocks[i] = 0.0
        blocks[i, np.arange(18), rng.permutation(18)] = rng.choice([-1.0, 1.0], 18) * 10.0 ** rng.integers(-6, 7, 18)
    blocks[1::3] *= (10.0 ** rng.integers(-8, 9, (len(blocks[1::3]), 18)))[:, :, None]   # badly scaled rows
    v = vals.clone()
    v[torch.from_numpy(diag).cuda()] = torch.from_numpy(blocks).cuda()
    dinv = ctx.block_jacobi(g, v).cpu().numpy()
    ctx.check()
    ref = np.linalg.inv(blocks)
    prod = np.einsum("nij,njk->nik", blocks, dinv)
    cond = np.linalg.cond(blocks, 1)
    assert (np.abs(prod - np.eye(18)).max(axis=(1, 2)) <= 1e-13 * cond).all()
    assert (np.abs(dinv - ref).max(axis=(1, 2)) <= 1e-13 * cond * np.abs(ref).max(axis=(1, 2))).all()
    # the inverse of a scaled signed permutation has the transposed pattern, exactly
    assert np.array_equal(dinv[0] != 0.0, (blocks[0] != 0.0).T)
    # a NaN in a diagonal block is reported, not propagated silently
    v[int(diag[2]), 4, 4] = float("nan")
    ctx.block_jacobi(g, v)
    with pytest.raises(api.TfaError) as e:
        ctx.check()
    assert e.value.code == -6


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [None, (1, 1), (1, 2), (1, 3), (2, 5), (3, 7), (10, 10)])
def test_block_jacobi_group_tails(W, shape):
    """The kernel works on five blocks per warp (six lanes each, lanes 30 and 31 idle) and twenty per CTA: cell
    counts of 1, 2, 4, 6, 20, 42 and 200 leave groups, warps and CTAs partly empty.  Random diagonal blocks with one
    singular block among them (zero inverse + count, its neighbours in the same warp untouched); numpy's inverse
    is the check."""
    import torch
    from paper_1809_02532_b200 import api, build
    build.build()
    if shape is None:
        g = api.Mesh(np.array([[0.0, 0], [1, 0], [0, 1]]), np.array([[0, 1, 2]], dtype=np.int32))
    else:
        g = api.Mesh.from_input(W.split_quad_mesh(*shape, periodic_x=False, periodic_y=False))
    n = g.n_cells
    rng = np.random.default_rng(n)
    blocks = rng.standard_normal((n, 18, 18)) + 3.0 * np.eye(18)
    bad = n // 2 if n > 1 else None
    if bad is not None:
        blocks[bad, :, 5] = 0.0                       # a zero column: singular
    ctx = api.Context(W.Physics())
    dinv = ctx.block_jacobi_packed(g, torch.from_numpy(blocks).cuda()).cpu().numpy()
    good = np.ones(n, dtype=bool)
    if bad is not None:
        good[bad] = False
        assert not dinv[bad].any()
        with pytest.raises(api.TfaError) as e:
            ctx.check()
        assert e.value.code == -6
    else:
        ctx.check()
    ref = np.linalg.inv(blocks[good])
    cond = np.linalg.cond(blocks[good], 1)
    assert (np.abs(dinv[good] - ref).max(axis=(1, 2)) <= 1e-13 * cond * np.abs(ref).max(axis=(1, 2))).all()
    # the same blocks through the BSR entry point (diagonal block found through the block map)
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    vals = torch.zeros((g.nnzb, 18, 18), dtype=torch.float64, device="cuda")
    diag = np.array([rp[i] + int(np.nonzero(col[rp[i]:rp[i + 1]] == i)[0][0]) for i in range(n)])
    vals[torch.from_numpy(diag).cuda()] = torch.from_numpy(blocks).cuda()
    ctx2 = api.Context(W.Physics())
    assert np.array_equal(ctx2.block_jacobi(g, vals).cpu().numpy(), dinv)


@pytest.mark.gpu
@pytest.mark.parametrize("precond", [True, False])
def test_gmres_parity(system, precond):
    import torch
    from oracle import solve
    api, ctx, g, rhs, vals = system
    rp, col = g.get("bsr_rowptr"), g.get("bsr_col")
    A = solve.bsr_matrix(vals.cpu().numpy(), rp, col)
    b = rhs.cpu().numpy().ravel()
    lu = spl.splu(A.tocsc())
    xd = lu.solve(b)                                  # external pin: the direct solution
    inv_op = spl.LinearOperator(A.shape, matvec=lu.solve, rmatvec=lambda v: lu.solve(v, "T"))
    cond1 = spl.onenormest(A) * spl.onenormest(inv_op)
    rtol = 1e-10 if precond else 1e-6          # the unpreconditioned iteration is slow on this stiff system
    dinv_o = solve.block_jacobi(vals.cpu().numpy(), rp, col) if precond else None
    xo, it_o, rel_o, _ = solve.gmres(A, b, dinv=dinv_o, restart=30, max_iters=600, rtol=rtol)
    dinv = ctx.block_jacobi(g, vals) if precond else None
    x, it, rel = ctx.gmres(g, vals, rhs.reshape(-1).contiguous(), dinv=dinv, restart=30, max_iters=600, rtol=rtol)
    ctx.check()
    x = x.cpu().numpy()
    assert rel <= rtol and rel_o <= rtol, (rel, rel_o, it, it_o)
    # the reported residual is the true one
    assert abs(np.linalg.norm(b - A @ x) / np.linalg.norm(b) - rel) <= 1e-3 * rel + 1e-15
    # both iterations stop within the tolerance of the direct solution; counts differ at most by the
    # rounding of the stopping test (classical Gram-Schmidt twice here, modified Gram-Schmidt in the oracle)
    tol = 10 * rtol * cond1
    assert np.abs(x - xd).max() <= tol * np.abs(xd).max() and np.abs(xo - xd).max() <= tol * np.abs(xd).max()
    assert abs(it - it_o) <= max(2, it_o // 20), (it, it_o)
    if precond:
        assert it < 600


@pytest.mark.gpu
def test_gmres_edge_cases(system):
    import torch
    api, ctx, g, rhs, vals = system
    n = 18 * g.n_cells
    z = torch.zeros(n, dtype=torch.float64, device="cuda")
    x, it, rel = ctx.gmres(g, vals, z, x=torch.ones_like(z))          # b = 0  ->  x = 0
    assert it == 0 and float(x.abs().max()) == 0.0
    b = rhs.reshape(-1).contiguous()
    x, it, rel = ctx.gmres(g, vals, b, max_iters=0)                    # no iterations allowed
    assert it == 0 and rel == pytest.approx(1.0)
    with pytest.raises(api.TfaError):
        ctx.gmres(g, vals, b, restart=0)
    # starting from the solution: nothing to do
    xs, it1, rel1 = ctx.gmres(g, vals, b, dinv=ctx.block_jacobi(g, vals), rtol=1e-9)
    x2, it2, rel2 = ctx.gmres(g, vals, b, x=xs.clone(), dinv=ctx.block_jacobi(g, vals), rtol=1e-9)
    assert it2 == 0 and rel2 == pytest.approx(rel1)
    # singular operator (A = 0): the Hessenberg column vanishes -> TFA_ESINGULAR, x left at the initial guess
    x0 = torch.full((n,), 0.5, dtype=torch.float64, device="cuda")
    with pytest.raises(api.TfaError) as e:
        ctx.gmres(g, torch.zeros_like(vals), b, x=x0)
    assert e.value.code == -6 and float((x0 - 0.5).abs().max()) == 0.0
    # NaN in the matrix: reported, not returned as success
    bad = vals.clone()
    bad[0, 0, 0] = float("nan")
    with pytest.raises(api.TfaError) as e:
        ctx.gmres(g, bad, b)
    assert e.value.code == -6


# ---------------------------------------------------------------------------------------------------
# matrix-free operator
# ---------------------------------------------------------------------------------------------------
@pytest.mark.gpu
def test_jfnk_solve_with_kernel_timing_enabled(W):
    """A matrix-free solve applies the operator more often than the timing ring of tfa_assemble has slots (64);
    the operator's evaluations are untimed, so the solve must not fail on it."""
    import torch
    from paper_1809_02532_b200 import api
    m = W.split_quad_mesh(12, 8)
    P = torch.from_numpy(W.wave_state(m.centroids(), seed=7)).cuda()
    g = api.Mesh.from_input(m)
    ctx = api.Context()
    rhs, vals = ctx.assemble(g, P, dt=0.05)
    dinv = ctx.block_jacobi(g, vals)
    ctx.timing_enable(True)
    x, it, rel = ctx.gmres_jfnk(g, P, rhs.reshape(-1).contiguous(), dt=0.05, restart=20, max_iters=90, rtol=1e-30)
    assert it == 90                                   # 90 operator applications > 64 ring slots
    ctx.assemble(g, P, dt=0.05)
    assert ctx.timing_read()[2] == 1                  # only the explicit assembly was timed
    ctx.timing_enable(False)
    ctx.check()


def _wave_case(W, orc):
    m = W.split_quad_mesh(12, 8)
    P = W.wave_state(m.centroids(), seed=7)
    o = orc.OracleMesh.from_input(m)
    pc = orc.physics_c(W.Physics())
    nu = orc.default_numerics(pc)
    return m, P, o, pc, nu


def test_oracle_jvp_against_central_differences(orc, W):
    """Forward difference of the oracle residual against the central one with a larger step (brute force)."""
    from oracle import solve
    m, P, o, pc, nu = _wave_case(W, orc)
    rhs_fn = lambda Q: orc.assemble(o, pc, nu, Q, P, P, 1e-2, jacobian=False)[0]
    rng = np.random.default_rng(8)
    v = rng.normal(size=P.shape) * np.maximum(np.abs(P), 1e-2)
    fwd = solve.jvp(rhs_fn, P, v, 1e-7)
    h = 1e-5
    cen = -(rhs_fn(P + h * v) - rhs_fn(P - h * v)) / (2 * h)
    assert np.abs(fwd - cen).max() <= 2e-4 * np.abs(cen).max()


@pytest.mark.gpu
def test_jvp_parity(W, orc):
    import torch
    from oracle import solve
    from paper_1809_02532_b200 import api, build
    build.build()
    m, P, o, pc, nu = _wave_case(W, orc)
    g = api.Mesh.from_input(m)
    ctx = api.Context(W.Physics())
    rng = np.random.default_rng(9)
    v = rng.normal(size=P.shape) * np.maximum(np.abs(P), 1e-2)
    eps = 1e-6
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = ctx.jvp(g, dev(P), dev(v).reshape(-1), dt=1e-2, eps=eps).cpu().numpy().reshape(-1, 18)
    ctx.check()
    rhs_fn = lambda Q: orc.assemble(o, pc, nu, Q, P, P, 1e-2, jacobian=False)[0]
    ref = solve.jvp(rhs_fn, P, v, eps)
    scale = orc.assemble(o, pc, nu, P, P, P, 1e-2, jacobian=False)[1]      # sum of |terms| of the residual
    # two residuals, each within 1e-12 of its scale (S18; measured 4e-16), differenced and divided by eps
    assert (np.abs(out - ref).max(axis=0) <= 2e-14 / eps * scale.max(axis=0)).all()
    # automatic step: same operator up to the O(eps) truncation of the forward difference
    auto = ctx.jvp(g, dev(P), dev(v).reshape(-1), dt=1e-2).cpu().numpy().reshape(-1, 18)
    assert np.abs(auto - ref).max() <= 1e-3 * np.abs(ref).max()


@pytest.mark.gpu
def test_gmres_jfnk_solves_the_newton_system(W, orc):
    """Matrix-free GMRES (block-Jacobi from the assembled, frozen Jacobian as preconditioner) against the same
    solve done on the host with the oracle's matrix-free operator; and against the assembled-matrix solve, from
    which it differs only by the frozen-gradient terms."""
    import torch
    from oracle import solve
    from paper_1809_02532_b200 import api, build
    build.build()
    m, P, o, pc, nu = _wave_case(W, orc)
    g = api.Mesh.from_input(m)
    ctx = api.Context(W.Physics())
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Pd = dev(P)
    rhs, vals = ctx.assemble(g, Pd, dt=1e-2)
    dinv = ctx.block_jacobi(g, vals)
    b = rhs.reshape(-1).contiguous()
    # (the forward difference leaves operator noise of about 1e-9 relative: 1e-6 is a reachable tolerance)
    x, it, rel = ctx.gmres_jfnk(g, Pd, b, dt=1e-2, dinv=dinv, restart=40, max_iters=400, rtol=1e-6)
    ctx.check()
    assert rel <= 1e-6 and it < 400
    # the solution satisfies the matrix-free system as the oracle sees it
    rhs_fn = lambda Q: orc.assemble(o, pc, nu, Q, P, P, 1e-2, jacobian=False)[0]
    xs = x.cpu().numpy().reshape(-1, 18)
    eps = 1e-7 * (1.0 + np.sqrt((P ** 2).mean())) / np.sqrt((xs ** 2).mean())
    r = rhs.cpu().numpy() - solve.jvp(rhs_fn, P, xs, eps)
    assert np.linalg.norm(r) <= 1e-4 * np.linalg.norm(rhs.cpu().numpy())
    # and is close to the frozen-Jacobian solution
    xa, _, _ = ctx.gmres(g, vals, b, dinv=dinv, restart=40, max_iters=400, rtol=1e-8)
    assert float((x - xa).norm() / xa.norm()) < 0.5
