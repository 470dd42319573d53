"""Pins for the oracle's gradient/limiter, residual and Jacobian.

north_star's four checks: free-stream preservation, periodic telescoping, brute-force central
differences on <= 64 cells, rotation covariance of the wave — plus closed forms for the
reconstruction and the BDF2 term.
"""
import numpy as np
import pytest

from conftest import random_state, rot18
from helpers import bsr_to_dense

RNG = np.random.default_rng(99)


def meshes(W):
    return {
        "periodic": W.split_quad_mesh(5, 5),
        "channel": W.split_quad_mesh(6, 4, *W.GEM_DOMAIN, periodic_x=True, periodic_y=False),
        "delaunay": W.delaunay_mesh(7, 5, *W.GEM_DOMAIN, jitter=0.3, seed=11, shuffle_cells=True),  # 48 cells
    }


# ------------------------------------------------------------------------------------------
# reconstruction
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("p", [0.0, 1.0, 2.0])
def test_gradient_exact_for_linear_fields(orc, W, p):
    """L74: least squares reproduces any linear field on any mesh, for any weight (S12)."""
    mi = meshes(W)["delaunay"]
    m = orc.OracleMesh.from_input(mi)
    nu = orc.default_numerics(lsq_weight_power=p)
    a = RNG.uniform(-1, 1, 18)
    gx, gy = RNG.uniform(-1, 1, 18), RNG.uniform(-1, 1, 18)
    cen = mi.centroids()
    P = a + np.outer(cen[:, 0], gx) + np.outer(cen[:, 1], gy)
    grad, _ = orc.gradients(m, nu, P)
    np.testing.assert_allclose(grad[:, :, 0], np.broadcast_to(gx, (m.n_cells, 18)), atol=1e-12)
    np.testing.assert_allclose(grad[:, :, 1], np.broadcast_to(gy, (m.n_cells, 18)), atol=1e-12)


def test_gradient_periodic_linear_field_is_exact_across_the_seam(orc, W):
    """S9: displacements use per-cell corner coordinates, so a field that is linear in the
    unwrapped coordinate is reproduced in cells whose stencil crosses the periodic seam only if
    the *differences* are linear; use a periodic field and check against an independent
    minimum-image least squares instead."""
    mi = W.split_quad_mesh(6, 6)
    m = orc.OracleMesh.from_input(mi)
    nu = orc.default_numerics()
    cen = mi.centroids()
    P = np.tile(np.sin(2 * np.pi * cen[:, 0])[:, None] * np.cos(2 * np.pi * cen[:, 1])[:, None], (1, 18))
    grad, _ = orc.gradients(m, nu, P)
    sp, si = m.get("stencil_ptr"), m.get("stencil_idx")
    for i in range(m.n_cells):
        js = si[sp[i]:sp[i + 1]]
        d = cen[js] - cen[i]
        d -= np.round(d)                    # minimum image on the unit square
        w = 1.0 / (d ** 2).sum(axis=1)
        A = (d * w[:, None]).T @ d
        b = (d * w[:, None]).T @ (P[js, 0] - P[i, 0])
        np.testing.assert_allclose(grad[i, 0], np.linalg.solve(A, b), atol=1e-11)


def test_limiter_closed_forms(orc, W):
    mi = meshes(W)["delaunay"]
    m = orc.OracleMesh.from_input(mi)
    cen = mi.centroids()
    # constant field: phi = 1
    _, phi = orc.gradients(m, orc.default_numerics(), np.ones((m.n_cells, 18)) * 3.0)
    assert (phi == 1.0).all()
    # K -> infinity switches the limiter off
    P = random_state(RNG, m.n_cells)
    _, phi = orc.gradients(m, orc.default_numerics(venkat_K=1e9), P)
    assert phi.min() > 1.0 - 1e-12 and phi.max() <= 1.0
    # K = 0 on a linear field: textbook Venkatakrishnan function of r = Delta1/Delta2,
    # phi(r) = (r^2 + 2r)/(r^2 + r + 2), so r = 1 gives 0.75 (S13)
    g = np.array([0.8, -0.5])
    lin = cen @ g
    P = np.tile(lin[:, None], (1, 18))
    grad, phi = orc.gradients(m, orc.default_numerics(venkat_K=0.0), P)
    sp, si = m.get("stencil_ptr"), m.get("stencil_idx")
    hit = 0
    for i in range(m.n_cells):
        js = si[sp[i]:sp[i + 1]]
        umax, umin = max(lin[js].max(), lin[i]), min(lin[js].min(), lin[i])
        X = mi.cell_xy[i]
        expect = 1.0
        for k in range(3):
            d2 = (0.5 * (X[k] + X[(k + 1) % 3]) - cen[i]) @ g
            if d2 == 0:
                continue
            r = ((umax if d2 > 0 else umin) - lin[i]) / d2
            expect = min(expect, (r * r + 2 * r) / (r * r + r + 2))
        assert abs(phi[i, 0] - expect) < 1e-10
        hit += expect < 1.0
    assert hit > 0                       # the limiter was active somewhere
    assert abs((1 + 2) / (1 + 1 + 2) - 0.75) == 0
    assert (phi >= 0).all() and (phi <= 1).all()      # K = 0: phi = 0 at local extrema (r = 0)
    _, phi = orc.gradients(m, orc.default_numerics(), random_state(RNG, m.n_cells))
    assert (phi > 0).all() and (phi <= 1).all()       # K > 0: phi in (0, 1]


@pytest.mark.parametrize("K", [1.0, 0.3, 2.5])
def test_limiter_finite_K_closed_form_on_a_linear_field(orc, W, K):
    """Pins eps^2 = (K sqrt(Omega))^3 (L208, S13) at finite K.  On a linear field the
    least-squares gradient is the exact slope g, so every quantity of Venkatakrishnan's function is known in
    closed form: Delta2 = g . (x_f - x_i), Delta1 = (max or min over the cell and its vertex neighbours) - P_i,
        phi_f = (Delta1^2 + eps^2 + 2 Delta1 Delta2) / (Delta1^2 + 2 Delta2^2 + Delta1 Delta2 + eps^2),
    phi_i = min(1, min_f phi_f).  Omega comes from the shoelace formula here.  The slope is sized so that eps^2 and
    Delta^2 are comparable: another exponent (h^2), h = Omega instead of sqrt(Omega), or K outside the cube
    changes phi by far more than the tolerance (asserted below)."""
    mi = meshes(W)["delaunay"]
    m = orc.OracleMesh.from_input(mi)
    cen = mi.centroids()
    X = mi.cell_xy
    area = 0.5 * ((X[:, 1, 0] - X[:, 0, 0]) * (X[:, 2, 1] - X[:, 0, 1]) - (X[:, 1, 1] - X[:, 0, 1]) * (X[:, 2, 0] - X[:, 0, 0]))
    g = np.array([1.7, -1.1]) * K ** 1.5
    lin = cen @ g + 0.3
    grad, phi = orc.gradients(m, orc.default_numerics(venkat_K=K), np.tile(lin[:, None], (1, 18)))
    sp, si = m.get("stencil_ptr"), m.get("stencil_idx")

    def expected(i, eps2):
        js = si[sp[i]:sp[i + 1]]
        umax, umin = max(lin[js].max(), lin[i]), min(lin[js].min(), lin[i])
        out = 1.0
        for k in range(3):
            d2 = (0.5 * (X[i, k] + X[i, (k + 1) % 3]) - cen[i]) @ g
            if d2 == 0:
                continue
            d1 = (umax if d2 > 0 else umin) - lin[i]
            out = min(out, (d1 * d1 + eps2 + 2 * d1 * d2) / (d1 * d1 + 2 * d2 * d2 + d1 * d2 + eps2))
        return out

    exp = np.array([expected(i, (K * np.sqrt(area[i])) ** 3) for i in range(m.n_cells)])
    np.testing.assert_allclose(phi[:, 0], exp, rtol=0, atol=1e-11)
    np.testing.assert_allclose(phi, np.tile(exp[:, None], (1, 18)), rtol=0, atol=1e-11)
    assert (exp < 0.999).sum() >= 5                       # the limiter is active (hull cells: no neighbour beyond the face)
    # the plausible mistakes are far outside the tolerance
    for wrong in (lambda a: (K * np.sqrt(a)) ** 2, lambda a: (K * a) ** 3, lambda a: K * np.sqrt(a) ** 3 if K != 1.0
                  else (K * np.sqrt(a)) ** 3 * 1.5, lambda a: 0.0):
        bad = np.array([expected(i, wrong(area[i])) for i in range(m.n_cells)])
        assert np.abs(bad - exp).max() > 1e-3


# ------------------------------------------------------------------------------------------
# residual
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["periodic", "channel", "delaunay"])
def test_free_stream_preservation(orc, W, kind):
    """Uniform state => zero convective residual, in boundary cells too (north_star check 1)."""
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, term_mask=1)
    P = np.tile(random_state(RNG, 1), (m.n_cells, 1))
    rhs, scale, _ = orc.assemble(m, ph, nu, P, jacobian=False)
    assert (np.abs(rhs) <= 1e-13 * scale.max(axis=0)).all()
    assert scale.max() > 1.0            # the individual face fluxes are not small


@pytest.mark.parametrize("kind", ["periodic"])
def test_periodic_telescoping(orc, W, kind):
    """Face fluxes cancel pairwise: the domain sum of the convective residual vanishes (check 2)."""
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, term_mask=1)
    P = random_state(RNG, m.n_cells)
    rhs, scale, _ = orc.assemble(m, ph, nu, P, jacobian=False)
    assert (np.abs(rhs.sum(axis=0)) <= 1e-12 * scale.sum(axis=0)).all()
    assert np.abs(rhs).max() > 1e-3     # while the residual itself is not zero


def test_time_term_bdf2(orc, W):
    """Eq. 13: with only the time term, rhs = -Omega (3U - 4U^n + U^n-1)/(2 dt).  For U^k sampled
    from a quadratic in time the BDF2 formula is the exact derivative (second-order)."""
    mi = meshes(W)["delaunay"]
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, term_mask=4)
    P = random_state(RNG, m.n_cells)
    rhs, sc, _ = orc.assemble(m, ph, nu, P, P, P, dt=1e-3, jacobian=False)
    assert np.abs(rhs).max() <= 1e-15 * sc.max()       # 3U - 4U + U up to rounding of 3U
    # EM rows (U = P): P(t) = a + b t + c t^2 at t = 0, -dt, -2dt ; dP/dt(0) = b
    dt = 0.05
    a, b, c = P, random_state(RNG, m.n_cells), random_state(RNG, m.n_cells)
    Pn, Pnm1 = a - b * dt + c * dt ** 2, a - 2 * b * dt + 4 * c * dt ** 2
    rhs, _, _ = orc.assemble(m, ph, nu, P, Pn, Pnm1, dt=dt, jacobian=False)
    vol = m.get("volume")
    np.testing.assert_allclose(rhs[:, :8], -(vol[:, None] * b[:, :8]), rtol=0, atol=1e-12)
    # species rows through U(P), recomputed here
    U = lambda Q: np.stack([orc.cons(ph, q) for q in Q])
    exp = -(vol[:, None] * (3 * U(P) - 4 * U(Pn) + U(Pnm1)) / (2 * dt))
    np.testing.assert_allclose(rhs, exp, rtol=0, atol=1e-12 * np.abs(exp).max())


@pytest.mark.parametrize("theta,K", [(0.37, 1e9), (np.pi / 2, 1.0)])
def test_rotation_covariance_of_the_wave(orc, W, theta, K):
    """north_star check 4 / S19: rotate the mesh and the in-plane vector components; rhs rows
    rotate with them, Jacobian blocks are conjugated.  The component-wise limiter is covariant
    only for multiples of 90 degrees, so the arbitrary angle runs with the limiter off."""
    mi = W.split_quad_mesh(6, 6)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, venkat_K=K)
    P = W.wave_state(mi.centroids(), seed=3)
    Q = rot18(theta)
    m0 = orc.OracleMesh.from_input(mi)
    m1 = orc.OracleMesh.from_input(mi.rotated(theta))
    np.testing.assert_array_equal(m0.get("face_cells"), m1.get("face_cells"))
    rhs0, sc0, v0 = orc.assemble(m0, ph, nu, P)
    rhs1, sc1, v1 = orc.assemble(m1, ph, nu, P @ Q.T)
    tol = 1e-11 * sc0.max()
    assert np.abs(rhs1 - rhs0 @ Q.T).max() < tol
    # Jacobian: J1 = Q J0 Q^T up to the FD truncation (the step sizes depend on the components)
    J0rot = np.einsum("ab,nbc,dc->nad", Q, v0, Q)
    assert np.abs(v1 - J0rot).max() < 2e-5 * np.abs(v0).max()


# ------------------------------------------------------------------------------------------
# Jacobian
# ------------------------------------------------------------------------------------------
def brute_force_jacobian(orc, m, ph, nu, P, grad, phi, dt):
    """Central differences of the oracle's own residual with frozen gradient and limiter (S8)."""
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
            J[:, j * 18 + k] = -((rp - rm) / (2 * h)).reshape(-1)     # rhs = -R~
    return J


@pytest.mark.parametrize("kind", ["periodic", "delaunay"])
def test_jacobian_vs_brute_force(orc, W, kind):
    """north_star check 3: <= 64 cells, forward-difference blocks vs central-difference brute force."""
    mi = meshes(W)[kind]
    m = orc.OracleMesh.from_input(mi)
    assert m.n_cells <= 64
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    cen = mi.centroids()
    P = W.wave_state(cen, seed=5) if kind == "periodic" else W.gem_state(cen) + RNG.uniform(-1e-3, 1e-3, (m.n_cells, 18))
    dt = 1e-3
    grad, phi = orc.gradients(m, nu, P)
    rhs, scale, vals = orc.assemble(m, ph, nu, P, dt=dt)
    # the residual_frozen entry reproduces assemble's rhs when fed assemble's own gradients
    np.testing.assert_array_equal(orc.residual_frozen(m, ph, nu, P, grad, phi, P, P, dt), rhs)
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    A = bsr_to_dense(vals, rp, col)
    J = brute_force_jacobian(orc, m, ph, nu, P, grad, phi, dt)
    rowmax = np.abs(J).max(axis=1, keepdims=True)
    err = np.abs(A - J) / rowmax
    assert err.max() < 1e-5, err.max()
    # the Maxwell rows are linear in P: forward differences are exact up to rounding (S7)
    em = np.concatenate([np.arange(18 * i, 18 * i + 8) for i in range(m.n_cells)])
    assert err[em].max() < 1e-9, err[em].max()
    # sparsity (S8): brute force has nothing outside self + face neighbours
    mask = np.kron(bsr_to_dense(np.ones_like(vals), rp, col)[::18, ::18] > 0, np.ones((18, 18))) > 0
    assert np.abs(J[~mask]).max() == 0.0
    # S6: the time term puts +3 Omega/(2 dt) dU/dP on the diagonal
    vol = m.get("volume")
    for i in range(0, m.n_cells, 7):
        assert A[18 * i, 18 * i] > 0.9 * 1.5 * vol[i] / dt


def test_flux_jacobian_block_structure(orc, W):
    """Off-diagonal blocks couple EM<->EM, ion<->ion, electron<->electron only: the other
    210 entries are exactly 0.0 (identical inputs -> identical outputs -> zero difference)."""
    mi = meshes(W)["delaunay"]
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    P = W.gem_state(mi.centroids()) + RNG.uniform(-1e-3, 1e-3, (m.n_cells, 18))
    _, _, vals = orc.assemble(m, ph, nu, P)
    rp, col = m.get("bsr_rowptr"), m.get("bsr_col")
    grp = np.array([0] * 8 + [1, 2] + [1] * 3 + [2] * 3 + [1, 2])
    coupled = grp[:, None] == grp[None, :]
    assert coupled.sum() == 114
    for i in range(m.n_cells):
        for q in range(rp[i], rp[i + 1]):
            if col[q] != i:
                assert (vals[q][~coupled] == 0.0).all()
                assert np.abs(vals[q][coupled]).max() > 0


def test_newton_step_solves_the_linear_maxwell_subsystem(orc, W):
    """S6 sign convention: A dP = rhs with A = dR~/dP, rhs = -R~.  Without sources the Maxwell
    rows are linear and decoupled, so one Newton step on them zeroes their (frozen) residual."""
    mi = W.split_quad_mesh(4, 4)
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, term_mask=1 | 4)
    P = W.wave_state(mi.centroids(), seed=8, noise=1e-2)
    Pn = W.perturb(P, 1, 1e-2)
    dt = 5e-3
    grad, phi = orc.gradients(m, nu, P)
    rhs, scale, vals = orc.assemble(m, ph, nu, P, Pn, Pn, dt=dt)
    A = bsr_to_dense(vals, m.get("bsr_rowptr"), m.get("bsr_col"))
    em = np.concatenate([np.arange(18 * i, 18 * i + 8) for i in range(m.n_cells)])
    dP = np.zeros(18 * m.n_cells)
    dP[em] = np.linalg.solve(A[np.ix_(em, em)], rhs.reshape(-1)[em])
    P1 = P + dP.reshape(-1, 18)
    r1 = orc.residual_frozen(m, ph, nu, P1, grad, phi, Pn, Pn, dt)
    assert np.abs(rhs[:, :8]).max() > 1e-3
    assert np.abs(r1[:, :8]).max() < 1e-9 * scale[:, :8].max()


def test_residual_signs_against_the_pde(orc, W):
    """Sign and orientation pins for Eq. 7/8/13 (S6), against the PDE itself.

    (a) flux term: for fields linear in space the reconstruction is exact and continuous, the
        dissipation vanishes and the midpoint rule is exact, so the Maxwell rows of the
        convective residual equal Omega * div F from Eq. 2:  curl E + gamma^2 grad Psi, etc.
    (b) source term: if U^n, U^n-1 lie on the straight line U - k dt S, BDF2 returns exactly S and
        the (time + source) residual of the Maxwell rows vanishes: dU/dt = S.
    """
    mi = meshes(W)["delaunay"]
    m = orc.OracleMesh.from_input(mi)
    ph = orc.physics_c()
    ph.gamma_psi, ph.chi_phi = 1.3, 0.7
    c, gp, chi = ph.c, ph.gamma_psi, ph.chi_phi
    vol = m.get("volume")
    cen = mi.centroids()
    # (a)
    nu = orc.default_numerics(ph, term_mask=1, venkat_K=1e12)
    a0 = random_state(RNG, 1)[0]
    gx, gy = RNG.uniform(-0.02, 0.02, 18), RNG.uniform(-0.02, 0.02, 18)
    gx[8:], gy[8:] = 0.0, 0.0
    P = a0 + np.outer(cen[:, 0], gx) + np.outer(cen[:, 1], gy)
    rhs, scale, _ = orc.assemble(m, ph, nu, P, jacobian=False)
    dx = lambda v: gx[v]
    dy = lambda v: gy[v]
    Bx, By, Bz, Ex, Ey, Ez, Psi, Phi = range(8)
    div = np.array([
        dy(Ez) + gp ** 2 * dx(Psi),                       # (curl E)_x + gamma^2 dPsi/dx
        -dx(Ez) + gp ** 2 * dy(Psi),                      # (curl E)_y + gamma^2 dPsi/dy
        dx(Ey) - dy(Ex),                                  # (curl E)_z
        -c ** 2 * dy(Bz) + (chi * c) ** 2 * dx(Phi),      # -c^2 (curl B)_x + (chi c)^2 dPhi/dx
        c ** 2 * dx(Bz) + (chi * c) ** 2 * dy(Phi),
        -c ** 2 * (dx(By) - dy(Bx)),
        c ** 2 * (dx(Bx) + dy(By)),                       # c^2 div B
        dx(Ex) + dy(Ey),                                  # div E
    ])
    np.testing.assert_allclose(rhs[:, :8], -vol[:, None] * div[None, :], rtol=0, atol=1e-11 * scale.max())
    assert np.abs(vol[:, None] * div[None, :]).max() > 1e-6 * scale.max()
    # (b)
    nu = orc.default_numerics(ph, term_mask=2 | 4)
    P = random_state(RNG, m.n_cells)
    S = np.stack([orc.source(ph, p) for p in P])
    dt = 1e-3
    Pn, Pnm1 = P.copy(), P.copy()
    Pn[:, :8] -= dt * S[:, :8]
    Pnm1[:, :8] -= 2 * dt * S[:, :8]
    rhs, scale, _ = orc.assemble(m, ph, nu, P, Pn, Pnm1, dt=dt, jacobian=False)
    assert np.abs(S[:, 3:6]).max() > 1.0
    assert np.abs(rhs[:, :8]).max() < 1e-12 * scale[:, :8].max()
