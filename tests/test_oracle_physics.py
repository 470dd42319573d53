"""Pins for the oracle's point-wise physics: Maxwell flux, AUSM+-up, source, U(P).

Each check compares the oracle with something fixed by the paper's equations or by mathematics and
computed here by a different route (numpy cross products, numpy eig, finite differences) — never by
re-calling the oracle's own formula.
"""
import numpy as np
import pytest

from conftest import random_state, rot18

RNG = np.random.default_rng(1234)


def normals(n):
    th = RNG.uniform(0, 2 * np.pi, n)
    return np.cos(th), np.sin(th)


# ------------------------------------------------------------------------------------------
# Maxwell + divergence cleaning  (Eq. 2, L91 Eq. 9)
# ------------------------------------------------------------------------------------------
def maxwell_Fn(U, n3, c, gpsi, chi):
    """F.n of Eq. 2 written with numpy cross products (n3 = (nx, ny, 0))."""
    B, E, Psi, Phi = U[0:3], U[3:6], U[6], U[7]
    return np.concatenate([np.cross(n3, E) + gpsi ** 2 * Psi * n3,
                           -c ** 2 * np.cross(n3, B) + (chi * c) ** 2 * Phi * n3,
                           [c ** 2 * np.dot(B, n3)], [np.dot(E, n3)]])


def maxwell_An(n3, c, gpsi, chi):
    return np.stack([maxwell_Fn(e, n3, c, gpsi, chi) for e in np.eye(8)], axis=1)


@pytest.mark.parametrize("gpsi,chi,alpha", [(1.0, 1.0, 1.0), (1.3, 0.7, 1.0), (1.3, 0.7, 0.35)])
def test_maxwell_flux(orc, gpsi, chi, alpha):
    ph = orc.physics_c()
    ph.gamma_psi, ph.chi_phi, ph.rusanov_alpha = gpsi, chi, alpha
    c = ph.c
    for nx, ny in zip(*normals(6)):
        n3 = np.array([nx, ny, 0.0])
        A = maxwell_An(n3, c, gpsi, chi)
        # S1: eigenvalues of A_n are +-c (x2), +-gamma_psi c, +-chi c
        lam = np.sort(np.linalg.eigvals(A).real)
        np.testing.assert_allclose(lam, np.sort([-c, -c, c, c, -gpsi * c, gpsi * c, -chi * c, chi * c]),
                                   rtol=1e-10)
        UL, UR = RNG.uniform(-1, 1, 8), RNG.uniform(-1, 1, 8)
        # consistency (L85)
        np.testing.assert_allclose(orc.flux_maxwell(ph, UL, UL, nx, ny), A @ UL, rtol=0, atol=1e-12 * c * c)
        # Eq. 9 with |A_n| = R |Lambda| R^-1 from numpy eig (S3)
        w, R = np.linalg.eig(A)
        absA = (R @ np.diag(np.abs(w)) @ np.linalg.inv(R)).real
        H = 0.5 * (A @ UL + A @ UR) - 0.5 * alpha * absA @ (UR - UL)
        np.testing.assert_allclose(orc.flux_maxwell(ph, UL, UR, nx, ny), H, rtol=0, atol=1e-10 * c * c)
        if alpha == 1.0:   # exact upwind flux A+ U_L + A- U_R
            Ap = (R @ np.diag(np.maximum(w.real, 0)) @ np.linalg.inv(R)).real
            Am = (R @ np.diag(np.minimum(w.real, 0)) @ np.linalg.inv(R)).real
            np.testing.assert_allclose(orc.flux_maxwell(ph, UL, UR, nx, ny), Ap @ UL + Am @ UR, atol=1e-10 * c * c)
        # conservation: H(L,R,n) = -H(R,L,-n)
        np.testing.assert_allclose(orc.flux_maxwell(ph, UL, UR, nx, ny), -orc.flux_maxwell(ph, UR, UL, -nx, -ny),
                                   rtol=0, atol=1e-12 * c * c)


def test_maxwell_plane_wave_sign(orc):
    """S2: a vacuum plane wave travelling along +x (E_y = c B_z) is an eigenvector with speed +c:
    A_n U = c U, so Faraday/Ampere signs are dB/dt + curl E = 0, dE/dt - c^2 curl B = 0."""
    ph = orc.physics_c()
    c = ph.c
    U = np.zeros(8)
    U[2], U[4] = 1.0, c           # Bz = 1, Ey = c
    np.testing.assert_allclose(orc.flux_maxwell(ph, U, U, 1.0, 0.0), c * U, atol=1e-12 * c * c)


# ------------------------------------------------------------------------------------------
# AUSM+-up  (Eq. 10; Liou 2006 = ref. [30])
# ------------------------------------------------------------------------------------------
def euler_Fn(P5, nx, ny, Rs, g):
    """F.n of Eq. 5 (L63): (rho un, rho un u + p n, rho un H), p = rho R T, H = eps + p/rho (L70)."""
    rho, u, T = P5[0], P5[1:4], P5[4]
    un = u[0] * nx + u[1] * ny
    p = rho * Rs * T
    eps = Rs / (g - 1) * T + 0.5 * np.dot(u, u)
    Ht = eps + p / rho
    return np.array([rho * un, rho * un * u[0] + p * nx, rho * un * u[1] + p * ny, rho * un * u[2], rho * un * Ht])


def species_state(s, mach=0.3, mass_ratio=25.0):
    Rs = 1.0 if s == 0 else mass_ratio
    rho = RNG.uniform(0.5, 1.5) / (1.0 if s == 0 else mass_ratio)
    T = RNG.uniform(0.3, 0.8)
    a = np.sqrt(5.0 / 3.0 * Rs * T)
    u = RNG.uniform(-1, 1, 3) * mach * a
    return np.array([rho, u[0], u[1], u[2], T])


@pytest.mark.parametrize("s", [0, 1])
@pytest.mark.parametrize("mach", [0.01, 0.4, 2.5])
@pytest.mark.parametrize("minf", [0.1, 1.0])
def test_ausm_consistency_antisymmetry(orc, s, mach, minf):
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, ausm_Minf=[minf, minf])
    Rs = 1.0 if s == 0 else ph.mass_ratio
    for nx, ny in zip(*normals(5)):
        L, R = species_state(s, mach), species_state(s, mach)
        F = euler_Fn(L, nx, ny, Rs, ph.gamma_gas)
        scale = np.abs(F).max() + L[0] * Rs * L[4]
        # consistency H(U,U,n) = F(U).n (L85)
        np.testing.assert_allclose(orc.flux_ausm(ph, nu, s, L, L, nx, ny), F, rtol=0, atol=4e-15 * scale)
        # conservation H(L,R,n) = -H(R,L,-n), exactly
        np.testing.assert_array_equal(orc.flux_ausm(ph, nu, s, L, R, nx, ny),
                                      -orc.flux_ausm(ph, nu, s, R, L, -nx, -ny))


@pytest.mark.parametrize("s", [0, 1])
def test_ausm_supersonic_upwinding(orc, s):
    """M_L, M_R >= 1  =>  H = F(U_L).n ;  M_L, M_R <= -1  =>  H = F(U_R).n  (pure upwinding)."""
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    Rs = 1.0 if s == 0 else ph.mass_ratio
    nx, ny = 0.6, 0.8
    for sign in (+1.0, -1.0):
        L, R = species_state(s, 0.1), species_state(s, 0.1)
        for Q in (L, R):
            a = np.sqrt(ph.gamma_gas * Rs * Q[4])
            Q[1:3] += sign * 3.0 * a * np.array([nx, ny])
        up = L if sign > 0 else R
        F = euler_Fn(up, nx, ny, Rs, ph.gamma_gas)
        np.testing.assert_allclose(orc.flux_ausm(ph, nu, s, L, R, nx, ny), F, rtol=1e-14, atol=0)


@pytest.mark.parametrize("s", [0, 1])
def test_ausm_contact_and_signs(orc, s):
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    Rs = 1.0 if s == 0 else ph.mass_ratio
    nx, ny = np.cos(0.3), np.sin(0.3)
    # stationary contact (u = 0, equal pressures, density jump) is preserved: H = (0, p n, 0)
    L = np.array([1.0, 0, 0, 0, 0.5]) / np.array([1 if s == 0 else 25.0, 1, 1, 1, 1])
    R = L.copy()
    R[0] *= 3.0
    R[4] /= 3.0
    p = L[0] * Rs * L[4]
    np.testing.assert_allclose(orc.flux_ausm(ph, nu, s, L, R, nx, ny), [0, p * nx, p * ny, 0, 0], atol=1e-15)
    # pressure-diffusion term M_p: fluid at rest, p_R > p_L  =>  mass flows from R to L (mdot < 0)
    R = L.copy()
    R[4] *= 1.2
    assert orc.flux_ausm(ph, nu, s, L, R, nx, ny)[0] < 0
    assert orc.flux_ausm(ph, nu, s, R, L, nx, ny)[0] > 0
    # velocity-diffusion term p_u: receding streams (u_nR - u_nL > 0) lower the interface pressure
    a = np.sqrt(ph.gamma_gas * Rs * L[4])
    Lm, Rp = L.copy(), L.copy()
    Lm[1:3] = -0.1 * a * np.array([nx, ny])
    Rp[1:3] = +0.1 * a * np.array([nx, ny])
    H = orc.flux_ausm(ph, nu, s, Lm, Rp, nx, ny)
    p_iface = H[1] * nx + H[2] * ny        # mdot = 0 by symmetry -> only the pressure part
    assert abs(H[0]) < 1e-15 and p_iface < p
    H = orc.flux_ausm(ph, nu, s, Rp, Lm, nx, ny)   # approaching streams raise it
    assert (H[1] * nx + H[2] * ny) > p


@pytest.mark.parametrize("s", [0, 1])
@pytest.mark.parametrize("Kp,sigma,minf", [(0.25, 1.0, 0.1), (0.4, 0.7, 0.3), (0.25, 1.0, 1.0)])
def test_ausm_pressure_diffusion_magnitude_at_rest(orc, s, Kp, sigma, minf):
    """Magnitude of M_p (Liou's AUSM+-up, ref. [30] via L99).  Both fluids at rest with
    different pressure, density and temperature: M_L = M_R = 0, the split Mach numbers cancel
    (M4+(0) + M4-(0) = 3/8 - 3/8), Mbar = 0 so M_o = M_inf, f_a = M_inf (2 - M_inf), and the whole mass flux is the
    pressure-diffusion term:
        mdot = a12 M_p rho_up,  M_p = -(K_p / f_a) (p_R - p_L) / (rho12 a12^2),
    with a12 = (a_L + a_R)/2, rho12 = (rho_L + rho_R)/2 and rho_up the side the flow comes from.  p_u vanishes
    (u_nR = u_nL), P5+-(0) = 1/2, so the interface pressure is the mean.  A wrong power of a12, a dropped 1/f_a,
    rho_L for rho12 or a geometric mean for a12 all fail."""
    ph = orc.physics_c()
    nu = orc.default_numerics(ph, ausm_Kp=Kp, ausm_sigma=sigma, ausm_Minf=[minf, minf])
    Rs = 1.0 if s == 0 else ph.mass_ratio
    g = ph.gamma_gas
    nx, ny = np.cos(1.1), np.sin(1.1)
    for rhoL, TL, rhoR, TR in [(1.0, 0.5, 1.7, 0.9), (1.3, 0.8, 0.6, 0.35), (0.9, 0.4, 0.9, 0.45)]:
        rhoL, rhoR = rhoL / (1.0 if s == 0 else 25.0), rhoR / (1.0 if s == 0 else 25.0)
        L, R = np.array([rhoL, 0, 0, 0, TL]), np.array([rhoR, 0, 0, 0, TR])
        pL, pR = rhoL * Rs * TL, rhoR * Rs * TR
        a12 = 0.5 * (np.sqrt(g * Rs * TL) + np.sqrt(g * Rs * TR))
        fa = minf * (2.0 - minf)
        Mp = -(Kp / fa) * (pR - pL) / (0.5 * (rhoL + rhoR) * a12 ** 2)
        up_rho, up_T = (rhoL, TL) if Mp > 0 else (rhoR, TR)
        mdot = a12 * Mp * up_rho
        p12 = 0.5 * (pL + pR)
        Ht = g * Rs / (g - 1.0) * up_T                       # total enthalpy of a fluid at rest
        expect = np.array([mdot, p12 * nx, p12 * ny, 0.0, mdot * Ht])
        H = orc.flux_ausm(ph, nu, s, L, R, nx, ny)
        np.testing.assert_allclose(H, expect, rtol=1e-13, atol=1e-15 * p12)
        assert abs(mdot) > 1e-3 * up_rho * a12                # the term is not negligible in this test


@pytest.mark.parametrize("s", [0, 1])
@pytest.mark.parametrize("Ku,minf", [(0.75, 0.1), (0.5, 0.4)])
def test_ausm_velocity_diffusion_magnitude_symmetric_streams(orc, s, Ku, minf):
    """Magnitude of p_u.  Symmetric receding (or approaching) streams, u_nL = -u, u_nR = +u,
    equal rho and T, M = u/a: M4+(-M) + M4-(M) = 0 and p_R = p_L, so mdot = 0 and the flux is (0, p12 n, 0) with
        p12 = (P5+(-M) + P5-(M)) p - K_u P5+(-M) P5-(M) (rho_L + rho_R) (f_a a) (u_nR - u_nL),
    Mbar^2 = M^2, M_o = sqrt(min(1, max(M^2, M_inf^2))), f_a = M_o (2 - M_o), alpha = 3/16 (-4 + 5 f_a^2).
    P5 is taken in Liou's published monomial form P5+-(M) = 1/4 (M +- 1)^2 (2 -+ M) +- alpha M (M^2 - 1)^2 (the
    oracle nests it differently); as a second route, the pressure-split part is measured from the oracle itself
    with K_u = 0 and only the difference is compared with the closed form of p_u."""
    ph = orc.physics_c()
    Rs = 1.0 if s == 0 else ph.mass_ratio
    g = ph.gamma_gas
    nu = orc.default_numerics(ph, ausm_Ku=Ku, ausm_Minf=[minf, minf])
    nu0 = orc.default_numerics(ph, ausm_Ku=0.0, ausm_Minf=[minf, minf])
    nx, ny = np.cos(-0.4), np.sin(-0.4)
    rho, T = 1.2 / (1.0 if s == 0 else 25.0), 0.6
    a, p = np.sqrt(g * Rs * T), rho * Rs * T
    for M in (0.05, 0.3, 0.7, -0.3, -0.7):                    # M > 0 receding, M < 0 approaching
        u = M * a
        L = np.array([rho, -u * nx, -u * ny, 0.3, T])
        R = np.array([rho, +u * nx, +u * ny, -0.2, T])
        Mo = np.sqrt(min(1.0, max(M * M, minf * minf)))
        fa = Mo * (2.0 - Mo)
        alpha = 3.0 / 16.0 * (-4.0 + 5.0 * fa * fa)
        P5p = lambda m: 0.25 * (m + 1) ** 2 * (2 - m) + alpha * m * (m * m - 1) ** 2
        P5m = lambda m: 0.25 * (m - 1) ** 2 * (2 + m) - alpha * m * (m * m - 1) ** 2
        Pp, Pm = P5p(-M), P5m(M)
        assert abs(Pp - Pm) < 1e-15                            # symmetry of the set-up
        pu = -Ku * Pp * Pm * (2 * rho) * (fa * a) * (2 * u)
        H = orc.flux_ausm(ph, nu, s, L, R, nx, ny)
        H0 = orc.flux_ausm(ph, nu0, s, L, R, nx, ny)
        assert abs(H[0]) < 1e-15 * rho * a and abs(H[3]) < 1e-15 * p and abs(H[4]) < 1e-14 * p * a
        p12, p12_0 = H[1] * nx + H[2] * ny, H0[1] * nx + H0[2] * ny
        np.testing.assert_allclose(p12, (Pp + Pm) * p + pu, rtol=1e-13)
        # second route: P from the K_u = 0 evaluation, p_u from the difference
        P_meas = p12_0 / (2 * p)
        np.testing.assert_allclose(p12 - p12_0, -Ku * P_meas ** 2 * (2 * rho) * (fa * a) * (2 * u), rtol=1e-11)
        assert abs(pu) > 1e-3 * p * abs(M)                     # the term matters here


def test_ausm_split_functions(orc):
    """Liou's polynomials: beta = 1/8 puts an inflection of M4+ at M = 0; alpha = 3/16 makes P5+
    twice differentiable at M = 1; M4+ + M4- = M and P5+ + P5- = 1 for any alpha, beta;
    |M| >= 1 gives the van Leer/upwind limits."""
    h = 1e-4
    d2 = lambda f, x: (f(x + h) - 2 * f(x) + f(x - h)) / h ** 2
    assert abs(d2(lambda M: orc.ausm_split(M)[0], 0.0)) < 1e-6
    assert abs(d2(lambda M: orc.ausm_split(M, beta=0.2)[0], 0.0)) > 0.1
    f = lambda M: orc.ausm_split(M)[2]
    # one-sided second derivative from below at M = 1 vanishes (above it is identically 0)
    assert abs((f(1 - 2 * h) - 2 * f(1 - h) + f(1.0)) / h ** 2) < 5e-3
    g = lambda M: orc.ausm_split(M, alpha=0.1)[2]
    assert abs((g(1 - 2 * h) - 2 * g(1 - h) + g(1.0)) / h ** 2) > 0.5
    for M in np.linspace(-1.7, 1.7, 35):
        for al, be in ((3 / 16, 1 / 8), (-0.3, 0.05)):
            o = orc.ausm_split(M, al, be)
            assert abs(o[0] + o[1] - M) < 1e-15 and abs(o[2] + o[3] - 1.0) < 1e-15
    np.testing.assert_allclose(orc.ausm_split(1.5), [1.5, 0, 1, 0], atol=1e-16)
    np.testing.assert_allclose(orc.ausm_split(-1.5), [0, -1.5, 0, 1], atol=1e-16)
    np.testing.assert_allclose(orc.ausm_split(0.0), [0.375, -0.375, 0.5, 0.5], atol=1e-16)


def test_face_flux_rotation_covariance(orc):
    """S19 at a face: rotating n and the in-plane vector components rotates the flux rows."""
    ph = orc.physics_c()
    nu = orc.default_numerics(ph)
    th = 0.7
    Q = rot18(th)
    PL, PR = random_state(RNG, 1)[0], random_state(RNG, 1)[0]
    nx, ny = np.cos(1.1), np.sin(1.1)
    H = orc.flux_face(ph, nu, PL, PR, nx, ny)
    nxr, nyr = np.cos(1.1 + th), np.sin(1.1 + th)
    Hr = orc.flux_face(ph, nu, Q @ PL, Q @ PR, nxr, nyr)
    np.testing.assert_allclose(Hr, Q @ H, rtol=0, atol=1e-12 * np.abs(H).max())
    # and the full-face consistency with the physical flux (L85)
    np.testing.assert_allclose(orc.flux_face(ph, nu, PL, PL, nx, ny), orc.phys_flux(ph, PL, nx, ny),
                               rtol=0, atol=1e-13 * ph.c ** 2)


# ------------------------------------------------------------------------------------------
# source (L60 Eq. 4, L65-68 Eq. 6) and conservative variables (L63 Eq. 5)
# ------------------------------------------------------------------------------------------
def test_source_bookkeeping(orc):
    ph = orc.physics_c()
    c2, mr = ph.c ** 2, ph.mass_ratio
    for P in random_state(RNG, 8):
        S = orc.source(ph, P)
        B, E = P[0:3], P[3:6]
        n_i, n_e = P[8] / 1.0, P[9] / (1.0 / mr)           # number densities, m_i = 1, m_e = 1/mr
        ui, ue = P[10:13], P[13:16]
        J = n_i * ui - n_e * ue                            # q_i = +1, q_e = -1
        rhoc = n_i - n_e
        tol = 1e-12 * c2
        np.testing.assert_allclose(S[3:6], -c2 * J, atol=tol)      # -J/eps0, eps0 = 1/c^2
        np.testing.assert_allclose(S[7], c2 * rhoc, atol=tol)      # rho_c/eps0
        assert np.all(S[[0, 1, 2, 6, 8, 9]] == 0.0)
        np.testing.assert_allclose(S[10:13] + S[13:16], rhoc * E + np.cross(J, B), atol=1e-12)
        np.testing.assert_allclose(S[16] + S[17], np.dot(J, E), atol=1e-12)
        np.testing.assert_allclose(S[10:13], n_i * (E + np.cross(ui, B)), atol=1e-12)
        np.testing.assert_allclose(S[17], -n_e * np.dot(ue, E), atol=1e-12)


def test_cons_and_dcons(orc):
    ph = orc.physics_c()
    g, mr = ph.gamma_gas, ph.mass_ratio
    for P in random_state(RNG, 4):
        U = orc.cons(ph, P)
        np.testing.assert_array_equal(U[:8], P[:8])
        for s, (ir, iu, iT, Rs) in enumerate([(8, 10, 16, 1.0), (9, 13, 17, mr)]):
            rho, u, T = P[ir], P[iu:iu + 3], P[iT]
            p = rho * Rs * T
            assert abs(U[ir] - rho) == 0
            np.testing.assert_allclose(U[iu:iu + 3], rho * u, rtol=1e-15)
            np.testing.assert_allclose(U[iT], p / (g - 1) + 0.5 * rho * np.dot(u, u), rtol=1e-14)
        D = orc.dcons_dprim(ph, P)
        Dfd = np.zeros((18, 18))
        for k in range(18):
            h = 1e-6
            e = np.zeros(18)
            e[k] = h
            Dfd[:, k] = (orc.cons(ph, P + e) - orc.cons(ph, P - e)) / (2 * h)
        np.testing.assert_allclose(D, Dfd, rtol=0, atol=1e-8 * np.abs(D).max())
