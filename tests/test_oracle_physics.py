"""Pins P5, P6, P7 (pointwise part), P15 and the wall / source functions of the oracle: special cases that
reduce to textbook formulas, invariants, and numerical differentiation of the paper's closed forms."""
import numpy as np
import pytest

from oracle import binding as ob
from paper_2502_17805_b200 import inputs as I

GAM = 5.0 / 3.0
RNG = np.random.default_rng(7)


def rand_state(with_B=True, with_psi=True):
    rho = RNG.uniform(0.5, 2.0); u = RNG.uniform(-1, 1, 3); p = RNG.uniform(0.5, 2.0)
    B = RNG.uniform(-1, 1, 3) if with_B else np.zeros(3)
    psi = RNG.uniform(-0.5, 0.5) if with_psi else 0.0
    return I.conserved(rho, u, p, B, np.float64(psi), GAM), (rho, u, p, B, psi)


def unit(v):
    return v / np.linalg.norm(v)


PH = I.Physics(gamma=GAM, R_gas=1.3, Cp=GAM * 1.3 / (GAM - 1), c_h=1.7, nu=0.03, kappa=0.05, eta=0.02)


def test_p5_euler_limit_is_textbook_euler_flux():
    for _ in range(5):
        Q, (rho, u, p, B, psi) = rand_state(with_B=False, with_psi=False)
        S = RNG.uniform(-1, 1, 3)
        un = u @ S
        E = p / (GAM - 1) + 0.5 * rho * u @ u
        ref = np.concatenate([[rho * un], rho * u * un + p * S, [(E + p) * un], np.zeros(3), [0.0]])
        np.testing.assert_allclose(ob.flux_inviscid(PH, Q, S), ref, rtol=0, atol=1e-14)


def test_p5_static_fluid_gives_maxwell_stress_only():
    Q, (rho, u, p, B, psi) = rand_state(with_psi=False)
    Q = I.conserved(rho, np.zeros(3), p, B, np.float64(0.0), GAM)
    S = RNG.uniform(-1, 1, 3)
    F = ob.flux_inviscid(PH, Q, S)
    np.testing.assert_allclose(F[1:4], (p + 0.5 * B @ B) * S - B * (B @ S), atol=1e-14)
    assert F[0] == 0 and F[4] == 0
    np.testing.assert_allclose(F[5:8], 0.0, atol=1e-15)
    np.testing.assert_allclose(F[8], PH.c_h * (B @ S), atol=1e-15)


def test_p5_flux_is_linear_in_S_and_rotationally_covariant():
    Q, _ = rand_state()
    S1, S2 = RNG.uniform(-1, 1, 3), RNG.uniform(-1, 1, 3)
    F = ob.flux_inviscid(PH, Q, 2.0 * S1 - 0.5 * S2)
    np.testing.assert_allclose(F, 2.0 * ob.flux_inviscid(PH, Q, S1) - 0.5 * ob.flux_inviscid(PH, Q, S2), atol=1e-13)
    # rotate the whole configuration: scalars invariant, vectors rotate
    A = np.linalg.qr(RNG.normal(size=(3, 3)))[0]
    if np.linalg.det(A) < 0:
        A[:, 0] *= -1
    Qr = Q.copy(); Qr[1:4] = A @ Q[1:4]; Qr[5:8] = A @ Q[5:8]
    Fr = ob.flux_inviscid(PH, Qr, A @ S1)
    F1 = ob.flux_inviscid(PH, Q, S1)
    np.testing.assert_allclose(Fr[[0, 4, 8]], F1[[0, 4, 8]], atol=1e-13)
    np.testing.assert_allclose(Fr[1:4], A @ F1[1:4], atol=1e-13)
    np.testing.assert_allclose(Fr[5:8], A @ F1[5:8], atol=1e-13)


def test_p5_induction_row_index_convention():
    """Reading G7: flux of B_i along j is u_j B_i - B_j u_i (antisymmetric), so the x-flux of B_x vanishes without GLM."""
    ph = PH.copy(c_h=0.0)
    Q, (rho, u, p, B, psi) = rand_state()
    F = ob.flux_inviscid(ph, Q, np.array([1.0, 0, 0]))
    assert abs(F[5]) < 1e-15
    np.testing.assert_allclose(F[6], u[0] * B[1] - B[0] * u[1], atol=1e-15)
    np.testing.assert_allclose(F[7], u[0] * B[2] - B[0] * u[2], atol=1e-15)


def test_p6_rusanov_consistency_and_antisymmetry():
    for _ in range(5):
        Qa, _ = rand_state(); Qb, _ = rand_state()
        nh = unit(RNG.normal(size=3))
        np.testing.assert_allclose(ob.flux_rusanov(PH, Qa, Qa, nh), ob.flux_inviscid(PH, Qa, nh), rtol=0, atol=1e-15)
        assert np.array_equal(ob.flux_rusanov(PH, Qa, Qb, nh), -ob.flux_rusanov(PH, Qb, Qa, -nh))    # bitwise
        # dissipation: F_c - central = -lambda/2 (Qb - Qa) with lambda >= every one-sided speed and >= C_h
        cen = 0.5 * (ob.flux_inviscid(PH, Qa, nh) + ob.flux_inviscid(PH, Qb, nh))
        d = ob.flux_rusanov(PH, Qa, Qb, nh) - cen
        lam = -2 * d[0] / (Qb[0] - Qa[0])
        np.testing.assert_allclose(d, -0.5 * lam * (Qb - Qa), atol=1e-12)
        for Q in (Qa, Qb):
            un = abs(Q[1:4] @ nh / Q[0])
            assert lam >= un + ob.fast_speed(PH, Q, nh) - 1e-12
        assert lam >= PH.c_h


def test_p6_fast_speed_limits():
    Q, (rho, u, p, B, psi) = rand_state()
    a = np.sqrt(GAM * p / rho); b = np.sqrt(B @ B / rho)
    Q0 = I.conserved(rho, u, p, np.zeros(3), np.float64(psi), GAM)
    assert abs(ob.fast_speed(PH, Q0, unit(RNG.normal(size=3))) - a) < 1e-14            # B = 0 -> sound speed
    nperp = unit(np.cross(B, RNG.normal(size=3)))
    assert abs(ob.fast_speed(PH, Q, nperp) - np.sqrt(a * a + b * b)) < 1e-13           # B perp n
    assert abs(ob.fast_speed(PH, Q, unit(B)) - max(a, b)) < 1e-13                      # B parallel n


def test_p15_wavespeed_is_max_over_directions():
    for _ in range(3):
        Q, (rho, u, p, B, psi) = rand_state()
        dirs = RNG.normal(size=(4000, 3)); dirs /= np.linalg.norm(dirs, axis=1)[:, None]
        dirs = np.vstack([dirs, unit(np.cross(B, [0.3, -0.2, 0.9]))])
        cf = max(ob.fast_speed(PH, Q, d) for d in dirs)
        assert abs(ob.wavespeed(PH, Q) - (np.linalg.norm(u) + cf)) < 1e-12
        assert ob.wavespeed(PH, Q) >= np.linalg.norm(u) + cf - 1e-14


# ---------------------------------------------------------------------------------------- viscous flux
def _grad_from_prims(rho, u, p, B, psi, drho, du, dp, dB, dpsi):
    """Gradient of the conserved variables from primitive gradients (product rule on Eq. 2-3).
    du[i][j] = d_j u_i, dB[i][j] = d_j B_i.  Returns G[27] with G[3v+j]."""
    G = np.zeros((9, 3))
    G[0] = drho
    for i in range(3):
        G[1 + i] = drho * u[i] + rho * du[i]
    G[4] = dp / (GAM - 1) + 0.5 * drho * (u @ u) + rho * (u @ du) + B @ dB + psi * dpsi
    for i in range(3):
        G[5 + i] = dB[i]
    G[8] = dpsi
    return G.reshape(-1)


def test_p7_viscous_flux_against_textbook_navier_stokes_and_ohm():
    for _ in range(5):
        Q, (rho, u, p, B, psi) = rand_state()
        drho, dp, dpsi = RNG.normal(size=3), RNG.normal(size=3), RNG.normal(size=3)
        du, dB = RNG.normal(size=(3, 3)), RNG.normal(size=(3, 3))
        G = _grad_from_prims(rho, u, p, B, psi, drho, du, dp, dB, dpsi)
        kr = 0.07
        mu = rho * PH.nu
        tau = mu * (du + du.T) - (2.0 / 3.0) * mu * np.trace(du) * np.eye(3)            # Eq. 8 with Stokes' hypothesis
        T = p / (rho * PH.R_gas)
        # grad S and grad T by central differences of the paper's closed forms (Eq. 10, Eq. 4)
        Sfun = lambda r_, p_: PH.Cp * np.log(p_ ** (1 / GAM) / r_)
        Tfun = lambda r_, p_: p_ / (r_ * PH.R_gas)
        h = 1e-6
        dS = np.array([(Sfun(rho + h * drho[j], p + h * dp[j]) - Sfun(rho - h * drho[j], p - h * dp[j])) / (2 * h) for j in range(3)])
        dT = np.array([(Tfun(rho + h * drho[j], p + h * dp[j]) - Tfun(rho - h * drho[j], p - h * dp[j])) / (2 * h) for j in range(3)])
        q = -PH.kappa * rho * T * dS - kr * rho * PH.Cp * dT                            # Eq. 9
        J = np.array([dB[2, 1] - dB[1, 2], dB[0, 2] - dB[2, 0], dB[1, 0] - dB[0, 1]])    # curl B
        S = RNG.normal(size=3)
        ref = np.zeros(9)
        ref[1:4] = tau @ S
        ref[4] = (u @ tau - q + PH.eta * np.cross(B, J)) @ S                             # Eq. 7 energy row
        ref[5:8] = PH.eta * (dB @ S - dB.T @ S)                                          # eta (d_j B_i - d_i B_j) S_j  (G10)
        F = ob.flux_viscous(PH, Q, G, S, kr)
        np.testing.assert_allclose(F, ref, atol=2e-8, rtol=0)      # limited by the finite differences
        np.testing.assert_allclose(F[[0, 8]], 0.0, atol=0)
        # everything except the heat flux is exact
        ref_noq = ref.copy(); ref_noq[4] += q @ S
        Fq = ob.flux_viscous(PH.copy(kappa=0.0), Q, G, S, 0.0)
        np.testing.assert_allclose(Fq, ref_noq, atol=1e-13, rtol=0)


def test_p7_resistive_flux_is_minus_curl_of_eta_J():
    """div of the induction rows = -curl(eta J) for B = (0, sin(kx), 0): x-flux of B_y = eta dB_y/dx (sign of G10)."""
    Q, (rho, u, p, B, psi) = rand_state()
    dB = np.zeros((3, 3)); dB[1, 0] = 0.8
    G = _grad_from_prims(rho, u, p, B, psi, np.zeros(3), np.zeros((3, 3)), np.zeros(3), dB, np.zeros(3))
    F = ob.flux_viscous(PH.copy(nu=0.0, kappa=0.0), Q, G, np.array([1.0, 0, 0]))
    np.testing.assert_allclose(F[6], PH.eta * 0.8, atol=1e-15)
    np.testing.assert_allclose(F[4], PH.eta * B[1] * 0.8, atol=1e-14)      # eta (B x J)_x = eta B_y dB_y/dx


def test_table1_identity_cp():
    assert abs((5 / 3) * 1.4e8 / (2 / 3) - 3.5e8) < 1e-6


# ---------------------------------------------------------------------------------------- walls, sources
@pytest.mark.parametrize("wall,bc", [(-1, I.BC_CONDUCTING), (-1, I.BC_RADIAL), (-2, I.BC_CONDUCTING), (-2, I.BC_RADIAL)])
def test_wall_state_and_fluxes(wall, bc):
    ph = PH.copy(bc_mag_inner=bc, bc_mag_outer=bc)
    Q, (rho, u, p, B, psi) = rand_state()
    nh = unit(RNG.normal(size=3))
    Qb = ob.wall_state(ph, wall, Q, nh)
    ub, Bb = Qb[1:4] / Qb[0], Qb[5:8]
    assert abs(ub @ nh) < 1e-15                                      # Eq. 33
    np.testing.assert_allclose(ub, u - (u @ nh) * nh, atol=1e-15)
    if bc == I.BC_CONDUCTING:
        assert abs(Bb @ nh) < 1e-15                                  # B_r = 0
    else:
        np.testing.assert_allclose(np.cross(Bb, nh), 0.0, atol=1e-15)   # B_theta = B_phi = 0
    pb = (GAM - 1) * (Qb[4] - 0.5 * rho * ub @ ub - 0.5 * Bb @ Bb - 0.5 * psi ** 2)
    assert abs(pb - p) < 1e-14 and Qb[0] == rho and Qb[8] == psi
    Fw = ob.flux_wall_inviscid(ph, Qb, nh)
    assert Fw[0] == 0.0                                              # impenetrable: exactly zero mass flux
    # equals the general flux evaluated on a state whose normal velocity is exactly zero
    np.testing.assert_allclose(Fw, ob.flux_inviscid(ph, Qb, nh), atol=1e-14)
    # viscous wall flux: traction purely normal, no viscous work
    G = RNG.normal(size=27)
    Fv = ob.flux_wall_viscous(ph, wall, Qb, G, nh)
    np.testing.assert_allclose(np.cross(Fv[1:4], nh), 0.0, atol=1e-15)
    if bc == I.BC_CONDUCTING:
        np.testing.assert_allclose(Fv[5:8], 0.0, atol=1e-14 * np.abs(G).max())   # J = J_r r_hat: no resistive flux through the wall
    gen = ob.flux_viscous(ph, Qb, G, nh)
    np.testing.assert_allclose(Fv[1:4] @ nh, gen[1:4] @ nh, atol=1e-13)      # normal traction kept


def test_wall_thermal_options():
    Q, (rho, u, p, B, psi) = rand_state()
    nh = unit(RNG.normal(size=3))
    ph = PH.copy(T_top=0.9, q_bottom=0.37, flags=I.FLAG_FIXED_T_OUTER | I.FLAG_FIXED_FLUX_INNER)
    Qb = ob.wall_state(ph, -2, Q, nh)
    ub, Bb = Qb[1:4] / Qb[0], Qb[5:8]
    pb = (GAM - 1) * (Qb[4] - 0.5 * rho * ub @ ub - 0.5 * Bb @ Bb - 0.5 * psi ** 2)
    assert abs(pb - rho * ph.R_gas * 0.9) < 1e-14                    # p_b = rho R T_top (Eq. 4)
    Qi = ob.wall_state(ph, -1, Q, nh)
    G = np.zeros(27)
    Fv = ob.flux_wall_viscous(ph, -1, Qi, G, nh)
    assert abs(Fv[4] - 0.37) < 1e-15                                 # -q.n with q.n = -q_bottom (Eq. 32)


def _rot(rng):
    A = rng.normal(size=(3, 3))
    Qm, _ = np.linalg.qr(A)
    return Qm * np.sign(np.linalg.det(Qm))


def test_wall_gradient_conditions_on_the_jacobian_of_B():
    """conductor B_r = d_r(r B_theta) = d_r(r B_phi) = 0; radial B_theta = B_phi = 0, d_r(r^2 B_r) = 0, imposed on
    the Jacobian of B in the spherical frame of the wall point (reading G29).  Fields that satisfy a condition exactly keep their
    Jacobian; a generic Jacobian loses its tangential current (conductor) or its radial current and its divergence (radial);
    the operation is covariant (independent of the tangent vectors chosen for the frame)."""
    rng = np.random.default_rng(11)
    x = np.array([0.31, -0.52, 0.44]); r = np.linalg.norm(x); er = x / r
    eye = np.eye(3)
    # perfectly radial field B = x/r^3 (B_r = 1/r^2): d_j B_i = delta_ij/r^3 - 3 x_i x_j/r^5
    B = x / r ** 3
    dB = eye / r ** 3 - 3 * np.outer(x, x) / r ** 5
    np.testing.assert_allclose(ob.wall_condition_gradB(I.BC_RADIAL, dB, B, er, r), dB, atol=1e-14 * np.abs(dB).max())
    # toroidal field B = (z_hat x x)/r^2 = sin(theta) phi_hat / r: B_r = 0, r B_phi independent of r
    A = np.array([-x[1], x[0], 0.0])
    dA = np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    B = A / r ** 2
    dB = dA / r ** 2 - 2 * np.outer(A, x) / r ** 4
    assert abs(B @ er) < 1e-16
    np.testing.assert_allclose(ob.wall_condition_gradB(I.BC_CONDUCTING, dB, B, er, r), dB, atol=1e-14 * np.abs(dB).max())
    assert np.abs(ob.wall_condition_gradB(I.BC_RADIAL, dB, 0 * B, er, r) - dB).max() > 0.1 * np.abs(dB).max()   # ... and is not a radial-wall field
    # generic Jacobians
    curl = lambda D: np.array([D[2, 1] - D[1, 2], D[0, 2] - D[2, 0], D[1, 0] - D[0, 1]])
    for _ in range(20):
        dB = rng.normal(size=(3, 3)); Bf = rng.normal(size=3); er = unit(rng.normal(size=3)); rw = rng.uniform(0.5, 2.0)
        Bt, Br = Bf - (Bf @ er) * er, (Bf @ er) * er
        Dc = ob.wall_condition_gradB(I.BC_CONDUCTING, dB, Bt, er, rw)
        Jc = curl(Dc)
        np.testing.assert_allclose(np.cross(Jc, er), 0.0, atol=1e-14)                  # J = J_r r_hat
        assert abs(Jc @ er - curl(dB) @ er) < 1e-14                                    # ... with J_r as computed
        assert abs(er @ Dc @ er - er @ dB @ er) < 1e-14                                # d_r B_r is not constrained
        Dr = ob.wall_condition_gradB(I.BC_RADIAL, dB, Br, er, rw)
        Jr = curl(Dr)
        assert abs(np.trace(Dr)) < 1e-14                                               # div B = 0 at the wall
        assert abs(Jr @ er) < 1e-14                                                    # no radial current
        np.testing.assert_allclose(np.cross(Jr, er), np.cross(curl(dB), er), atol=1e-14)   # tangential current as computed
        assert abs(er @ Dr @ er + 2 * (Bf @ er) / rw) < 1e-14                          # d_r(r^2 B_r) = 0
        Rm = _rot(rng)                                                                 # covariance
        for bc, Bw in ((I.BC_CONDUCTING, Bt), (I.BC_RADIAL, Br)):
            D0 = ob.wall_condition_gradB(bc, dB, Bw, er, rw)
            D1 = ob.wall_condition_gradB(bc, Rm @ dB @ Rm.T, Rm @ Bw, Rm @ er, rw)
            np.testing.assert_allclose(D1, Rm @ D0 @ Rm.T, atol=1e-14)


@pytest.mark.parametrize("wall,bc", [(-1, I.BC_CONDUCTING), (-1, I.BC_RADIAL), (-2, I.BC_CONDUCTING), (-2, I.BC_RADIAL)])
@pytest.mark.parametrize("thermal", [0, I.FLAG_FIXED_T_OUTER | I.FLAG_FIXED_FLUX_INNER])
def test_wall_viscous_flux_with_conditioned_gradients_closed_form(wall, bc, thermal):
    """The wall viscous flux built from the conditioned wall gradients equals, term by term, the closed form the conditions
    imply: traction (n.tau.n) n with tau of Eq. 8, no viscous work, heat flux -q.n with q of Eq. 9 (or q_bottom, Eq. 32), no
    resistive flux through a perfect conductor, -eta n x J for a radial-field wall and no Poynting flux in either case; and it
    does not depend on the radius of the wall (the curvature terms only enter components that carry no flux)."""
    rng = np.random.default_rng(100 + 7 * wall + bc)
    ph = PH.copy(bc_mag_inner=bc, bc_mag_outer=bc, T_top=0.9, q_bottom=0.37, flags=I.FLAG_DIFFUSION | thermal)
    for _ in range(5):
        Q, _ = rand_state()
        nh = unit(rng.normal(size=3))
        Qb = ob.wall_state(ph, wall, Q, nh)
        rho, ub, Bb, psi = Qb[0], Qb[1:4] / Qb[0], Qb[5:8], Qb[8]
        pb = (GAM - 1) * (Qb[4] - 0.5 * rho * ub @ ub - 0.5 * Bb @ Bb - 0.5 * psi ** 2)
        G = rng.normal(size=27)
        kr = 0.013
        Fv = ob.flux_wall_viscous(ph, wall, Qb, G, nh, kr=kr, rw=0.83)
        g = G.reshape(9, 3)
        du = (g[1:4] - np.outer(ub, g[0])) / rho                                       # d_j u_i
        tau = rho * ph.nu * (du + du.T) - (2 / 3) * rho * ph.nu * np.trace(du) * np.eye(3)   # Eq. 8, mu = rho nu, Stokes
        dp = (GAM - 1) * (g[4] - ub @ g[1:4] + 0.5 * (ub @ ub) * g[0] - Bb @ g[5:8] - psi * g[8])
        dT = (dp - pb / rho * g[0]) / (rho * ph.R_gas)
        dS = ph.Cp * (dp / (GAM * pb) - g[0] / rho)
        q = -ph.kappa * rho * (pb / (rho * ph.R_gas)) * dS - kr * rho * ph.Cp * dT     # Eq. 9
        qn = q @ nh
        if wall == -1 and thermal:
            qn = -0.37
        ref = np.zeros(9)
        ref[1:4] = (nh @ tau @ nh) * nh
        ref[4] = -qn
        J = np.array([g[7, 1] - g[6, 2], g[5, 2] - g[7, 0], g[6, 0] - g[5, 1]])
        if bc == I.BC_RADIAL:
            ref[5:8] = -ph.eta * np.cross(nh, J)
        np.testing.assert_allclose(Fv, ref, atol=2e-13 * max(1.0, np.abs(ref).max()))
        for rw in (0.0, 0.3, 5.0):
            np.testing.assert_allclose(ob.flux_wall_viscous(ph, wall, Qb, G, nh, kr=kr, rw=rw), Fv, atol=1e-13 * max(1.0, np.abs(ref).max()))


def test_source_terms():
    ph = PH.copy(GM=1.3, Omega=0.4, a_psi=2.5,
                 flags=I.FLAG_GRAVITY | I.FLAG_CORIOLIS | I.FLAG_POWELL | I.FLAG_GLM_DAMP)
    Q, (rho, u, p, B, psi) = rand_state()
    G = RNG.normal(size=27)
    x = RNG.normal(size=3)
    M, Ma = ob.source(ph, Q, G, x)
    r = np.linalg.norm(x)
    g = -ph.GM * x / r ** 3
    divB = G[15] + G[19] + G[23]
    ref = np.zeros(9)
    ref[1:4] = rho * g - 2 * rho * np.cross([0, 0, ph.Omega], u) - divB * B          # Eq. 5
    ref[4] = rho * u @ g - divB * (u @ B)
    ref[5:8] = -divB * u
    ref[8] = -ph.a_psi * psi
    np.testing.assert_allclose(M, ref, atol=1e-13)
    assert M[0] == 0.0 and np.all(Ma >= np.abs(M) - 1e-15)
    # each flag gates its own term
    M0, _ = ob.source(ph.copy(flags=0), Q, G, x)
    assert np.all(M0 == 0)
    Mc, _ = ob.source(ph.copy(flags=I.FLAG_CENTRIFUGAL), Q, G, x)
    cen = -rho * np.cross([0, 0, ph.Omega], np.cross([0, 0, ph.Omega], x))          # -rho Omega x (Omega x x)  (reading G22)
    np.testing.assert_allclose(Mc[1:4], cen, atol=1e-14)
    np.testing.assert_allclose(Mc[4], u @ cen, atol=1e-14)                            # its work term, the energy row
    assert Mc[0] == 0.0 and np.all(Mc[5:] == 0.0)
