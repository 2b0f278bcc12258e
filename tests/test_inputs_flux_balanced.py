"""Pins of the flux-balanced initial stratification (Eq. 28-31; inputs.flux_balanced_profile): the isentropic
special case is the polytrope of Eq. 26 in closed form; the general case agrees with an adaptive ODE integration of the same
equations (scipy), is in hydrostatic balance (Eq. 25) and carries the luminosity L through every radial layer (Eq. 28)."""
import numpy as np
from scipy.integrate import solve_ivp

from paper_2502_17805_b200 import inputs as I


def test_isentropic_case_is_the_polytrope():
    sh = I.Shell(N_rho=3.0)
    prof = I.flux_balanced_profile(sh, L=0.0, kappa=1e-3, n_grid=2001)
    rho, p, T = sh.profile(prof["r"])
    assert np.abs(prof["dSdr"]).max() == 0.0 and np.ptp(prof["S"]) == 0.0
    np.testing.assert_allclose(prof["rho"], rho, rtol=1e-11)
    np.testing.assert_allclose(prof["p"], p, rtol=1e-11)
    np.testing.assert_allclose(prof["T"], T, rtol=1e-11)
    assert abs(np.log(prof["rho"][0] / prof["rho"][-1]) - 3.0) < 1e-10          # N_rho = ln(rho_b/rho_t)


def test_general_case_against_adaptive_integration_and_its_invariants():
    sh = I.Shell(N_rho=3.0)
    L, kappa = 2e-5, 2e-3
    kr = lambda r: 1e-5 * (1.0 - 0.8 * (1.7 * r) + 0.6 * (1.7 * r) ** 2)         # the profile form of PAPER.md:216
    prof = I.flux_balanced_profile(sh, L, kappa, kr, n_grid=4001)
    r = prof["r"]
    g, Cp, gam = sh.GM, sh.Cp, sh.gamma
    # (a) Eq. 28 on the polytrope: -kappa rho0 T0 dS/dr - kr rho0 Cp dT0/dr = L / (4 pi r^2)
    rho0, _, T0 = sh.profile(r)
    q = -kappa * rho0 * T0 * prof["dSdr"] - kr(r) * rho0 * Cp * (-g / (Cp * r * r))
    np.testing.assert_allclose(4 * np.pi * r * r * q, L, rtol=1e-13)
    # radiation carries more than L at the bottom (stable, dS/dr > 0) and less at the top (dS/dr < 0), as in the Sun
    assert prof["dSdr"][0] > 0 > prof["dSdr"][-1]
    # (b) the same ODE system (Eq. 29-31) by an adaptive integrator
    rho_b, p_b, _ = sh.profile(sh.r_b)

    def dS(rr):
        a, _, t = sh.profile(rr)
        return -(L / (4 * np.pi * rr * rr) + kr(rr) * a * Cp * (-g / (Cp * rr * rr))) / (kappa * a * t)

    def rhs(rr, y):
        S, rho = y
        return [dS(rr), -(rho / Cp * dS(rr) + g / (rr * rr) / gam * rho ** (2 - gam) * np.exp(-gam * S / Cp))]

    sol = solve_ivp(rhs, (sh.r_b, sh.r_t), [Cp * np.log(p_b ** (1 / gam) / rho_b), rho_b], t_eval=r, rtol=1e-12, atol=1e-14, method="DOP853")
    np.testing.assert_allclose(prof["S"], sol.y[0], rtol=0, atol=1e-10 * np.abs(sol.y[0]).max())
    np.testing.assert_allclose(prof["rho"], sol.y[1], rtol=1e-9)
    # (c) hydrostatic balance dp/dr = -rho g (Eq. 25), by 4th-order differences of the tabulated p
    h = r[1] - r[0]
    dp = (prof["p"][:-4] - 8 * prof["p"][1:-3] + 8 * prof["p"][3:-1] - prof["p"][4:]) / (12 * h)
    rhs_h = -(prof["rho"] * g / (r * r))[2:-2]
    np.testing.assert_allclose(dp, rhs_h, rtol=1e-8)
    # (d) Eq. 10 links the three profiles; T = p / (rho R)
    np.testing.assert_allclose(prof["S"], Cp * np.log(prof["p"] ** (1 / gam) / prof["rho"]), rtol=0, atol=1e-12)
    np.testing.assert_allclose(prof["T"], prof["p"] / (prof["rho"] * sh.R_gas), rtol=1e-15)
    # (e) a state built on it is what shell_state hands to the solver
    x = np.stack([np.linspace(0.72, 0.93, 50), np.zeros(50), np.zeros(50)])[:, None, :]
    Q = I.shell_state(x, sh, 3, u_amp=0.0, b_amp=0.0, background=prof)
    np.testing.assert_allclose(Q[0, 0], np.interp(x[0, 0], r, prof["rho"]), rtol=1e-6)       # log-linear vs linear interpolation
