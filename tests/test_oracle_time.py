"""Pins P10, P11, P12, P16 and the wiring of oracle_step: design-order convergence of an Alfven wave, decay
of div B under GLM, conservation of mass with impenetrable walls, the long-double round-off floor."""
import numpy as np
import pytest

from oracle import binding as ob
from paper_2502_17805_b200 import inputs as I
from helpers import w3, g24_error
from test_oracle_operator import alfven_wave, box_oracle, GAM


def test_step_is_the_shu_osher_combination_of_residuals():
    """oracle_step(dt, s) == literal Shu-Osher loop driven by oracle_residual."""
    n = 3
    phys = I.Physics(c_h=1.0, flags=I.FLAG_POWELL)
    o, x, _ = box_oracle(n, (2, 2, 1), phys, distort=0.05)
    Q0, _ = alfven_wave(x)
    for s in (1, 3, 5):
        al, be = ob.rk_tableau(s)
        dt = 2e-3
        u, F = [Q0], []
        for i in range(1, s + 1):
            o.set_state(u[i - 1])
            F.append(o.residual())
            u.append(sum(al[i - 1, k] * u[k] + dt * be[i - 1, k] * F[k] for k in range(i)))
        o.set_state(Q0)
        o.step(dt, s)
        np.testing.assert_allclose(o.get_state(), u[-1], rtol=0, atol=1e-14)


@pytest.mark.parametrize("n,Ns", [(3, (6, 12)), (4, (6, 12)), (5, (4, 8)), (6, (3, 6))])
def test_p10_alfven_wave_design_order(n, Ns):
    """Circularly polarised Alfven wave, B0 oblique to the box axes, periodic box: the L2 and max errors after
    a fixed time fall with h at (about) order n (north_star: "design-order convergence of a linear Alfven wave").
    dt is small enough that the RK3 error is far below the spatial error."""
    phys = I.Physics(c_h=1.0, flags=I.FLAG_POWELL)
    T = 0.2
    e_inf, e_2 = [], []
    for N in Ns:
        o, x, _ = box_oracle(n, (N, N, 1), phys)
        W = o.geometry()["detJ"] * w3(n)[None, :]
        Q0, _ = alfven_wave(x, 0.0)
        o.set_state(Q0)
        nsteps = 20 * N
        for _ in range(nsteps):
            o.step(T / nsteps, 5)
        Qex, _ = alfven_wave(x, T)
        d = o.get_state()[5:8] - Qex[5:8]
        e_inf.append(np.abs(d).max())
        e_2.append(np.sqrt((W[None] * d ** 2).sum()))
    assert np.log2(e_2[0] / e_2[1]) > n - 0.5, (e_2, e_inf)
    assert np.log2(e_inf[0] / e_inf[1]) > n - 0.7, (e_2, e_inf)
    assert np.log2(e_2[0] / e_2[1]) < n + 1.5          # and not accidentally better than the scheme can be


def _divB2(o, geo, n):
    G = o.gradient()
    divB = G[15] + G[19] + G[23]
    return float((divB ** 2 * geo["detJ"] * w3(n)[None, :]).sum())


def test_p11_glm_reduces_divB():
    """A non-solenoidal blob dB = grad(phi) on the periodic box (north_star: "decay of div B under GLM").
    Eq. 5-6 make (div B, psi) a wave system of speed C_h: without damping sum w|J|(div B)^2 oscillates as
    cos^2(C_h |k| t) (first zero at t = pi/(2 C_h |k|), full recurrence at twice that); with a > 0 the envelope
    decays; with C_h = 0 and a = 0 nothing cleans."""
    n, N = 4, 3
    c_h, k = 1.5, 2 * np.pi
    dt, sub, nsamp = 4e-3, 4, 16
    hist = {}
    for name, ch, a, flags in (("off", 0.0, 0.0, I.FLAG_POWELL), ("glm", c_h, 0.0, I.FLAG_POWELL),
                               ("damped", c_h, 8.0, I.FLAG_POWELL | I.FLAG_GLM_DAMP)):
        phys = I.Physics(c_h=ch, a_psi=a, flags=flags)
        o, x, _ = box_oracle(n, (N, N, N), phys)
        geo = o.geometry()
        one = np.ones_like(x[0])
        B = np.stack([0.3 * one + 0.05 * k * np.cos(k * x[0]) * np.sin(k * x[1]), 0.2 * one + 0.05 * k * np.sin(k * x[0]) * np.cos(k * x[1]), 0.1 * one])
        o.set_state(I.conserved(one, np.zeros_like(B), one, B, 0 * one, GAM))
        h = [_divB2(o, geo, n)]
        for _ in range(nsamp):
            for _ in range(sub):
                o.step(dt, 5)
            h.append(_divB2(o, geo, n))
        hist[name] = np.array(h)
    t = np.arange(nsamp + 1) * dt * sub
    omega = c_h * k * np.sqrt(2.0)
    assert np.abs(hist["off"] / hist["off"][0] - 1).max() < 0.01
    g = hist["glm"] / hist["glm"][0]
    np.testing.assert_allclose(g, np.cos(omega * t) ** 2, atol=0.03)           # pins C_h in the B and psi rows
    d = hist["damped"] / hist["damped"][0]
    half = int(np.ceil(np.pi / (2 * omega) / (dt * sub)))
    assert np.all(np.diff(d[:half]) < 0)                                        # monotone up to the first zero
    assert d[half:].max() < 0.2 and g[half:].max() > 0.9                        # the damped envelope has decayed


def test_p12_mass_conservation_with_impenetrable_walls():
    """Impenetrable walls: the Fejer-quadrature integral of the density residual telescopes to zero, and
    the total mass is unchanged after 10 RK steps (north_star invariant)."""
    w = I.workload("config0")
    n = 4
    m = I.cubed_sphere_shell(3, 2, w.shell.r_b, w.shell.r_t, I.lobatto_abscissae(n + 1))
    o = ob.Oracle(m, n, I.Physics())
    geo = o.geometry()
    Q = I.shell_state(geo["xsol"], w.shell, seed=11, u_amp=0.05, b_amp=0.05)
    o.set_state(Q)
    c_h = o.max_wavespeed()
    phys = I.Physics(GM=1.0, Omega=I.OMEGA_ND, nu=2e-3, kappa=2e-3, eta=2e-3, c_h=c_h, a_psi=c_h / 0.045,
                     flags=I.FLAG_DIFFUSION | I.FLAG_GRAVITY | I.FLAG_CORIOLIS | I.FLAG_POWELL | I.FLAG_GLM_DAMP)
    o.set_physics(phys)
    W = geo["detJ"] * w3(n)[None, :]
    r, a = o.residual(True)
    assert abs((W * r[0]).sum()) <= 1e-12 * (W * a[0]).sum()
    assert np.abs(r[0]).max() > 1e-6                         # the density residual itself is not small
    mass0 = (W * Q[0]).sum()
    for _ in range(10):
        o.step(2e-4, 5)
    Q1 = o.get_state()
    assert np.abs(Q1 - Q).max() > 1e-8
    assert abs((W * Q1[0]).sum() / mass0 - 1) < 1e-13


def test_p16_fp64_roundoff_floor_against_long_double():
    """Distance of the fp64 oracle from its long-double instance in the G24 norm: the floor against which
    the GPU's distance from the oracle is judged (tolerance 1e-12)."""
    w = I.workload("config0")
    n = 6
    m = I.cubed_sphere_shell(2, 2, w.shell.r_b, w.shell.r_t, I.lobatto_abscissae(n + 1))
    od = ob.Oracle(m, n, I.Physics())
    Q = w.state(od.geometry()["xsol"])
    od.set_state(Q)
    c_h = od.max_wavespeed()
    for diff in (0.0, 1e-3):
        phys = I.Workload("t", n, 2, 2, 1.0, 0, diff, shell=w.shell).physics(c_h)
        od.set_physics(phys)
        ol = ob.Oracle(m, n, phys, prec=1)
        ol.set_state(Q)
        rd, ad = od.residual(True)
        rl = ol.residual()
        err = g24_error(rd, rl, ad)
        assert err.max() < 3e-13, err      # dominated by the fp64 curl-form metrics (two derivative passes)
