"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded inputs.

Tolerances (BASELINE.json north_star; norms of DESIGN.md readings G24 / G25):
  residual   max |dR_c| / max A_c  <= 1e-12   (A = the oracle's magnitude residual)
  state      max |dQ_c| / max |Q_c| <= 1e-9    after 10 RK steps
  geometry   <= 1e-12 relative to the array's max (fp64 curl-form metrics; see test_p16 for the floor)
"""
import numpy as np
import pytest

import paper_2502_17805_b200 as P
from paper_2502_17805_b200 import inputs as I
from oracle import binding as ob
from helpers import g24_error, g25_error

pytestmark = pytest.mark.gpu

RES_TOL = 1e-12
STATE_TOL = 1e-9
GEO_TOL = 1e-12


def shell_case(n, nz, nr, N_rho, seed, diff, dipole=True, u_amp=1e-4, b_amp=1e-3, flatten=0.0, extra_flags=0, **phys_kw):
    sh = I.Shell(N_rho=N_rho)
    w = I.Workload("case", n, nz, nr, N_rho, seed, diff, dipole, shell=sh)
    mesh = w.mesh()
    o = ob.Oracle(mesh, n, I.Physics())
    xs = o.geometry()["xsol"]
    Q = I.shell_state(xs, sh, seed, u_amp=u_amp, b_amp=b_amp, dipole=dipole, flatten=flatten)
    o.set_state(Q)
    c_h = o.max_wavespeed()
    phys = w.physics(c_h)
    if extra_flags or phys_kw:
        phys = phys.copy(flags=phys.flags | extra_flags, **phys_kw)
    o.set_physics(phys)
    g = P.Chorus(mesh, n, phys)
    g.set_state(Q)
    return w, mesh, o, g, Q, phys


def check_residual(o, g, tol=RES_TOL):
    r_ref, a_ref = o.residual(True)
    r = g.residual()
    err = g24_error(r, r_ref, a_ref)
    assert np.isfinite(r).all()
    assert err.max() <= tol, err
    return err


def test_geometry_parity_shell_and_box():
    for mesh, n in ((I.cubed_sphere_shell(4, 2, 0.7, 0.95, I.lobatto_abscissae(7)), 6),
                    (I.scrambled_box(2, 2, 2, (1.0, 1.1, 0.9), I.lobatto_abscissae(5), seed=2, distort=0.1), 4),
                    (I.cubed_sphere_shell(2, 1, 0.7, 0.95, I.lobatto_abscissae(4)), 7)):
        go = ob.Oracle(mesh, n, I.Physics()).geometry()
        gg = P.Chorus(mesh, n, I.Physics()).geometry()
        for k in ("detJ", "S", "xsol", "jinv"):
            assert np.abs(gg[k] - go[k]).max() <= GEO_TOL * np.abs(go[k]).max(), k


def test_config0_residual_gradient_wavespeed_parity():
    """BASELINE config 0: 6x4x4x2 shell, n = 6, N_rho = 1, gravity + Coriolis + GLM, diffusion off."""
    w, mesh, o, g, Q, phys = shell_case(6, 4, 2, 1.0, 0, 0.0)
    assert mesh["n_elem"] == 192
    check_residual(o, g)
    assert abs(g.max_wavespeed() / o.max_wavespeed() - 1) < 1e-14
    np.testing.assert_array_equal(g.get_state(), Q)               # set/get round trip is exact
    G_ref = o.gradient()
    G = g.gradient()
    assert np.abs(G - G_ref).max() <= 1e-12 * np.abs(G_ref).max()


def test_config0_ten_rk_stages_and_ten_steps():
    w, mesh, o, g, Q, phys = shell_case(6, 4, 2, 1.0, 0, 0.0)
    _, xf, _, _ = P.get_operators(6)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):                                             # "10 RK stages" = 2 steps of SSPRK(5,3)
        o.step(dt, 5); g.step(dt, 5)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL
    for _ in range(8):                                             # ... and the 10-step state check of north_star
        o.step(dt, 5); g.step(dt, 5)
    q = g.get_state()
    err = g25_error(q, o.get_state(), phys.c_h)
    assert np.isfinite(q).all() and err.max() <= STATE_TOL, err
    assert np.abs(q - Q).max() > 1e-9                              # the state did move
    check_residual(o, g)


def test_full_physics_shell_parity():
    """Config-1 physics (N_rho = 3, nu = kappa = eta = 1e-3, all terms) on a 6x4x4x3 shell."""
    w, mesh, o, g, Q, phys = shell_case(6, 4, 3, 3.0, 1, 1e-3)
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(6)
    for _ in range(10):
        dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
        assert abs(g.max_wavespeed() / o.max_wavespeed() - 1) < 1e-12
        o.step(dt, 5); g.step(dt, 5)
    err = g25_error(g.get_state(), o.get_state(), phys.c_h)
    assert err.max() <= STATE_TOL, err
    check_residual(o, g)


def test_nonequilibrium_input_naive_relative_error():
    """Reading G24, second half: on a non-equilibrium input (perturbations x1000, background flattened) the plain
    relative error max|dR_c| / max|R_c| is itself <= 1e-12 for the variables that evolve."""
    w, mesh, o, g, Q, phys = shell_case(6, 4, 2, 3.0, 5, 1e-3, u_amp=0.1, b_amp=1.0, flatten=0.7)
    r_ref, a_ref = o.residual(True)
    r = g.residual()
    naive = np.abs(r - r_ref).reshape(9, -1).max(1) / np.abs(r_ref).reshape(9, -1).max(1)
    assert naive.max() <= 1e-12, naive
    assert g24_error(r, r_ref, a_ref).max() <= RES_TOL


@pytest.mark.parametrize("wall_opts", [dict(bc_mag_inner=I.BC_RADIAL, bc_mag_outer=I.BC_CONDUCTING),
                                       dict(bc_mag_inner=I.BC_CONDUCTING, bc_mag_outer=I.BC_CONDUCTING),
                                       dict(bc_mag_inner=I.BC_RADIAL, bc_mag_outer=I.BC_RADIAL, T_top=0.05, q_bottom=0.02,
                                            extra_flags=I.FLAG_FIXED_T_OUTER | I.FLAG_FIXED_FLUX_INNER),
                                       dict(bc_mag_inner=I.BC_CONDUCTING, bc_mag_outer=I.BC_RADIAL, kr_scale=2e-3, kr_c=(1.0, -0.5, 0.25),
                                            T_top=0.05, q_bottom=0.02, extra_flags=I.FLAG_FIXED_T_OUTER | I.FLAG_FIXED_FLUX_INNER),
                                       dict(T_top=0.05, q_bottom=0.02, extra_flags=I.FLAG_FIXED_T_OUTER | I.FLAG_FIXED_FLUX_INNER),
                                       dict(extra_flags=I.FLAG_CENTRIFUGAL),
                                       dict(kr_scale=2e-3, kr_c=(1.0, -0.5, 0.25), kr_wscale=1.3)])
def test_wall_and_option_variants_parity(wall_opts):
    kw = dict(wall_opts)
    extra = kw.pop("extra_flags", 0)
    """Both magnetic wall types on each wall, thermal wall options, centrifugal term, kappa_r(r).  The oracle applies the wall
    conditions to the wall gradients literally (Jacobian of B and stress tensor in the spherical frame of the wall point,
    PAPER.md:198, reading G29); the kernels use the closed form those conditions reduce to (DESIGN.md 2)."""
    w, mesh, o, g, Q, phys = shell_case(5, 3, 2, 3.0, 7, 2e-3, u_amp=0.01, b_amp=0.05, extra_flags=extra, **kw)
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(5)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):
        o.step(dt, 5); g.step(dt, 5)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL


def test_all_orientation_codes_parity():
    n = 4
    mesh = I.scrambled_box(3, 3, 3, (1.0, 1.1, 0.9), I.lobatto_abscissae(n + 1), seed=5, distort=0.1)
    for flags in (I.FLAG_POWELL, I.FLAG_POWELL | I.FLAG_DIFFUSION):
        phys = I.Physics(c_h=1.2, nu=0.01, kappa=0.02, eta=0.015, flags=flags)
        o = ob.Oracle(mesh, n, phys)
        g = P.Chorus(mesh, n, phys)
        x = o.geometry()["xsol"]
        rng = np.random.default_rng(3)
        sh = x.shape[1:]
        Q = I.conserved(1 + 0.2 * np.sin(3 * x[0]) + 0.05 * rng.uniform(-1, 1, sh), 0.2 * rng.uniform(-1, 1, (3,) + sh) + 0.1,
                        1 + 0.1 * np.cos(2 * x[1]), 0.3 * rng.uniform(-1, 1, (3,) + sh) + 0.2, 0.1 * rng.uniform(-1, 1, sh), 5 / 3)
        o.set_state(Q); g.set_state(Q)
        check_residual(o, g)
        # free stream on the GPU: uniform static state is preserved to round-off through every orientation
        Q[:] = I.conserved(1.2, np.zeros(3), 1.5, np.zeros(3), np.float64(0.0), 5 / 3)[:, None, None]
        o.set_state(Q); g.set_state(Q)
        _, a = o.residual(True)
        assert np.abs(g.residual()).max() <= 1e-13 * a.max()


@pytest.mark.parametrize("n,diff", [(2, 1e-3), (3, 1e-3), (4, 1e-3), (5, 1e-3), (6, 1e-3), (7, 0.0), (7, 1e-3), (8, 0.0),
                                    (8, 1e-3), (9, 0.0), (9, 1e-3)])
def test_order_sweep_parity(n, diff):
    """BASELINE config 4 (order sweep), at sizes the oracle finishes in seconds."""
    w, mesh, o, g, Q, phys = shell_case(n, 3, 2, 3.0, 4, diff)
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):
        o.step(dt, 5); g.step(dt, 5)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL


@pytest.mark.parametrize("n,diff", [(4, 1e-3), (4, 0.0), (5, 1e-3), (5, 0.0), (6, 1e-3), (6, 0.0), (7, 1e-3), (7, 0.0), (8, 1e-3), (8, 0.0)])
def test_persistent_loop_parity(n, diff):
    """Meshes with more elements (6x8x8x2 = 768) than the element kernel's grid (2 CTAs x 148 SMs, 1 x 148 at n = 7), so that
    every CTA runs its persistent loop several times -- barrier phases, bulk copies into live shared memory, tail-task rotation,
    the new state passing through sQ for its traces -- in RESIDUAL and in STEP mode, against the whole-mesh oracle."""
    w, mesh, o, g, Q, phys = shell_case(n, 8, 2, 3.0, 12, diff)
    assert mesh["n_elem"] == 768
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):
        o.step(dt, 5); g.step(dt, 5)
    err = g25_error(g.get_state(), o.get_state(), phys.c_h)
    assert err.max() <= STATE_TOL, err
    check_residual(o, g)


@pytest.mark.parametrize("nstages", [1, 3])
def test_other_rk_schemes_parity(nstages):
    w, mesh, o, g, Q, phys = shell_case(4, 3, 2, 1.0, 9, 1e-3)
    _, xf, _, _ = P.get_operators(4)
    dt = 0.5 * w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(3):
        o.step(dt, nstages); g.step(dt, nstages)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL


def test_device_pointers_and_streams():
    import torch
    w, mesh, o, g, Q, phys = shell_case(4, 3, 2, 1.0, 9, 1e-3)
    qd = torch.from_numpy(Q).cuda()
    g.set_state(qd)
    r_dev = g.residual(device=True)
    r_host = g.residual()
    torch.cuda.synchronize()
    np.testing.assert_array_equal(r_dev.cpu().numpy(), r_host)
    np.testing.assert_array_equal(g.get_state(device=True).cpu().numpy(), Q)
    n0 = g.launch_count()
    g.step(1e-4, 5)
    assert g.launch_count() - n0 == 10            # main kernel + viscous face kernel per stage (traces are emitted by the face kernel)


def test_error_paths():
    mesh = I.periodic_box(2, 1, 1, (1, 1, 1), I.lobatto_abscissae(4))
    g = P.Chorus(mesh, 3, I.Physics(c_h=1.0))
    with pytest.raises(P.ChorusError) as ei:
        g.residual()
    assert ei.value.code == -4                    # CHORUS_ESTATE: no state set
    with pytest.raises(P.ChorusError):
        g.step(1e-3, 4)                           # unsupported stage count
    with pytest.raises(P.ChorusError):
        P.Chorus(mesh, 10, I.Physics())
    bad = dict(mesh); bad["nbr_elem"] = mesh["nbr_elem"].copy(); bad["nbr_elem"][0, 0] = 99
    with pytest.raises(P.ChorusError):
        P.Chorus(bad, 3, I.Physics())
    Q = np.zeros(g.shape); Q[0] = 1.0; Q[4] = np.nan
    g.set_state(Q)
    with pytest.raises(P.ChorusError) as ei:
        g.max_wavespeed()
    assert ei.value.code == -4                    # non-finite wave speed


def test_empty_and_single_element_edge_cases():
    mesh = I.periodic_box(1, 1, 1, (1, 1, 1), I.lobatto_abscissae(3))       # one element, its own neighbour
    phys = I.Physics(c_h=1.0, nu=0.01, kappa=0.01, eta=0.01, flags=I.FLAG_DIFFUSION | I.FLAG_POWELL)
    o, g = ob.Oracle(mesh, 3, phys), P.Chorus(mesh, 3, phys)
    x = o.geometry()["xsol"]
    Q = I.conserved(1 + 0.1 * np.sin(2 * np.pi * x[0]), 0.1 * np.stack([np.cos(2 * np.pi * x[1])] * 3), 1 + 0 * x[0],
                    0.2 * np.stack([np.sin(2 * np.pi * x[2])] * 3), 0 * x[0], 5 / 3)
    o.set_state(Q); g.set_state(Q)
    check_residual(o, g)
    empty = dict(mesh); empty["n_elem"] = 0
    with pytest.raises(P.ChorusError):
        P.Chorus(empty, 3, phys)


@pytest.mark.parametrize("n,diff", [(6, 1e-3), (6, 0.0), (5, 1e-3), (4, 1e-3), (7, 1e-3), (8, 1e-3)])
def test_bitwise_reproducible_across_launches(n, diff):
    """The element kernel is warp-specialised (chain and helper warps hand shared memory to each other through named
    barriers) and has no atomics on its data path: repeated launches must agree bit for bit.  A missing barrier shows up
    here as run-to-run differences (compute-sanitizer is not available on the GPU pool)."""
    w, mesh, o, g, Q, phys = shell_case(n, 6, 3, 3.0, 8, diff)
    r0 = g.residual()
    for _ in range(15):
        np.testing.assert_array_equal(g.residual(), r0)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    finals = []
    for _ in range(3):
        g.set_state(Q)
        for _ in range(3):
            g.step(dt, 5)
        finals.append(g.get_state())
    np.testing.assert_array_equal(finals[0], finals[1])
    np.testing.assert_array_equal(finals[0], finals[2])


def test_diagnostics_parity_and_reproducibility():
    """chorus_diagnostics (V, KE of Eq. 34, E_B of Eq. 35) against the oracle's literal long-double sums, on a small and on a
    768-element shell, before and after a step; the tree reduction has no atomics: bit-identical from call to call."""
    for nz, nr, n in ((4, 2, 6), (8, 2, 5)):
        w, mesh, o, g, Q, phys = shell_case(n, nz, nr, 3.0, 21, 1e-3, u_amp=0.05, b_amp=0.2)
        for it in range(2):
            d, d_ref = g.diagnostics(), o.diagnostics()
            for k in ("V", "KE", "EB"):
                assert abs(d[k] / d_ref[k] - 1) <= 1e-13, (k, d[k], d_ref[k])
            assert g.diagnostics() == d
            _, xf, _, _ = P.get_operators(n)
            dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
            o.step(dt, 5); g.step(dt, 5)
    g2 = P.Chorus(mesh, n, phys)
    with pytest.raises(P.ChorusError) as ei:
        g2.diagnostics()
    assert ei.value.code == -4


@pytest.mark.parametrize("obl", [0.1, 0.3])
def test_oblate_shell_geometry_and_residual_parity(obl):
    """Oblate shells through the generic geometry-node input: metrics, residual with all terms, two steps."""
    n = 6
    sh = I.Shell(N_rho=3.0)
    w = I.Workload("oblate", n, 4, 2, 3.0, 13, 1e-3, True, shell=sh)
    mesh = I.cubed_sphere_shell(4, 2, sh.r_b, sh.r_t, I.lobatto_abscissae(n + 1), oblateness=obl)
    o = ob.Oracle(mesh, n, I.Physics())
    go = o.geometry()
    Q = I.shell_state(go["xsol"], sh, 13, u_amp=0.01, b_amp=0.05)
    o.set_state(Q)
    phys = w.physics(o.max_wavespeed())
    o.set_physics(phys)
    g = P.Chorus(mesh, n, phys)
    gg = g.geometry()
    for k in ("detJ", "S", "xsol", "jinv"):
        assert np.abs(gg[k] - go[k]).max() <= GEO_TOL * np.abs(go[k]).max(), k
    g.set_state(Q)
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):
        o.step(dt, 5); g.step(dt, 5)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL
    # free stream on the GPU: a uniform static state is preserved to round-off on the oblate mesh
    g.set_physics(phys.copy(flags=I.FLAG_DIFFUSION))
    o.set_physics(phys.copy(flags=I.FLAG_DIFFUSION))
    U = np.empty_like(Q)
    U[:] = I.conserved(1.2, np.zeros(3), 1.5, np.zeros(3), np.float64(0.0), 5 / 3)[:, None, None]
    g.set_state(U); o.set_state(U)
    _, a = o.residual(True)
    assert np.abs(g.residual()).max() <= 1e-12 * a.max()


def test_gpu_against_long_double_oracle():
    """The kernels against the oracle's long-double instance (P16 measures the fp64 oracle's own distance from it): the CUDA
    path is no further from the extended-precision result than the tolerance allows, so the 1e-12 bar is not met by sharing
    the fp64 oracle's rounding."""
    n = 6
    for diff in (0.0, 1e-3):
        w, mesh, o, g, Q, phys = shell_case(n, 2, 2, 3.0, 5, diff)
        ol = ob.Oracle(mesh, n, phys, prec=1)
        ol.set_state(Q)
        rl = ol.residual()
        rd, ad = o.residual(True)
        e_gpu = g24_error(g.residual(), rl, ad)
        e_cpu = g24_error(rd, rl, ad)
        assert e_gpu.max() <= RES_TOL, e_gpu
        assert e_gpu.max() <= 10 * max(e_cpu.max(), 1e-14), (e_gpu, e_cpu)     # same order as the fp64 oracle's own floor


def test_flux_balanced_background_with_radiative_profile_parity():
    """The solar-type set-up of PAPER.md:169-186, :216: the state built on the flux-balanced stratification (Eq. 28-31) with the
    radiative diffusivity profile kappa_r(r) and a bottom heat flux; residual, and two steps."""
    n = 6
    sh = I.Shell(N_rho=3.0)
    kr_scale, kr_c, kr_w = 1e-5, (1.0, -0.8, 0.6), 1.7
    kr = lambda r: kr_scale * (kr_c[0] + kr_c[1] * (kr_w * r) + kr_c[2] * (kr_w * r) ** 2)
    L = 2e-5
    prof = I.flux_balanced_profile(sh, L, 2e-3, kr, n_grid=2001)
    w = I.Workload("solar", n, 4, 3, 3.0, 17, 2e-3, True, shell=sh)
    mesh = w.mesh()
    o = ob.Oracle(mesh, n, I.Physics())
    Q = I.shell_state(o.geometry()["xsol"], sh, 17, u_amp=1e-3, b_amp=1e-2, background=prof)
    o.set_state(Q)
    phys = w.physics(o.max_wavespeed()).copy(kr_scale=kr_scale, kr_c=kr_c, kr_wscale=kr_w,
                                             q_bottom=L / (4 * np.pi * sh.r_b ** 2))
    o.set_physics(phys)
    g = P.Chorus(mesh, n, phys)
    g.set_state(Q)
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):
        o.step(dt, 5); g.step(dt, 5)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL
    # the radiative term matters in this case: without it the residual differs far above the tolerance
    o.set_physics(phys.copy(kr_scale=0.0))
    r0, a0 = o.residual(True)
    o.set_physics(phys)
    r1, _ = o.residual(True)
    assert g24_error(r1, r0, a0).max() > 1e-6


@pytest.mark.parametrize("wall_opts", [dict(bc_mag_inner=I.BC_RADIAL, bc_mag_outer=I.BC_CONDUCTING, kr_scale=2e-3, kr_c=(1.0, -0.5, 0.25),
                                            kr_wscale=1.3, T_top=0.05, q_bottom=0.02,
                                            extra_flags=I.FLAG_FIXED_T_OUTER | I.FLAG_FIXED_FLUX_INNER | I.FLAG_CENTRIFUGAL),
                                       dict(bc_mag_inner=I.BC_CONDUCTING, bc_mag_outer=I.BC_RADIAL)])
def test_order8_walls_and_orientations_parity(wall_opts):
    """n = 8 on the DMMA pipeline: its tiles hold the interior flux points and the face point m = n; the face point m = 0 goes
    through the helper warps (own-side viscous flux) and a third k-step (flux derivative).  Both wall types on both walls with
    the thermal options and kappa_r(r), and every face orientation of a scrambled box with diffusion."""
    kw = dict(wall_opts)
    extra = kw.pop("extra_flags", 0)
    w, mesh, o, g, Q, phys = shell_case(8, 3, 2, 3.0, 7, 2e-3, u_amp=0.01, b_amp=0.05, extra_flags=extra, **kw)
    check_residual(o, g)
    _, xf, _, _ = P.get_operators(8)
    dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
    for _ in range(2):
        o.step(dt, 5); g.step(dt, 5)
    assert g25_error(g.get_state(), o.get_state(), phys.c_h).max() <= STATE_TOL
    n = 8
    mesh = I.scrambled_box(2, 2, 3, (1.0, 1.1, 0.9), I.lobatto_abscissae(n + 1), seed=8, distort=0.1)
    physb = I.Physics(c_h=1.2, nu=0.01, kappa=0.02, eta=0.015, flags=I.FLAG_POWELL | I.FLAG_DIFFUSION)
    o, g = ob.Oracle(mesh, n, physb), P.Chorus(mesh, n, physb)
    x = o.geometry()["xsol"]
    rng = np.random.default_rng(3)
    sh = x.shape[1:]
    Q = I.conserved(1 + 0.2 * np.sin(3 * x[0]) + 0.05 * rng.uniform(-1, 1, sh), 0.2 * rng.uniform(-1, 1, (3,) + sh) + 0.1,
                    1 + 0.1 * np.cos(2 * x[1]), 0.3 * rng.uniform(-1, 1, (3,) + sh) + 0.2, 0.1 * rng.uniform(-1, 1, sh), 5 / 3)
    o.set_state(Q); g.set_state(Q)
    check_residual(o, g)
    Q[:] = I.conserved(1.2, np.zeros(3), 1.5, np.zeros(3), np.float64(0.0), 5 / 3)[:, None, None]
    o.set_state(Q); g.set_state(Q)
    _, a = o.residual(True)
    assert np.abs(g.residual()).max() <= 1e-13 * a.max()
