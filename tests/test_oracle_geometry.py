"""Pins P3, P4: mesh generator counts; metrics of the oracle against free-stream preservation, closed-form
volume / area of the spherical shell, and face consistency between neighbours."""
import collections

import numpy as np
import pytest

from oracle import binding as ob
from paper_2502_17805_b200 import inputs as I
from helpers import fejer1_weights, w3

RB, RT = 0.70, 0.95


@pytest.mark.parametrize("nz,nr", [(4, 2), (3, 3)])
def test_p4_shell_mesh_counts_and_connectivity(nz, nr):
    m = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(3))
    E = m["n_elem"]
    assert E == 6 * nr * nz * nz
    ne, nf, no = m["nbr_elem"], m["nbr_face"], m["nbr_orient"]
    assert (ne >= 0).sum() == 2 * (3 * E - 6 * nz * nz)                  # interior faces, counted from both sides
    assert (ne == -1).sum() == 6 * nz * nz and (ne == -2).sum() == 6 * nz * nz
    for e in range(E):
        for f in range(6):
            if ne[e, f] >= 0:
                assert ne[ne[e, f], nf[e, f]] == e and nf[ne[e, f], nf[e, f]] == f
    # walls are the zeta faces; only "identity" and "reverse a" orientations occur on this mesh
    assert set(np.argwhere(ne < 0)[:, 1]) == {4, 5}
    assert set(no[ne >= 0].tolist()) <= {0, 2}
    # right-handed elements: corner triple product > 0
    X = m["xyz"].reshape(E, 3, 3, 3, 3)       # [E,comp,c,b,a]
    d1 = X[:, :, 0, 0, 2] - X[:, :, 0, 0, 0]; d2 = X[:, :, 0, 2, 0] - X[:, :, 0, 0, 0]; d3 = X[:, :, 2, 0, 0] - X[:, :, 0, 0, 0]
    assert np.einsum("ei,ei->e", np.cross(d1, d2), d3).min() > 0


def test_p4_orientation_codes_all_eight():
    """The generic 3-bit code: a randomly re-oriented neighbour is recovered by hex_connectivity."""
    g = np.array([0.0, 1.0])
    A, B, C = np.meshgrid(g, g, g, indexing="ij")
    base = np.stack([A, B, C])                                  # [3,xi,eta,zeta]
    seen = set()
    for perm in [(0, 1, 2), (1, 0, 2), (0, 2, 1), (2, 1, 0), (1, 2, 0), (2, 0, 1)]:
        for flips in range(8):
            c2 = base.copy(); c2[0] += 1.0                      # neighbour occupies [1,2]x[0,1]x[0,1]
            c2 = np.transpose(c2, (0,) + tuple(1 + p for p in perm))
            for ax in range(3):
                if flips >> ax & 1:
                    c2 = np.flip(c2, axis=1 + ax)
            corners = np.stack([base, c2])
            try:
                ne, nf, no = I.hex_connectivity(corners)
            except ValueError:
                continue
            f = 1
            assert ne[0, f] == 1
            code, f2 = int(no[0, f]), int(nf[0, f])
            seen.add(code)
            P1 = np.take(corners[0], 1, axis=1)
            P2 = np.take(corners[1], f2 % 2, axis=1 + f2 // 2)
            for a in range(2):
                for b in range(2):
                    a2, b2 = I.orient_map(code, a, b, 2)
                    np.testing.assert_allclose(P1[:, a, b], P2[:, a2, b2], atol=1e-12)
    assert seen == set(range(8))


@pytest.mark.parametrize("n,nz,nr", [(6, 4, 3), (4, 3, 3)])
def test_p3_freestream_on_curved_shell(n, nz, nr):
    """Uniform state, sources off => residual at round-off (north_star invariant)."""
    m = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(n + 1))
    o = ob.Oracle(m, n, I.Physics(c_h=1.0, flags=0))
    E = m["n_elem"]
    Q = np.zeros((9, E, n ** 3))
    Q[:] = I.conserved(1.0, np.zeros(3), 1.5, np.zeros(3), np.float64(0.0), 5 / 3)[:, None, None]
    o.set_state(Q)
    r, a = o.residual(True)
    assert np.abs(r).max() <= 1e-12 * a.max()                   # U = 0: walls are compatible, every element checked
    Q[:] = I.conserved(1.0, np.array([0.3, -0.2, 0.1]), 1.5, np.array([0.5, 0.25, -0.4]), np.float64(0.1), 5 / 3)[:, None, None]
    o.set_state(Q)
    r, a = o.residual(True)
    mid = (np.arange(E) // (nz * nz)) % nr == 1                 # elements not touching a wall
    assert np.abs(r[:, mid]).max() <= 1e-12 * a[:, mid].max()
    assert np.abs(r[:, ~mid]).max() > 1e-3 * a.max()            # the wall really acts on a non-tangent flow


@pytest.mark.parametrize("diff", [False, True])
def test_p3_freestream_on_curvilinear_periodic_box(diff):
    n = 5
    m = I.periodic_box(3, 2, 2, (1.0, 0.8, 1.2), I.lobatto_abscissae(n + 1), distort=0.15)
    flags = I.FLAG_DIFFUSION if diff else 0
    o = ob.Oracle(m, n, I.Physics(c_h=0.8, nu=0.01, kappa=0.02, eta=0.03, flags=flags))
    geo = o.geometry()
    assert geo["detJ"].min() > 0
    Q = np.zeros(o.shape)
    Q[:] = I.conserved(1.2, np.array([0.3, -0.2, 0.1]), 1.5, np.array([0.5, 0.25, -0.4]), np.float64(0.1), 5 / 3)[:, None, None]
    o.set_state(Q)
    r, a = o.residual(True)
    assert np.abs(r).max() <= 1e-12 * a.max()
    assert np.abs(o.gradient()).max() < 1e-11


@pytest.mark.parametrize("n,tol", [(4, 1e-5), (6, 1e-8), (8, 1e-11)])
def test_p3_shell_volume_and_wall_area_closed_forms(n, tol):
    nz, nr = 4, 2
    m = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(n + 1))
    o = ob.Oracle(m, n, I.Physics())
    geo = o.geometry()
    vol = (geo["detJ"] * w3(n)[None, :]).sum()
    assert abs(vol / (4 * np.pi / 3 * (RT ** 3 - RB ** 3)) - 1) < tol
    w = fejer1_weights(n)
    w2 = (w[:, None] * w[None, :]).reshape(-1)                  # face index b*n+a
    S = geo["S"]                                                # [E,3 fam,3 comp,nf]; zeta family index (m*n+b)*n+a
    inner = np.argwhere(m["nbr_elem"][:, 4] == -1)[:, 0]
    outer = np.argwhere(m["nbr_elem"][:, 5] == -2)[:, 0]
    Sin = S[inner, 2][:, :, : n * n]                            # m = 0
    Sout = S[outer, 2][:, :, n * n * n:]                        # m = n
    area_in = (np.sqrt((Sin ** 2).sum(1)) * w2[None, :]).sum()
    area_out = (np.sqrt((Sout ** 2).sum(1)) * w2[None, :]).sum()
    assert abs(area_in / (4 * np.pi * RB ** 2) - 1) < tol
    assert abs(area_out / (4 * np.pi * RT ** 2) - 1) < tol
    # solution-point coordinates lie in the shell, and the outward wall normals are radial
    r = np.sqrt((geo["xsol"] ** 2).sum(0))
    assert r.min() > RB and r.max() < RT


def test_p3_face_metrics_match_across_faces_and_seams():
    n, nz, nr = 5, 3, 2
    m = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(n + 1))
    o = ob.Oracle(m, n, I.Physics())
    S = o.geometry()["S"]
    N1 = n + 1

    def fidx(d, mm, a, b):
        return [(b * n + a) * N1 + mm, (b * N1 + mm) * n + a, (mm * n + b) * n + a][d]
    worst = 0.0
    kinds = collections.Counter()
    for e in range(m["n_elem"]):
        for f in range(6):
            ne = m["nbr_elem"][e, f]
            if ne < 0:
                continue
            f2, code = int(m["nbr_face"][e, f]), int(m["nbr_orient"][e, f])
            kinds[(f, f2, code)] += 1
            for a in range(n):
                for b in range(n):
                    a2, b2 = I.orient_map(code, a, b, n)
                    s1 = S[e, f // 2, :, fidx(f // 2, n if f & 1 else 0, a, b)] * (1 if f & 1 else -1)
                    s2 = S[ne, f2 // 2, :, fidx(f2 // 2, n if f2 & 1 else 0, a2, b2)] * (1 if f2 & 1 else -1)
                    worst = max(worst, np.abs(s1 + s2).max() / np.abs(s1).max())     # outward area vectors opposite
    assert worst < 1e-12
    assert len(kinds) >= 10          # several distinct seam pairings were exercised


def test_p3_geometry_independent_of_geometry_node_set():
    """The metrics depend on the map, not on which abscissae the mesh file samples (both are degree-n exact
    representations only for polynomial maps, so use a polynomial-mapped box)."""
    n = 4
    xs, xf = ob.nodes(n)
    mA = I.periodic_box(2, 2, 2, (1, 1, 1), I.lobatto_abscissae(n + 1))
    mB = I.periodic_box(2, 2, 2, (1, 1, 1), xf)
    gA = ob.Oracle(mA, n, I.Physics()).geometry()
    gB = ob.Oracle(mB, n, I.Physics()).geometry()
    for k in ("detJ", "S", "xsol", "jinv"):
        np.testing.assert_allclose(gA[k], gB[k], atol=1e-13)
    np.testing.assert_allclose(gA["detJ"], 0.125, atol=1e-14)
    np.testing.assert_allclose(gA["jinv"][:, 0, 0], 2.0, atol=1e-13)


def test_p3_freestream_through_every_orientation_code():
    """Walled box whose elements carry random local-axis rotations: all 8 orientation codes and xi/eta/zeta face
    pairings occur; the uniform-state residual of the interior element stays at round-off (inviscid), and a static
    uniform state is preserved everywhere including the walls."""
    n = 4
    m = I.scrambled_box(3, 3, 3, (1.0, 1.1, 0.9), I.lobatto_abscissae(n + 1), seed=5, distort=0.1)
    assert set(m["nbr_orient"][m["nbr_elem"] >= 0].tolist()) == set(range(8))
    o = ob.Oracle(m, n, I.Physics(c_h=1.0, flags=0))
    assert o.geometry()["detJ"].min() > 0
    Q = np.zeros(o.shape)
    Q[:] = I.conserved(1.2, np.array([0.3, -0.2, 0.1]), 1.5, np.array([0.5, 0.25, -0.4]), np.float64(0.1), 5 / 3)[:, None, None]
    o.set_state(Q)
    r, a = o.residual(True)
    assert np.abs(r[:, 13]).max() <= 1e-13 * a.max()
    Q[:] = I.conserved(1.2, np.zeros(3), 1.5, np.zeros(3), np.float64(0.0), 5 / 3)[:, None, None]
    o.set_state(Q)
    r, a = o.residual(True)
    assert np.abs(r).max() <= 1e-13 * a.max()


# ------------------------------------------------------------------------------- oblate shells
@pytest.mark.parametrize("n,obl", [(6, 0.1), (4, 0.25)])
def test_p3_oblate_shell_freestream_and_volume(n, obl):
    """"It is also possible to generate oblate meshes": the z axis of the shell scaled by 1 - e.  The map is no
    longer radial, so nothing of the spherical closed form of the metrics survives -- but the curl-form metrics still preserve
    a free stream to round-off, the mesh stays right-handed, and the volume is exactly (1 - e) times the spherical one."""
    nz, nr = 4, 3
    m = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(n + 1), oblateness=obl)
    ms = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(n + 1))
    np.testing.assert_array_equal(m["nbr_elem"], ms["nbr_elem"])          # same topology
    np.testing.assert_allclose(m["xyz"][:, 2], (1 - obl) * ms["xyz"][:, 2], rtol=1e-15)
    o = ob.Oracle(m, n, I.Physics(c_h=1.0, flags=0))
    geo, geo_s = o.geometry(), ob.Oracle(ms, n, I.Physics()).geometry()
    assert geo["detJ"].min() > 0
    E = m["n_elem"]
    Q = np.zeros((9, E, n ** 3))
    Q[:] = I.conserved(1.0, np.array([0.3, -0.2, 0.1]), 1.5, np.array([0.5, 0.25, -0.4]), np.float64(0.1), 5 / 3)[:, None, None]
    o.set_state(Q)
    r, a = o.residual(True)
    mid = (np.arange(E) // (nz * nz)) % nr == 1                 # elements not touching a wall
    assert np.abs(r[:, mid]).max() <= 1e-12 * a[:, mid].max()
    assert np.abs(o.gradient()[:, mid]).max() < 1e-11
    # |J| = (1 - e) |J|_sphere point by point (the map is the spherical one followed by a linear stretch), hence the volume
    np.testing.assert_allclose(geo["detJ"], (1 - obl) * geo_s["detJ"], rtol=1e-11)
    vol = (geo["detJ"] * w3(n)[None, :]).sum()
    assert abs(vol / ((1 - obl) * 4 * np.pi / 3 * (RT ** 3 - RB ** 3)) - 1) < (1e-8 if n == 6 else 1e-5)
    # the area vectors transform with the cofactor of diag(1, 1, 1 - e): (S_x, S_y, S_z) = ((1-e) S_x, (1-e) S_y, S_z)_sphere
    np.testing.assert_allclose(geo["S"][:, :, 0], (1 - obl) * geo_s["S"][:, :, 0], rtol=0, atol=1e-12 * np.abs(geo_s["S"]).max())
    np.testing.assert_allclose(geo["S"][:, :, 2], geo_s["S"][:, :, 2], rtol=0, atol=1e-12 * np.abs(geo_s["S"]).max())


# ------------------------------------------------------------------------------- volume integrals (Eq. 34-35)
def test_quadrature_weights_closed_form_exactness_and_telescoping():
    """w_i = int_0^1 h_i (the oracle integrates the Lagrange basis of Eq. 19 with a Gauss rule): equal to Fejer's first rule in
    closed form, exact for x^k, k <= n-1, and sum_i w_i l'_m(X_s,i) = delta_{m,n} - delta_{m,0} (the telescoping
    identity behind mass conservation, pin P12)."""
    for n in range(2, 10):
        w = ob.quadrature_weights(n)
        np.testing.assert_allclose(w, fejer1_weights(n), rtol=0, atol=2e-16)
        xs, _ = ob.nodes(n)
        for k in range(n):
            assert abs(w @ xs ** k - 1.0 / (k + 1)) < 1e-15
        assert abs(w @ xs ** (n + 1) - 1.0 / (n + 2)) > 1e-9 or n % 2 == 1     # and not beyond its degree (symmetric rules gain one)
        _, Dfs, _, _ = ob.operators(n)
        tel = w @ Dfs
        ref = np.zeros(n + 1); ref[0], ref[n] = -1.0, 1.0
        np.testing.assert_allclose(tel, ref, rtol=0, atol=1e-13)


def test_diagnostics_closed_forms_on_the_shell():
    """KE and E_B of Eq. 34-35 for fields with closed forms on the spherical shell: rigid rotation of a uniform-density fluid,
    int (x^2 + y^2) dV = (2/3) 4 pi (r_t^5 - r_b^5)/5; a uniform field (E_B = |B|^2/2 exactly, whatever V); |B| = r."""
    n, nz, nr = 6, 4, 2
    m = I.cubed_sphere_shell(nz, nr, RB, RT, I.lobatto_abscissae(n + 1))
    o = ob.Oracle(m, n, I.Physics())
    x = o.geometry()["xsol"]
    V_ref = 4 * np.pi / 3 * (RT ** 3 - RB ** 3)
    I5 = 4 * np.pi * (RT ** 5 - RB ** 5) / 5                    # int r^2 dV
    rho0, Om = 1.7, 0.4
    one = np.ones_like(x[0])
    U = np.stack([-Om * x[1], Om * x[0], 0 * one])
    B0 = np.array([0.3, -0.2, 0.5])
    o.set_state(I.conserved(rho0 * one, U, one, B0[:, None, None] * one, 0 * one, 5 / 3))
    d = o.diagnostics()
    assert abs(d["V"] / V_ref - 1) < 1e-8
    assert abs(d["KE"] / (0.5 * rho0 * Om ** 2 * (2 / 3) * I5 / V_ref) - 1) < 1e-7
    assert abs(d["EB"] / (0.5 * B0 @ B0) - 1) < 1e-14
    o.set_state(I.conserved(rho0 * one, 0 * U, one, x, 0 * one, 5 / 3))           # B = x, |B| = r
    d = o.diagnostics()
    assert d["KE"] == 0.0 and abs(d["EB"] / (0.5 * I5 / V_ref) - 1) < 1e-7
