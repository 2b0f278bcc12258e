"""Pins P1, P2, P13: node sets, 1-D operators and the RK tableau of the oracle against what the paper
and the mathematics fix (closed forms, a worked example, numpy's Gauss-Legendre, order conditions)."""
import os

import numpy as np
import pytest

from oracle import binding as ob

GOLD = os.path.join(os.path.dirname(__file__), "golden")
ORDERS = list(range(2, 10))


def _golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        out[k] = v
    return out


def test_p1_worked_example_order3():
    g = _golden("nodes_order3.txt")
    xs, xf = ob.nodes(3)
    np.testing.assert_allclose(xs, np.array(g["xs"], float), atol=2e-16, rtol=0)
    np.testing.assert_allclose(xf, np.array(g["xf"], float), atol=2e-16, rtol=0)


@pytest.mark.parametrize("n", ORDERS)
def test_p1_nodes_closed_forms(n):
    xs, xf = ob.nodes(n)
    k = np.arange(1, n + 1)
    np.testing.assert_allclose(xs, 0.5 * (1 - np.cos((2 * k - 1) * np.pi / (2 * n))), atol=1e-15)     # Eq. 18
    assert xf.size == n + 1 and xf[0] == 0.0 and xf[-1] == 1.0
    gl, _ = np.polynomial.legendre.leggauss(n - 1)                                                       # roots of P_{n-1}
    np.testing.assert_allclose(xf[1:-1], 0.5 * (1 + gl), atol=1e-15)
    np.testing.assert_allclose(xs + xs[::-1], 1.0, atol=1e-15)                                           # symmetry X -> 1-X
    np.testing.assert_allclose(xf + xf[::-1], 1.0, atol=1e-15)
    assert np.all(np.diff(xs) > 0) and np.all(np.diff(xf) > 0)


@pytest.mark.parametrize("n", ORDERS)
def test_p2_operators_polynomial_exactness(n):
    xs, xf = ob.nodes(n)
    Isf, Dfs, Efs, Dff = ob.operators(n)
    np.testing.assert_allclose(Isf.sum(1), 1.0, atol=1e-13)
    np.testing.assert_allclose(Efs.sum(1), 1.0, atol=1e-13)
    np.testing.assert_allclose(Dfs.sum(1), 0.0, atol=1e-11)
    np.testing.assert_allclose(Dff.sum(1), 0.0, atol=1e-11)
    for deg in range(n + 1):
        c = np.zeros(deg + 1); c[deg] = 1.0
        p = np.polynomial.Polynomial(c)
        if deg <= n - 1:      # solution polynomial has degree n-1 (Eq. 19)
            np.testing.assert_allclose(Isf @ p(xs), p(xf), atol=1e-12)
        # flux polynomial has degree n (Eq. 20): evaluation and derivative exact
        np.testing.assert_allclose(Efs @ p(xf), p(xs), atol=1e-12)
        np.testing.assert_allclose(Dfs @ p(xf), p.deriv()(xs), atol=2e-11)
        np.testing.assert_allclose(Dff @ p(xf), p.deriv()(xf), atol=2e-11)
    # north_star: "exact derivatives of polynomials of degree at most N-1" through interpolate -> differentiate
    for deg in range(n):
        c = np.zeros(deg + 1); c[deg] = 1.0
        p = np.polynomial.Polynomial(c)
        np.testing.assert_allclose(Dfs @ (Isf @ p(xs)), p.deriv()(xs), atol=2e-11)
    # a degree-(n+1) monomial must NOT be differentiated exactly (the operator really is degree n)
    p = np.polynomial.Polynomial([0] * (n + 1) + [1.0])
    assert np.abs(Dfs @ p(xf) - p.deriv()(xs)).max() > 1e-8


def test_p2_operators_are_not_transposed():
    n = 4
    xs, xf = ob.nodes(n)
    Isf, Dfs, Efs, Dff = ob.operators(n)
    assert Isf.shape == (n + 1, n) and Dfs.shape == (n, n + 1)
    # h_i(X_f,m) at the end point X_f = 0: extrapolation weights alternate in sign and the first dominates
    assert Isf[0, 0] > 1.0 and Isf[0, 1] < 0.0
    # l'_m(X_s,i): derivative of the first flux basis function is negative near xi = 0
    assert Dfs[0, 0] < 0.0 and Dfs[-1, -1] > 0.0


def _butcher(alpha, beta, s):
    K = np.zeros((s + 1, s))
    for i in range(1, s + 1):
        for k in range(i):
            K[i] += alpha[i - 1, k] * K[k]
            K[i, k] += beta[i - 1, k]
    A, b = K[:s], K[s]
    return A, b, A.sum(1)


def test_p13_ssprk53_order_conditions_and_ssp_coefficient():
    al, be = ob.rk_tableau(5)
    np.testing.assert_allclose(al.sum(1), 1.0, atol=1e-13)              # consistency of each stage
    A, b, c = _butcher(al, be, 5)
    assert abs(b.sum() - 1) < 1e-9 and abs(b @ c - 0.5) < 1e-9          # orders 1, 2
    assert abs(b @ c ** 2 - 1 / 3) < 1e-9 and abs(b @ A @ c - 1 / 6) < 1e-9   # order 3
    assert abs(b @ c ** 3 - 0.25) > 1e-3                                # third order only
    assert (al >= 0).all() and (be >= 0).all()
    m = be > 0
    assert not ((al == 0) & m).any()
    ssp = np.min(al[m] / be[m])
    assert abs(ssp - 2.65062919) < 1e-6                                 # Ruuth's optimal SSPRK(5,3) coefficient


def test_p13_ssprk33_and_euler_tableaux():
    al, be = ob.rk_tableau(3)
    A, b, c = _butcher(al[:3, :3], be[:3, :3], 3)
    np.testing.assert_allclose(b, [1 / 6, 1 / 6, 2 / 3], atol=1e-15)
    np.testing.assert_allclose(c, [0, 1, 0.5], atol=1e-15)
    al, be = ob.rk_tableau(1)
    assert al[0, 0] == 1.0 and be[0, 0] == 1.0


@pytest.mark.parametrize("s,order", [(5, 3), (3, 3), (1, 1)])
def test_p13_observed_order_on_scalar_ode(s, order):
    al, be = ob.rk_tableau(s)

    def integrate(dt, nsteps):
        y = 1.0
        for _ in range(nsteps):
            u = [y]
            for i in range(1, s + 1):
                u.append(sum(al[i - 1, k] * u[k] + dt * be[i - 1, k] * (-u[k]) for k in range(i)))
            y = u[-1]
        return y
    e1 = abs(integrate(0.1, 10) - np.exp(-1.0))
    e2 = abs(integrate(0.05, 20) - np.exp(-1.0))
    assert abs(np.log2(e1 / e2) - order) < 0.15


def test_paper_counts():
    for line in open(os.path.join(GOLD, "paper_counts.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, nr, nz, order, ncells, ndof = line.split()
        assert 6 * int(nr) * int(nz) ** 2 == int(ncells)
        assert int(ncells) * int(order) ** 3 == int(ndof)
