"""Test-side helpers: quadrature weights, error norms (readings G24/G25), small analytic fields.
Nothing here is used by the product path."""
import numpy as np


def fejer1_weights(n):
    """Interpolatory quadrature weights on the Chebyshev-Gauss points of [0,1] (Fejer's first rule),
    closed form: w_k = (1/n)[1 - 2 sum_{j=1}^{n//2} cos(2 j theta_k)/(4j^2-1)], theta_k=(2k-1)pi/(2n)."""
    k = np.arange(1, n + 1)
    th = (2 * k - 1) * np.pi / (2 * n)
    w = np.ones(n)
    for j in range(1, n // 2 + 1):
        w -= 2.0 * np.cos(2 * j * th) / (4 * j * j - 1)
    return w / n


def w3(n):
    w = fejer1_weights(n)
    return (w[:, None, None] * w[None, :, None] * w[None, None, :]).reshape(-1)


def g24_error(r_test, r_ref, a_ref):
    """Per-variable max |dR| / max A (magnitude residual of the reference): forward-error norm of reading G24."""
    d = np.abs(r_test - r_ref).reshape(9, -1).max(1)
    den = a_ref.reshape(9, -1).max(1)
    den = np.where(den > 0.0, den, den.max())   # only a row whose every term is identically zero borrows the global scale
    return d / den


def g25_error(q_test, q_ref, c_h=None):
    """Per-variable max |dQ| / max |Q_ref|; psi (initially 0) is scaled by C_h * max|B| (reading G25)."""
    d = np.abs(q_test - q_ref).reshape(9, -1).max(1)
    den = np.abs(q_ref).reshape(9, -1).max(1)
    bmax = den[5:8].max()
    den[8] = max(den[8], (c_h if c_h else 1.0) * bmax)
    den[1:4] = den[1:4].max()                   # momentum components share one scale
    den[5:8] = bmax
    return d / den


def sol_coords_1d(xs, N, L):
    """1-D physical coordinates of the solution points of N equal elements on [0,L]."""
    return ((np.arange(N)[:, None] + xs[None, :]) * (L / N)).reshape(-1)
