"""ctypes binding of oracle/sd_mhd_oracle.h (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class _Mesh(C.Structure):
    _fields_ = [("n_elem", C.c_int64), ("n_geom", C.c_int32), ("geom_nodes", C.c_void_p), ("xyz", C.c_void_p),
                ("nbr_elem", C.c_void_p), ("nbr_face", C.c_void_p), ("nbr_orient", C.c_void_p)]


class _Phys(C.Structure):
    _fields_ = [("gamma", C.c_double), ("R_gas", C.c_double), ("Cp", C.c_double), ("GM", C.c_double),
                ("Omega", C.c_double), ("nu", C.c_double), ("kappa", C.c_double), ("eta", C.c_double),
                ("kr_scale", C.c_double), ("kr_c", C.c_double * 3), ("kr_wscale", C.c_double),
                ("c_h", C.c_double), ("a_psi", C.c_double), ("q_bottom", C.c_double), ("T_top", C.c_double),
                ("bc_mag_inner", C.c_int32), ("bc_mag_outer", C.c_int32), ("flags", C.c_uint32)]


def physics_struct(p) -> _Phys:
    s = _Phys()
    for name, _ in _Phys._fields_:
        v = getattr(p, name)
        if name == "kr_c":
            s.kr_c = (C.c_double * 3)(*v)
        else:
            setattr(s, name, v)
    return s


def lib():
    global _lib
    if _lib is None:
        # the oracle's OpenMP threads share the box with other work: sleep, do not spin, at barriers
        os.environ.setdefault("OMP_WAIT_POLICY", "passive")
        L = C.CDLL(_build.build())
        L.oracle_init.restype = C.c_void_p
        L.oracle_init.argtypes = [C.POINTER(_Mesh), C.c_int, C.POINTER(_Phys), C.c_int]
        L.oracle_free.argtypes = [C.c_void_p]
        L.oracle_free.restype = None
        for f in ("oracle_set_state", "oracle_get_state", "oracle_max_wavespeed", "oracle_get_gradient"):
            getattr(L, f).argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_set_physics.argtypes = [C.c_void_p, C.POINTER(_Phys)]
        L.oracle_residual.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.oracle_get_geometry.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.oracle_nodes.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_quadrature_weights.argtypes = [C.c_int, C.c_void_p]
        L.oracle_diagnostics.argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_operators.argtypes = [C.c_int] + [C.c_void_p] * 4
        L.oracle_rk_tableau.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        P, V = C.POINTER(_Phys), C.c_void_p
        L.oracle_flux_inviscid.argtypes = [P, V, V, V]
        L.oracle_flux_viscous.argtypes = [P, V, V, V, C.c_double, V]
        L.oracle_flux_rusanov.argtypes = [P, V, V, V, V]
        L.oracle_fast_speed.argtypes = [P, V, V]
        L.oracle_fast_speed.restype = C.c_double
        L.oracle_wavespeed.argtypes = [P, V]
        L.oracle_wavespeed.restype = C.c_double
        L.oracle_wall_state.argtypes = [P, C.c_int, V, V, V]
        L.oracle_flux_wall_inviscid.argtypes = [P, V, V, V]
        L.oracle_flux_wall_viscous.argtypes = [P, C.c_int, V, V, V, C.c_double, C.c_double, V]
        L.oracle_wall_condition_gradB.argtypes = [C.c_int, V, V, V, C.c_double, V]
        L.oracle_wall_condition_gradB.restype = None
        L.oracle_source.argtypes = [P, V, V, V, V, V]
        for f in ("oracle_flux_inviscid", "oracle_flux_viscous", "oracle_flux_rusanov", "oracle_wall_state",
                  "oracle_flux_wall_inviscid", "oracle_flux_wall_viscous", "oracle_source"):
            getattr(L, f).restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ---- 1-D building blocks ---------------------------------------------------------------
def nodes(n):
    xs, xf = np.empty(n), np.empty(n + 1)
    assert lib().oracle_nodes(n, _p(xs), _p(xf)) == 0
    return xs, xf


def quadrature_weights(n):
    w = np.empty(n)
    assert lib().oracle_quadrature_weights(n, _p(w)) == 0
    return w


def operators(n):
    Isf, Dfs, Efs, Dff = np.empty((n + 1, n)), np.empty((n, n + 1)), np.empty((n, n + 1)), np.empty((n + 1, n + 1))
    assert lib().oracle_operators(n, _p(Isf), _p(Dfs), _p(Efs), _p(Dff)) == 0
    return Isf, Dfs, Efs, Dff


def rk_tableau(nstages):
    al, be = np.empty((5, 5)), np.empty((5, 5))
    assert lib().oracle_rk_tableau(nstages, _p(al), _p(be)) == 0
    return al, be


# ---- pointwise physics -----------------------------------------------------------------
def flux_inviscid(phys, Q, S):
    F = np.empty(9); Q, S = _d(Q), _d(S)
    lib().oracle_flux_inviscid(C.byref(physics_struct(phys)), _p(Q), _p(S), _p(F))
    return F


def flux_viscous(phys, Q, G, S, kr=0.0):
    F = np.empty(9); Q, G, S = _d(Q), _d(G), _d(S)
    lib().oracle_flux_viscous(C.byref(physics_struct(phys)), _p(Q), _p(G), _p(S), kr, _p(F))
    return F


def flux_rusanov(phys, Qi, Qo, nh):
    F = np.empty(9); Qi, Qo, nh = _d(Qi), _d(Qo), _d(nh)
    lib().oracle_flux_rusanov(C.byref(physics_struct(phys)), _p(Qi), _p(Qo), _p(nh), _p(F))
    return F


def fast_speed(phys, Q, nh):
    Q, nh = _d(Q), _d(nh)
    return lib().oracle_fast_speed(C.byref(physics_struct(phys)), _p(Q), _p(nh))


def wavespeed(phys, Q):
    Q = _d(Q)
    return lib().oracle_wavespeed(C.byref(physics_struct(phys)), _p(Q))


def wall_state(phys, wall, Q, nh):
    Qb = np.empty(9); Q, nh = _d(Q), _d(nh)
    lib().oracle_wall_state(C.byref(physics_struct(phys)), wall, _p(Q), _p(nh), _p(Qb))
    return Qb


def flux_wall_inviscid(phys, Qb, nh):
    F = np.empty(9); Qb, nh = _d(Qb), _d(nh)
    lib().oracle_flux_wall_inviscid(C.byref(physics_struct(phys)), _p(Qb), _p(nh), _p(F))
    return F


def flux_wall_viscous(phys, wall, Qb, G, nh, kr=0.0, rw=0.0):
    F = np.empty(9)
    Qb, G, nh = _d(Qb), _d(G), _d(nh)
    lib().oracle_flux_wall_viscous(C.byref(physics_struct(phys)), wall, _p(Qb), _p(G), _p(nh), float(rw), float(kr), _p(F))
    return F


def wall_condition_gradB(bc, dB, Bb, er, rw):
    out = np.empty((3, 3))
    dB, Bb, er = _d(dB), _d(Bb), _d(er)
    lib().oracle_wall_condition_gradB(int(bc), _p(dB), _p(Bb), _p(er), float(rw), _p(out))
    return out


def source(phys, Q, G, x):
    M, Ma = np.empty(9), np.empty(9); Q, G, x = _d(Q), _d(G), _d(x)
    lib().oracle_source(C.byref(physics_struct(phys)), _p(Q), _p(G), _p(x), _p(M), _p(Ma))
    return M, Ma


# ---- whole-mesh solver -----------------------------------------------------------------
class Oracle:
    """oracle_ctx wrapper.  mesh: dict from paper_2502_17805_b200.inputs; phys: inputs.Physics."""

    def __init__(self, mesh, order, phys, prec=0):
        self.n, self.E = order, int(mesh["n_elem"])
        self._keep = [_d(mesh["geom_nodes"]), _d(mesh["xyz"]), np.ascontiguousarray(mesh["nbr_elem"], np.int32),
                      np.ascontiguousarray(mesh["nbr_face"], np.uint8), np.ascontiguousarray(mesh["nbr_orient"], np.uint8)]
        m = _Mesh(self.E, int(mesh["n_geom"]), *[_p(a) for a in self._keep])
        self._ctx = lib().oracle_init(C.byref(m), order, C.byref(physics_struct(phys)), prec)
        if not self._ctx:
            raise ValueError("oracle_init failed")

    def close(self):
        if self._ctx:
            lib().oracle_free(self._ctx)
            self._ctx = None

    __del__ = close

    @property
    def shape(self):
        return (9, self.E, self.n ** 3)

    def set_physics(self, phys):
        assert lib().oracle_set_physics(self._ctx, C.byref(physics_struct(phys))) == 0

    def set_state(self, q):
        q = _d(q)
        assert q.shape == self.shape
        assert lib().oracle_set_state(self._ctx, _p(q)) == 0

    def get_state(self):
        q = np.empty(self.shape)
        assert lib().oracle_get_state(self._ctx, _p(q)) == 0
        return q

    def residual(self, magnitude=False):
        r = np.empty(self.shape)
        a = np.empty(self.shape) if magnitude else None
        assert lib().oracle_residual(self._ctx, _p(r), _p(a)) == 0
        return (r, a) if magnitude else r

    def step(self, dt, nstages=5):
        assert lib().oracle_step(self._ctx, float(dt), nstages) == 0

    def max_wavespeed(self):
        out = np.empty(1)
        assert lib().oracle_max_wavespeed(self._ctx, _p(out)) == 0
        return float(out[0])

    def diagnostics(self):
        """dict(V, KE, EB): shell volume, volume-averaged kinetic and magnetic energy (Eq. 34-35)."""
        out = np.empty(3)
        assert lib().oracle_diagnostics(self._ctx, _p(out)) == 0
        return dict(V=float(out[0]), KE=float(out[1]), EB=float(out[2]))

    def gradient(self):
        g = np.empty((27, self.E, self.n ** 3))
        assert lib().oracle_get_gradient(self._ctx, _p(g)) == 0
        return g

    def geometry(self):
        n, E = self.n, self.E
        detJ, S = np.empty((E, n ** 3)), np.empty((E, 3, 3, n * n * (n + 1)))
        xsol, jinv = np.empty((3, E, n ** 3)), np.empty((E, 3, 3, n ** 3))
        assert lib().oracle_get_geometry(self._ctx, _p(detJ), _p(S), _p(xsol), _p(jinv)) == 0
        return dict(detJ=detJ, S=S, xsol=xsol, jinv=jinv)
