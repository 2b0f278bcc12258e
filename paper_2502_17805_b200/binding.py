"""Thin ctypes binding of include/chorus.h (argument marshalling only; every step of the hot path runs in the
CUDA kernels of libchorus_b200.so).  There is no CPU fallback: importing works without a GPU (so that the symbol
table can be checked), but creating a `Chorus` without the built library or without a CUDA device raises.

Host data are numpy arrays; device data are torch CUDA tensors (torch is used for device memory and streams only).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("CHORUS_LIB", os.path.join(HERE, "libchorus_b200.so"))   # override: A/B testing of builds

CHORUS_OK, CHORUS_EINVAL, CHORUS_ENOMEM, CHORUS_ECUDA, CHORUS_ESTATE = 0, -1, -2, -3, -4
STATIC_DIAG_MAX_POINTS = 1 << 25     # CHORUS_STATIC_DIAG_MAX_POINTS of include/chorus.h

# every symbol include/chorus.h declares
SYMBOLS = ("chorus_init", "chorus_free", "chorus_set_physics", "chorus_set_state", "chorus_get_state", "chorus_residual",
           "chorus_step", "chorus_step_begin", "chorus_stage_main", "chorus_stage_face", "chorus_set_owned", "chorus_halo_setup",
           "chorus_halo_pack", "chorus_halo_unpack", "chorus_diagnostics_sums", "chorus_max_wavespeed", "chorus_diagnostics", "chorus_last_error", "chorus_get_geometry", "chorus_get_gradient",
           "chorus_get_operators", "chorus_launch_count", "chorus_profile", "chorus_profile_read", "chorus_fp64_peak",
           "chorus_diagnostics_static", "chorus_static_last_error", "chorus_step_host", "chorus_sync")


class ChorusError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"chorus error {code}: {msg}")
        self.code = code


class _Mesh(C.Structure):
    _fields_ = [("n_elem", C.c_int64), ("n_geom", C.c_int32), ("geom_nodes", C.c_void_p), ("xyz", C.c_void_p),
                ("nbr_elem", C.c_void_p), ("nbr_face", C.c_void_p), ("nbr_orient", C.c_void_p)]


class _Phys(C.Structure):
    _fields_ = [("gamma", C.c_double), ("R_gas", C.c_double), ("Cp", C.c_double), ("GM", C.c_double),
                ("Omega", C.c_double), ("nu", C.c_double), ("kappa", C.c_double), ("eta", C.c_double),
                ("kr_scale", C.c_double), ("kr_c", C.c_double * 3), ("kr_wscale", C.c_double),
                ("c_h", C.c_double), ("a_psi", C.c_double), ("q_bottom", C.c_double), ("T_top", C.c_double),
                ("bc_mag_inner", C.c_int32), ("bc_mag_outer", C.c_int32), ("flags", C.c_uint32)]


def _phys_struct(p) -> _Phys:
    s = _Phys()
    for name, _ in _Phys._fields_:
        v = getattr(p, name)
        if name == "kr_c":
            s.kr_c = (C.c_double * 3)(*v)
        else:
            setattr(s, name, v)
    return s


_lib = None


def lib():
    """Load libchorus_b200.so (built in-tree by paper_2502_17805_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ChorusError(CHORUS_ECUDA, f"{LIB_PATH} is not built (run python -m paper_2502_17805_b200.build); "
                                            "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        V, I, D = C.c_void_p, C.c_int, C.c_double
        L.chorus_init.argtypes = [C.POINTER(V), C.POINTER(_Mesh), I, C.POINTER(_Phys), V]
        L.chorus_free.argtypes = [V]
        L.chorus_free.restype = None
        L.chorus_set_physics.argtypes = [V, C.POINTER(_Phys)]
        L.chorus_set_state.argtypes = [V, V, I]
        L.chorus_get_state.argtypes = [V, V, I]
        L.chorus_residual.argtypes = [V, V, I]
        L.chorus_step.argtypes = [V, D, I]
        L.chorus_max_wavespeed.argtypes = [V, C.POINTER(D)]
        L.chorus_diagnostics.argtypes = [V, V]
        L.chorus_diagnostics_sums.argtypes = [V, V]
        L.chorus_step_begin.argtypes = [V, D, I]
        L.chorus_stage_main.argtypes = [V, I]
        L.chorus_stage_face.argtypes = [V, I]
        L.chorus_set_owned.argtypes = [V, C.c_int64]
        L.chorus_halo_setup.argtypes = [V, C.c_int64, V, V, C.c_int64, V, V]
        L.chorus_halo_pack.argtypes = [V, I, V]
        L.chorus_halo_unpack.argtypes = [V, I, V]
        L.chorus_last_error.argtypes = [V]
        L.chorus_last_error.restype = C.c_char_p
        L.chorus_get_geometry.argtypes = [V, V, V, V, V, I]
        L.chorus_get_gradient.argtypes = [V, V, I]
        L.chorus_get_operators.argtypes = [I, V, V, V, V]
        L.chorus_launch_count.argtypes = [V]
        L.chorus_launch_count.restype = C.c_int64
        L.chorus_profile.argtypes = [V, I]
        L.chorus_profile_read.argtypes = [V, V, V]
        L.chorus_step_host.argtypes = [V, V, V, D, I, V]
        L.chorus_sync.argtypes = [V]
        L.chorus_diagnostics_static.argtypes = [I, C.c_int64, V, V, V, V]
        L.chorus_static_last_error.argtypes = []
        L.chorus_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _ptr(a):
    """(pointer, on_device) of a contiguous fp64 numpy array or torch tensor."""
    if _is_torch(a):
        import torch
        assert a.dtype == torch.float64 and a.is_contiguous()
        return C.c_void_p(a.data_ptr()), int(a.is_cuda)
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.c_void_p), 0


def get_operators(order):
    """Node sets and 1-D operators the library uses: xs, xf, Isf [(n+1),n], Dfs [n,(n+1)]."""
    n = order
    xs, xf, Isf, Dfs = np.empty(n), np.empty(n + 1), np.empty((n + 1, n)), np.empty((n, n + 1))
    rc = lib().chorus_get_operators(n, *[a.ctypes.data_as(C.c_void_p) for a in (xs, xf, Isf, Dfs)])
    if rc:
        raise ChorusError(rc, "chorus_get_operators")
    return xs, xf, Isf, Dfs


def diagnostics_static(order, q, detJ, out, stream=None):
    """chorus_diagnostics_static (include/chorus.h): V, KE, E_B of a state WITHOUT a context and without any allocation.
    q [9][E][n^3], detJ [E][n^3], out [3]: contiguous fp64 CUDA tensors of the current device; asynchronous on `stream`
    (a torch.cuda.Stream, or None for the default stream).  Nothing is returned: the result lands in `out`."""
    for a in (q, detJ, out):
        if not (_is_torch(a) and a.is_cuda):
            raise ChorusError(CHORUS_EINVAL, "diagnostics_static takes CUDA tensors")
    n3 = int(order) ** 3
    E = detJ.numel() // n3
    if detJ.numel() != E * n3 or q.numel() != 9 * E * n3 or out.numel() != 3:
        raise ChorusError(CHORUS_EINVAL, "diagnostics_static: q [9][E][n^3], detJ [E][n^3], out [3]")
    st = C.c_void_p(stream.cuda_stream) if stream is not None else C.c_void_p(0)
    rc = lib().chorus_diagnostics_static(int(order), E, _ptr(q)[0], _ptr(detJ)[0], _ptr(out)[0], st)
    if rc != 0:
        raise ChorusError(rc, lib().chorus_static_last_error().decode())


def fp64_peak(mode=0, seconds=1.0):
    """Sustained FP64 rate of the current device in TFLOP/s: (total, DFMA share, DMMA share).  mode 0 DFMA, 1 DMMA, 2 both."""
    import torch
    if not torch.cuda.is_available():
        raise ChorusError(CHORUS_ECUDA, "no CUDA device")
    t, a, b = C.c_double(), C.c_double(), C.c_double()
    f = lib().chorus_fp64_peak
    f.argtypes = [C.c_int, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    rc = f(int(mode), float(seconds), C.byref(t), C.byref(a), C.byref(b))
    if rc:
        raise ChorusError(rc, "chorus_fp64_peak")
    return t.value, a.value, b.value


class Chorus:
    """One chorus_ctx: `mesh` is a dict from paper_2502_17805_b200.inputs, `phys` an inputs.Physics."""

    def __init__(self, mesh, order, phys, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise ChorusError(CHORUS_ECUDA, "no CUDA device: the hot path has no CPU fallback")
        self.n, self.E = int(order), int(mesh["n_elem"])
        keep = [np.ascontiguousarray(mesh["geom_nodes"], np.float64), np.ascontiguousarray(mesh["xyz"], np.float64),
                np.ascontiguousarray(mesh["nbr_elem"], np.int32), np.ascontiguousarray(mesh["nbr_face"], np.uint8),
                np.ascontiguousarray(mesh["nbr_orient"], np.uint8)]
        m = _Mesh(self.E, int(mesh["n_geom"]), *[a.ctypes.data_as(C.c_void_p) for a in keep])
        self._stream = torch.cuda.current_stream().cuda_stream if stream is None else stream
        self._ctx = C.c_void_p()
        rc = lib().chorus_init(C.byref(self._ctx), C.byref(m), self.n, C.byref(_phys_struct(phys)), C.c_void_p(self._stream))
        if rc:
            self._ctx = C.c_void_p()
            raise ChorusError(rc, "chorus_init failed")

    # -- plumbing
    def _check(self, rc):
        if rc:
            raise ChorusError(rc, lib().chorus_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None):
            lib().chorus_free(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def shape(self):
        return (9, self.E, self.n ** 3)

    def _out(self, shape, like_device):
        if like_device:
            import torch
            return torch.empty(shape, dtype=torch.float64, device="cuda")
        return np.empty(shape)

    # -- the C ABI, same names
    def set_physics(self, phys):
        self._check(lib().chorus_set_physics(self._ctx, C.byref(_phys_struct(phys))))

    def set_state(self, q):
        assert tuple(q.shape) == self.shape
        p, dev = _ptr(q)
        self._check(lib().chorus_set_state(self._ctx, p, dev))

    def get_state(self, out=None, device=False):
        out = self._out(self.shape, device) if out is None else out
        p, dev = _ptr(out)
        self._check(lib().chorus_get_state(self._ctx, p, dev))
        return out

    def residual(self, out=None, device=False):
        out = self._out(self.shape, device) if out is None else out
        p, dev = _ptr(out)
        self._check(lib().chorus_residual(self._ctx, p, dev))
        return out

    def step(self, dt, nstages=5):
        self._check(lib().chorus_step(self._ctx, float(dt), int(nstages)))

    def step_begin(self, dt, nstages=5):
        self._check(lib().chorus_step_begin(self._ctx, float(dt), int(nstages)))

    def stage_main(self, istage):
        self._check(lib().chorus_stage_main(self._ctx, int(istage)))

    def stage_face(self, istage):
        self._check(lib().chorus_stage_face(self._ctx, int(istage)))

    def set_owned(self, n_owned):
        self._check(lib().chorus_set_owned(self._ctx, int(n_owned)))

    def halo_setup(self, send_elem, send_face, recv_elem, recv_face):
        se, sf = np.ascontiguousarray(send_elem, np.int32), np.ascontiguousarray(send_face, np.uint8)
        re_, rf = np.ascontiguousarray(recv_elem, np.int32), np.ascontiguousarray(recv_face, np.uint8)
        assert se.size == sf.size and re_.size == rf.size
        ps = [a.ctypes.data_as(C.c_void_p) if a.size else None for a in (se, sf, re_, rf)]
        self._check(lib().chorus_halo_setup(self._ctx, se.size, ps[0], ps[1], re_.size, ps[2], ps[3]))

    def halo_pack(self, field, buf):
        """buf: torch CUDA float64 tensor [n_send, w n^2] (w = 9 traces, 7 viscous)."""
        self._check(lib().chorus_halo_pack(self._ctx, int(field), C.c_void_p(buf.data_ptr())))

    def halo_unpack(self, field, buf):
        self._check(lib().chorus_halo_unpack(self._ctx, int(field), C.c_void_p(buf.data_ptr())))

    def step_host(self, q_in, q_out, dt, nstages=5, ws_out=None):
        """chorus_step_host: one pipelined host job.  q_in, q_out: contiguous fp64 HOST arrays [9][E][n^3] (numpy or CPU torch,
        pinned for overlap); ws_out: a 1-element fp64 HOST array or None.  Nothing is valid before sync()."""
        assert tuple(q_in.shape) == self.shape and tuple(q_out.shape) == self.shape
        (pi, di), (po, do) = _ptr(q_in), _ptr(q_out)
        if di or do:
            raise ChorusError(CHORUS_EINVAL, "step_host takes HOST buffers")
        pw = _ptr(ws_out)[0] if ws_out is not None else C.c_void_p(0)
        self._check(lib().chorus_step_host(self._ctx, pi, po, float(dt), int(nstages), pw))

    def sync(self):
        self._check(lib().chorus_sync(self._ctx))

    def diagnostics_sums(self):
        out = np.empty(3)
        self._check(lib().chorus_diagnostics_sums(self._ctx, out.ctypes.data_as(C.c_void_p)))
        return out

    def max_wavespeed(self):
        v = C.c_double()
        self._check(lib().chorus_max_wavespeed(self._ctx, C.byref(v)))
        return v.value

    def diagnostics(self):
        """dict(V, KE, EB): shell volume, volume-averaged kinetic and magnetic energy (Eq. 34-35)."""
        out = np.empty(3)
        self._check(lib().chorus_diagnostics(self._ctx, out.ctypes.data_as(C.c_void_p)))
        return dict(V=float(out[0]), KE=float(out[1]), EB=float(out[2]))

    def gradient(self, device=False):
        out = self._out((27, self.E, self.n ** 3), device)
        p, dev = _ptr(out)
        self._check(lib().chorus_get_gradient(self._ctx, p, dev))
        return out

    def geometry(self):
        n, E = self.n, self.E
        detJ, S = np.empty((E, n ** 3)), np.empty((E, 3, 3, n * n * (n + 1)))
        xsol, jinv = np.empty((3, E, n ** 3)), np.empty((E, 3, 3, n ** 3))
        ps = [a.ctypes.data_as(C.c_void_p) for a in (detJ, S, xsol, jinv)]
        self._check(lib().chorus_get_geometry(self._ctx, *ps, 0))
        return dict(detJ=detJ, S=S, xsol=xsol, jinv=jinv)

    def xsol(self):
        out = np.empty((3, self.E, self.n ** 3))
        self._check(lib().chorus_get_geometry(self._ctx, None, None, out.ctypes.data_as(C.c_void_p), None, 0))
        return out

    def launch_count(self):
        return int(lib().chorus_launch_count(self._ctx))

    def profile(self, enable=True):
        self._check(lib().chorus_profile(self._ctx, int(enable)))

    def profile_read(self):
        """{'trace': (ms, launches), 'face': ..., 'main': ...} accumulated since the last read.  'face' is the viscous face kernel
        (the gradient kernel on the scalar path), 'main' the element kernel (stage_main_kernel / residual_kernel)."""
        ms, cnt = np.zeros(3), np.zeros(3, np.int64)
        self._check(lib().chorus_profile_read(self._ctx, ms.ctypes.data_as(C.c_void_p), cnt.ctypes.data_as(C.c_void_p)))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(("trace", "face", "main"))}
