"""chorus_diagnostics_static (include/chorus.h): the diagnostics of Eq. 34-35 through the entry point that allocates nothing
-- its scratch is a fixed device array inside the library -- against the existing path (chorus_diagnostics of a context) and
against the oracle, on two calls in a row.  Collected last on purpose (the suite runs with pytest -x)."""
import ctypes as C

import numpy as np
import pytest

import paper_2502_17805_b200 as P
from paper_2502_17805_b200 import inputs as I
from oracle import binding as ob

pytestmark = pytest.mark.gpu

TOL = 1e-13      # relative, the tolerance of test_diagnostics_parity_and_reproducibility


def _case(n, nz, nr, seed):
    sh = I.Shell(N_rho=3.0)
    w = I.Workload("case", n, nz, nr, 3.0, seed, 1e-3, True, shell=sh)
    mesh = w.mesh()
    o = ob.Oracle(mesh, n, I.Physics())
    Q = I.shell_state(o.geometry()["xsol"], sh, seed, u_amp=0.05, b_amp=0.2)
    o.set_state(Q)
    phys = w.physics(o.max_wavespeed())
    o.set_physics(phys)
    g = P.Chorus(mesh, n, phys)
    g.set_state(Q)
    return w, o, g


def test_static_diagnostics_two_calls_in_a_row_against_the_context_path():
    import torch
    # call 1: a 768-element shell at n = 5 (96,000 points: 12 blocks of partial sums); call 2: a SMALLER mesh at n = 6 (20,736
    # points: 3 blocks), so that stale partial sums of call 1 sit in the shared scratch beyond what call 2 may read
    outs = []
    for n, nz, nr, seed in ((5, 8, 2, 21), (6, 4, 1, 22)):
        w, o, g = _case(n, nz, nr, seed)
        _, xf, _, _ = P.get_operators(n)
        dt = w.dt(o.max_wavespeed(), xf[1] - xf[0])
        o.step(dt, 5); g.step(dt, 5)                      # a state that has been through the kernels
        ref, ref_oracle = g.diagnostics(), o.diagnostics()
        q = g.get_state(device=True)
        detJ = torch.from_numpy(g.geometry()["detJ"]).cuda()
        out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        P.diagnostics_static(n, q, detJ, out)
        torch.cuda.synchronize()
        first = out.cpu().numpy().copy()
        out.fill_(float("nan"))
        P.diagnostics_static(n, q, detJ, out)             # again on the same inputs: the scratch keeps nothing that matters
        torch.cuda.synchronize()
        second = out.cpu().numpy().copy()
        if outs:                                          # (the very first call may load the module's kernels lazily)
            assert torch.cuda.mem_get_info()[0] == free0  # no device memory was taken
        np.testing.assert_array_equal(first, second)      # fixed summation tree: bit-identical
        for k, v in zip(("V", "KE", "EB"), first):
            assert abs(v / ref[k] - 1) <= TOL, (k, v, ref[k])
            assert abs(v / ref_oracle[k] - 1) <= TOL, (k, v, ref_oracle[k])
        outs.append(first)
    assert not np.array_equal(outs[0], outs[1])


def test_static_diagnostics_on_a_side_stream_and_its_limits():
    import torch
    n = 4
    w, o, g = _case(n, 4, 2, 23)
    ref = g.diagnostics()
    q = g.get_state(device=True)
    detJ = torch.from_numpy(g.geometry()["detJ"]).cuda()
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    torch.cuda.synchronize()
    P.diagnostics_static(n, q, detJ, out, stream=st)
    st.synchronize()
    for k, v in zip(("V", "KE", "EB"), out.cpu().numpy()):
        assert abs(v / ref[k] - 1) <= TOL, (k, v, ref[k])
    # beyond the static scratch's maximum: rejected with a clear message, nothing launched
    L = P.lib()
    p = C.c_void_p(out.data_ptr())
    n_elem = P.binding.STATIC_DIAG_MAX_POINTS // n ** 3 + 1
    assert L.chorus_diagnostics_static(n, n_elem, p, p, p, None) == -1
    msg = L.chorus_static_last_error().decode()
    assert "maximum" in msg and str(P.binding.STATIC_DIAG_MAX_POINTS) in msg, msg
    assert L.chorus_diagnostics_static(n, P.binding.STATIC_DIAG_MAX_POINTS // n ** 3, None, p, p, None) == -1   # null pointer
    assert L.chorus_diagnostics_static(10, 1, p, p, p, None) == -1 and "order" in L.chorus_static_last_error().decode()
    assert L.chorus_diagnostics_static(n, 0, p, p, p, None) == -1
    with pytest.raises(P.ChorusError):
        P.diagnostics_static(n, q.cpu(), detJ, out)
    torch.cuda.synchronize()
    # the entry point still works after the rejected calls
    out.zero_()
    P.diagnostics_static(n, q, detJ, out)
    torch.cuda.synchronize()
    assert abs(float(out[0]) / ref["V"] - 1) <= TOL
