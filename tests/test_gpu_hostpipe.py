"""chorus_step_host / chorus_sync: pipelined host jobs (H2D, step, D2H on three streams through two staging slots) give, bit for
bit, what the three separate synchronous calls give -- over more jobs than there are slots, with different inputs per job."""
import numpy as np
import pytest

import paper_2502_17805_b200 as P
from paper_2502_17805_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n,diff", [(6, 1e-3), (5, 0.0)])
def test_pipelined_host_jobs_equal_the_separate_calls(n, diff):
    import torch
    sh = I.Shell(N_rho=3.0)
    w = I.Workload("pipe", n, 8, 2, 3.0, 31, diff, True, shell=sh)
    mesh = w.mesh()
    g = P.Chorus(mesh, n, I.Physics())
    xs = g.xsol()
    states = [I.shell_state(xs, sh, 31 + j, u_amp=1e-3 * (j + 1), b_amp=1e-2) for j in range(5)]
    g.set_state(states[0])
    c_h = g.max_wavespeed()
    g.set_physics(w.physics(c_h))
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(c_h, xf[1] - xf[0])
    # the separate calls
    ref, ref_ws = [], []
    for q in states:
        g.set_state(q)
        g.step(dt, 5)
        ref.append(g.get_state())
        ref_ws.append(g.max_wavespeed())
    # the same five jobs, pipelined, from and into pinned memory
    hin = [torch.from_numpy(q).pin_memory() for q in states]
    hout = [torch.full(states[0].shape, float("nan"), dtype=torch.float64).pin_memory() for _ in states]
    ws = [torch.zeros(1, dtype=torch.float64).pin_memory() for _ in states]
    for j in range(5):
        g.step_host(hin[j], hout[j], dt, 5, ws[j] if j != 2 else None)      # job 2 without the wave speed
    g.sync()
    for j in range(5):
        np.testing.assert_array_equal(hout[j].numpy(), ref[j])
        if j != 2:
            assert float(ws[j][0]) == ref_ws[j]
    # the context's state is the last job's result, and the synchronous calls still work after the pipeline
    np.testing.assert_array_equal(g.get_state(), ref[4])
    g.set_state(states[1]); g.step(dt, 5)
    np.testing.assert_array_equal(g.get_state(), ref[1])
    # numpy (pageable) buffers work too
    out = np.empty_like(states[3])
    g.step_host(states[3], out, dt, 5)
    g.sync()
    np.testing.assert_array_equal(out, ref[3])
    with pytest.raises(P.ChorusError):
        g.step_host(hin[0], hout[0], dt, 4)
