"""The element-partitioned path on ONE GPU: P partitions of a mesh, each behind its own library context with owned and ghost
elements, advanced stage by stage with their halo (face traces, viscous face fluxes) packed, routed and unpacked exactly as the
multi-GPU driver does it (paper_2502_17805_b200.partition) -- only the transport is a device copy instead of NCCL.  The result
must not depend on P: every element sees the same inputs and runs the same kernel arithmetic, so the states agree BIT FOR BIT
with the unpartitioned run (SURVEY.md S8(e) "results must be independent of P")."""
import numpy as np
import pytest

import paper_2502_17805_b200 as P
from paper_2502_17805_b200 import inputs as I
from paper_2502_17805_b200.partition import EmulatedPartitions
from oracle import binding as ob
from helpers import g25_error

pytestmark = pytest.mark.gpu


def _case(n, nz, nr, diff, seed=31):
    sh = I.Shell(N_rho=3.0)
    w = I.Workload("part", n, nz, nr, 3.0, seed, diff, True, shell=sh)
    mesh = w.mesh()
    g = P.Chorus(mesh, n, I.Physics())
    Q = I.shell_state(g.xsol(), sh, seed, u_amp=0.01, b_amp=0.05)
    g.set_state(Q)
    phys = w.physics(g.max_wavespeed())
    g.set_physics(phys)
    _, xf, _, _ = P.get_operators(n)
    return w, mesh, g, Q, phys, w.dt(g.max_wavespeed(), xf[1] - xf[0])


@pytest.mark.parametrize("n,diff", [(6, 1e-3), (6, 0.0), (4, 1e-3), (5, 0.0), (7, 1e-3), (8, 1e-3)])
def test_results_do_not_depend_on_the_number_of_partitions(n, diff):
    w, mesh, g, Q, phys, dt = _case(n, 6, 3, diff)
    for _ in range(2):
        g.step(dt, 5)
    q1, ws1, d1 = g.get_state(), g.max_wavespeed(), g.diagnostics()
    for nparts in (2, 3):
        ep = EmulatedPartitions(mesh, n, phys, nparts)
        assert sum(p.info["n_owned"] for p in ep.parts) == mesh["n_elem"] and all(p.n_recv > 0 for p in ep.parts)
        ep.set_state(Q)
        for _ in range(2):
            ep.step(dt, 5)
        np.testing.assert_array_equal(ep.get_state(), q1)
        assert ep.max_wavespeed() == ws1
        d = ep.diagnostics()
        for k in ("V", "KE", "EB"):
            assert abs(d[k] / d1[k] - 1) <= 1e-13


def test_split_step_is_the_step_and_guards_its_sequence():
    w, mesh, g, Q, phys, dt = _case(6, 4, 2, 1e-3)
    g.step(dt, 5)
    q_ref = g.get_state()
    g2 = P.Chorus(mesh, 6, phys)
    g2.set_state(Q)
    g2.step_begin(dt, 5)
    with pytest.raises(P.ChorusError):
        g2.stage_face(0)                       # face before main
    with pytest.raises(P.ChorusError):
        g2.step(dt, 5)                         # whole step inside a split step
    for i in range(5):
        g2.stage_main(i)
        with pytest.raises(P.ChorusError):
            g2.stage_main(i)                   # twice
        g2.stage_face(i)
    np.testing.assert_array_equal(g2.get_state(), q_ref)
    with pytest.raises(P.ChorusError):
        g2.stage_main(0)                       # no step in progress
    # a partition refuses the whole-mesh calls and bad halo lists
    g2.set_owned(mesh["n_elem"] - 10)
    with pytest.raises(P.ChorusError):
        g2.step(dt, 5)
    with pytest.raises(P.ChorusError):
        g2.residual()
    with pytest.raises(P.ChorusError):
        g2.halo_setup([mesh["n_elem"] - 1], [0], [], [])        # a ghost in the send list
    with pytest.raises(P.ChorusError):
        g2.halo_setup([], [], [0], [7])                          # an owned element / bad face in the receive list


def test_partitioned_run_against_the_oracle():
    """... and against the CPU oracle on the whole mesh (the oracle knows nothing of partitions)."""
    w, mesh, g, Q, phys, dt = _case(6, 4, 3, 1e-3, seed=32)
    o = ob.Oracle(mesh, 6, phys)
    o.set_state(Q)
    ep = EmulatedPartitions(mesh, 6, phys, 4)
    ep.set_state(Q)
    for _ in range(2):
        o.step(dt, 5); ep.step(dt, 5)
    assert g25_error(ep.get_state(), o.get_state(), phys.c_h).max() <= 1e-9
    assert abs(ep.max_wavespeed() / o.max_wavespeed() - 1) <= 1e-12
