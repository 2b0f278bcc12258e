"""The 2-ring patch used for full-size GPU parity (tests/test_gpu_fullsize.py) is pinned against the oracle itself on a mesh
the oracle can run whole: the residual of the centre element of an extracted patch equals the whole-mesh residual there."""
import numpy as np
import pytest

from paper_2502_17805_b200 import inputs as I
from oracle import binding as ob


@pytest.mark.parametrize("center", [0, 37, 100, 191])      # wall elements, panel-seam elements, interior
def test_two_ring_patch_reproduces_the_centre_residual(center):
    n = 4
    w = I.Workload("t", n, 4, 2, 3.0, 11, 2e-3, True, shell=I.Shell(N_rho=3.0))
    mesh = w.mesh()
    o = ob.Oracle(mesh, n, I.Physics())
    Q = I.shell_state(o.geometry()["xsol"], w.shell, 11, u_amp=0.02, b_amp=0.1)
    o.set_state(Q)
    phys = w.physics(o.max_wavespeed())
    o.set_physics(phys)
    r_full, a_full = o.residual(True)
    patch, elems = I.extract_patch(mesh, center, rings=2)
    assert elems[0] == center and patch["n_elem"] <= 25
    op = ob.Oracle(patch, n, phys)
    op.set_state(np.ascontiguousarray(Q[:, elems]))
    r_p, _ = op.residual(True)
    scale = a_full[:, center].reshape(9, -1).max(1)
    scale = np.where(scale > 0.0, scale, scale.max())
    err = np.abs(r_p[:, 0] - r_full[:, center]).reshape(9, -1).max(1) / scale
    assert err.max() <= 1e-13, err
    # one ring is NOT enough with diffusion (the neighbours' gradients need their own neighbours)
    p1, e1 = I.extract_patch(mesh, center, rings=1)
    o1 = ob.Oracle(p1, n, phys)
    o1.set_state(np.ascontiguousarray(Q[:, e1]))
    r1, _ = o1.residual(True)
    err1 = np.abs(r1[:, 0] - r_full[:, center]).reshape(9, -1).max(1) / scale
    assert err1.max() > 1e-9
