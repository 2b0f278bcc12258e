"""CPU-side checks of the CUDA library and its binding (no GPU compute): the C-ABI library loads and exports every
symbol include/chorus.h declares, its host-side node sets / operators agree with the pinned oracle, the product path
refuses to run without a device (no CPU fallback), and the product package never imports the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2502_17805_b200 as P
from paper_2502_17805_b200 import binding as B, inputs as I
from oracle import binding as ob

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_header_and_library_symbols_match():
    hdr = open(os.path.join(ROOT, "include", "chorus.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(chorus_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(P.SYMBOLS)
    L = P.lib()
    for s in P.SYMBOLS:
        assert hasattr(L, s), s


@pytest.mark.parametrize("n", range(2, 10))
def test_library_operators_agree_with_oracle(n):
    xs, xf, Isf, Dfs = P.get_operators(n)
    oxs, oxf = ob.nodes(n)
    oI, oD, _, _ = ob.operators(n)
    np.testing.assert_allclose(xs, oxs, atol=1e-15)
    np.testing.assert_allclose(xf, oxf, atol=1e-15)
    np.testing.assert_allclose(Isf, oI, atol=1e-13)
    np.testing.assert_allclose(Dfs, oD, atol=1e-13 * np.abs(oD).max())
    assert P.lib().chorus_get_operators(1, None, None, None, None) == B.CHORUS_EINVAL
    assert P.lib().chorus_get_operators(10, None, None, None, None) == B.CHORUS_EINVAL


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    m = I.periodic_box(1, 1, 1, (1, 1, 1), I.lobatto_abscissae(3))
    with pytest.raises(P.ChorusError):
        P.Chorus(m, 2, I.Physics())
    # the C entry point itself reports the missing device
    keep = [np.ascontiguousarray(m["geom_nodes"]), np.ascontiguousarray(m["xyz"]), m["nbr_elem"], m["nbr_face"], m["nbr_orient"]]
    ms = B._Mesh(1, 3, *[a.ctypes.data_as(C.c_void_p) for a in keep])
    ctx = C.c_void_p()
    rc = P.lib().chorus_init(C.byref(ctx), C.byref(ms), 2, C.byref(B._phys_struct(I.Physics())), None)
    assert rc == B.CHORUS_ECUDA and not ctx.value


def test_init_rejects_bad_arguments():
    ctx = C.c_void_p()
    assert P.lib().chorus_init(C.byref(ctx), None, 6, None, None) == B.CHORUS_EINVAL
    assert P.lib().chorus_init(None, None, 6, None, None) == B.CHORUS_EINVAL
    assert P.lib().chorus_set_state(None, None, 0) == B.CHORUS_EINVAL
    assert P.lib().chorus_launch_count(None) == 0


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2502_17805_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "sd_mhd_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "csrc" not in src.replace("paper_2502_17805_b200/csrc).", "") and "#include \"../" not in src


def test_context_free_entry_points_reject_bad_arguments_without_a_device():
    """chorus_diagnostics_static validates its arguments before it touches the device: bad order, empty mesh, null pointers and a
    size beyond the static scratch's maximum come back as CHORUS_EINVAL with a message; chorus_step_host / chorus_sync refuse a
    null context.  (No compute call is made: there is no GPU here.)"""
    L = P.lib()
    buf = (C.c_double * 4)()
    p = C.cast(buf, C.c_void_p)
    assert L.chorus_diagnostics_static(10, 1, p, p, p, None) == B.CHORUS_EINVAL
    assert b"order" in L.chorus_static_last_error()
    assert L.chorus_diagnostics_static(6, 0, p, p, p, None) == B.CHORUS_EINVAL
    assert L.chorus_diagnostics_static(6, 1, None, p, p, None) == B.CHORUS_EINVAL
    too_many = B.STATIC_DIAG_MAX_POINTS // 216 + 1
    assert L.chorus_diagnostics_static(6, too_many, p, p, p, None) == B.CHORUS_EINVAL
    msg = L.chorus_static_last_error().decode()
    assert "maximum" in msg and str(B.STATIC_DIAG_MAX_POINTS) in msg
    assert L.chorus_step_host(None, p, p, 1e-3, 5, None) == B.CHORUS_EINVAL
    assert L.chorus_sync(None) == B.CHORUS_EINVAL
    import torch
    with pytest.raises(P.ChorusError):
        P.diagnostics_static(6, torch.zeros(9, 1, 216, dtype=torch.float64), torch.zeros(1, 216, dtype=torch.float64),
                             torch.zeros(3, dtype=torch.float64))
