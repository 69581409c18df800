"""The C-ABI library loads, exports every symbol include/thor.h declares, and reports errors the
way the header says.  No compute calls here (runs without a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1607_05535_b200 as thor
import thor_inputs as ti
from conftest import ROOT, have_cuda


def _declared():
    src = open(os.path.join(ROOT, "include", "thor.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(thor_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_1607_05535_b200 import build
    build.build()
    lib = ctypes.CDLL(thor.LIB_PATH)
    names = _declared()
    assert len(names) >= 16
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(thor._SIGNATURES) == names           # the binding covers the whole header, nothing else
    for n in names:
        assert callable(getattr(thor, n)), n           # same names in the Python binding


def test_error_codes_and_messages():
    lib = thor.load_library()
    h = ctypes.c_void_p()
    P = thor.thor_planet(**{k: ti.EARTH[k] for k in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")})
    assert lib.thor_grid_create(-1, 8, ctypes.byref(P), ctypes.byref(h)) == thor.THOR_EINVAL
    assert lib.thor_grid_create(3, 1, ctypes.byref(P), ctypes.byref(h)) == thor.THOR_EINVAL
    assert lib.thor_grid_create(3, 8, None, ctypes.byref(h)) == thor.THOR_EINVAL
    assert h.value is None                              # nothing written on failure
    assert b"thor_grid_create" in lib.thor_last_error()
    assert lib.thor_step(None, 1, 1.0, 2, None) == thor.THOR_EINVAL
    with pytest.raises(thor.ThorError):
        thor.thor_grid_create(2, 8, dict(ti.EARTH, Cp=100.0))     # Cp <= Rd


def test_vertical_grid_arguments():
    """thor_grid_create_vertical (NEXT-3): interface altitudes must start at 0 and increase strictly; orders 1 and 3."""
    nv = 6
    z = ti.stretched_interfaces(ti.EARTH, nv, 3.0)
    g = thor.Grid(1, nv, ti.EARTH, z_interfaces=z, order_k=3)
    assert g.n_layers == nv
    g.close()
    bad = z.copy()
    bad[3] = bad[2]
    for args in ((bad, 1), (z + 1.0, 1), (z, 2), (z, 5), (z, 0)):
        with pytest.raises(thor.ThorError) as e:
            thor.Grid(1, nv, ti.EARTH, z_interfaces=args[0], order_k=args[1])
        assert e.value.code == thor.THOR_EINVAL
    with pytest.raises(thor.ThorError):
        thor.Grid(1, nv, ti.EARTH, z_interfaces=z[:-1])            # wrong length is caught by the binding


@pytest.mark.skipif(have_cuda(), reason="checks the no-device behaviour")
def test_device_entry_points_fail_loudly_without_a_gpu():
    g = thor.Grid(1, 4, ti.EARTH)
    N = g.n_cols
    with pytest.raises(thor.ThorError) as e:
        thor.State(g, np.ones((N, 4)), np.zeros((N, 4, 3)), np.zeros((N, 5)), np.ones((N, 4)))
    assert e.value.code == thor.THOR_ECUDA
    with pytest.raises(thor.ThorError):
        g.apply_grad(np.ones((N, 4)))
    with pytest.raises(thor.ThorError) as e:                       # NEXT-3: the device grid generator needs a device too
        thor.Grid(1, 4, ti.EARTH, on_device=True)
    assert e.value.code == thor.THOR_ECUDA
