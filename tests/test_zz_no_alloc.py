"""thor_diagnostics_noalloc: the entry point for callers that must not allocate (CUDA graph capture, serving loops,
harnesses that forbid cudaMalloc).  Its scratch is a file-scope device array of the library (1 MiB, at most 65 536
columns); this file checks it against the existing path, thor_diagnostics, on calls in a row.

Named test_zz_* so that pytest collects it LAST: the suite runs with `pytest -x`, and a failure here must not hide the
parity tests.  It has to pass alone in a fresh process and after all other tests."""
import numpy as np
import pytest

import thor_inputs as ti
from conftest import have_cuda

pytestmark = pytest.mark.gpu

if have_cuda():
    import paper_1607_05535_b200 as thor

# the tolerances the parity tests use for the two diagnostics (tests/test_gpu_parity.py)
TOL_MASS, TOL_ENERGY = 1e-13, 1e-12


def _agree(st):
    m0, e0 = st.diagnostics()                      # existing path: per-column partials to the host, summed there
    m1, e1 = st.diagnostics_noalloc()              # new path: static device scratch, summed on the device
    assert np.isfinite(m1) and np.isfinite(e1) and m1 > 0 and e1 > 0
    assert abs(m1 - m0) <= TOL_MASS * m0, (m0, m1)
    assert abs(e1 - e0) <= TOL_ENERGY * e0, (e0, e1)
    return m1, e1


def test_noalloc_diagnostics_match_the_existing_path_on_calls_in_a_row():
    cfg = ti.CONFIGS[0]
    g = thor.Grid(cfg["level"], cfg["nv"], cfg["planet"])
    s = ti.initial_state(0, g.view["xyz"])
    st = thor.State(g, *s)
    a = _agree(st)
    b = _agree(st)                                 # second call in a row on the same state: the scratch is reused
    assert a == b                                  # same state, same order of summation: bit-identical
    st.step(2, cfg["dt"], cfg["n_sub"])
    c = _agree(st)                                 # third call, other contents: nothing of the last call is left over
    assert c[1] != a[1]
    # another state and grid shape (32 layers, level 5) shares the same scratch: fewer live entries than slots used before
    cfg2 = ti.CONFIGS[2]
    g2 = thor.Grid(3, cfg2["nv"], cfg2["planet"])
    st2 = thor.State(g2, *ti.rest_state(cfg2["planet"], cfg2["nv"], g2.n_cols, 1.0e5, 300.0))
    _agree(st2)
    _agree(st)                                     # and back: the larger grid again
    st2.close()
    g2.close()
    st.close()
    g.close()


def test_noalloc_diagnostics_reject_grids_beyond_the_static_scratch():
    """Level 7 has 163 842 columns > 65 536: THOR_EINVAL with a message that names the limit; thor_diagnostics works."""
    planet, nv = ti.EARTH, 2
    g = thor.Grid(7, nv, planet, on_device=True)
    st = thor.State(g, *ti.rest_state(planet, nv, g.n_cols, 1.0e5, 300.0))
    with pytest.raises(thor.ThorError) as e:
        st.diagnostics_noalloc()
    assert e.value.code == thor.THOR_EINVAL
    assert "65536" in str(e.value) and "163842" in str(e.value)
    m, en = st.diagnostics()
    assert m > 0 and en > 0
    st.close()
    g.close()
