"""paper_1607_05535_b200 -- thin Python binding of the C-ABI in include/thor.h.

Argument marshalling only: every step of the THOR HE-VI hot path (arXiv 1607.05535, Fig. 6) runs
in the CUDA kernels of libthor_b200.so.  Functions carry the names of the C entry points; `Grid`
and `State` are small conveniences over them.  There is no CPU fallback: if the shared library is
missing or no CUDA device is present, device calls raise `ThorError`.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libthor_b200.so")

THOR_OK, THOR_EINVAL, THOR_ENOMEM, THOR_ECUDA = 0, -1, -2, -3

_D = ctypes.POINTER(ctypes.c_double)
_I = ctypes.POINTER(ctypes.c_int)
_V = ctypes.c_void_p


class ThorError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("thor error %d: %s" % (code, msg))
        self.code = code


class thor_planet(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")]


class thor_grid_view(ctypes.Structure):
    _fields_ = [("level", ctypes.c_int), ("n_cols", ctypes.c_int), ("n_layers", ctypes.c_int),
                ("xyz", _D), ("nbr", _I), ("cv_vertex", _D), ("area", _D), ("edge_len", _D),
                ("edge_nrm", _D), ("device_order", _I), ("spring_iterations", ctypes.c_int)]


class thor_forcing(ctypes.Structure):
    _fields_ = [("T_eq", _D), ("k_T", _D), ("k_v", _D), ("resident", ctypes.c_int)]


class thor_held_suarez(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in ("T_surf", "dT_y", "dth_z", "T_min", "k_a", "k_s", "k_f", "sigma_b", "p_star")]


class thor_hot_jupiter(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in ("T_surf", "Gamma", "dT_stra", "z_stra", "sigma_stra", "dT_EP", "tau_rad")]


class thor_diag(ctypes.Structure):
    _fields_ = [("total_mass", ctypes.c_double), ("total_energy", ctypes.c_double)]


# name -> (restype, argtypes); also the list the ABI test checks against include/thor.h
_SIGNATURES = {
    "thor_grid_create": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.POINTER(thor_planet), ctypes.POINTER(_V)]),
    "thor_grid_create_vertical": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.POINTER(thor_planet), _D, ctypes.c_int,
                                                 ctypes.POINTER(_V)]),
    "thor_grid_create_shallow": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.POINTER(thor_planet), _D, ctypes.POINTER(_V)]),
    "thor_grid_create_device": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.POINTER(thor_planet), _D, ctypes.c_int,
                                               ctypes.POINTER(_V)]),
    "thor_grid_get": (ctypes.c_int, [_V, ctypes.POINTER(thor_grid_view)]),
    "thor_grid_destroy": (None, [_V]),
    "thor_state_init": (ctypes.c_int, [_V, _D, _D, _D, _D, _V, ctypes.POINTER(_V)]),
    "thor_state_set": (ctypes.c_int, [_V, _D, _D, _D, _D]),
    "thor_state_get": (ctypes.c_int, [_V, _D, _D, _D, _D]),
    "thor_state_destroy": (None, [_V]),
    "thor_step": (ctypes.c_int, [_V, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.POINTER(thor_forcing)]),
    "thor_state_set_diffusion": (ctypes.c_int, [_V, ctypes.c_double, ctypes.c_double]),
    "thor_state_set_energy_fixer": (ctypes.c_int, [_V, ctypes.c_int]),
    "thor_state_set_held_suarez": (ctypes.c_int, [_V, ctypes.POINTER(thor_held_suarez)]),
    "thor_state_set_hot_jupiter": (ctypes.c_int, [_V, ctypes.POINTER(thor_hot_jupiter)]),
    "thor_acoustic_substeps": (ctypes.c_int, [_V, ctypes.c_int, ctypes.c_double, ctypes.c_int]),
    "thor_diagnostics": (ctypes.c_int, [_V, ctypes.POINTER(thor_diag)]),
    "thor_diagnostics_noalloc": (ctypes.c_int, [_V, ctypes.POINTER(thor_diag)]),
    "thor_apply_div": (ctypes.c_int, [_V, _D, _D]),
    "thor_apply_grad": (ctypes.c_int, [_V, _D, _D]),
    "thor_apply_div_device": (ctypes.c_int, [_V, _V, _V, _V, _V, _V]),
    "thor_apply_grad_device": (ctypes.c_int, [_V, _V, _V, _V, _V, _V]),
    "thor_apply_lap": (ctypes.c_int, [_V, _D, _D]),
    "thor_apply_lap_device": (ctypes.c_int, [_V, _V, _V, _V]),
    "thor_launch_count": (ctypes.c_longlong, []),
    "thor_last_error": (ctypes.c_char_p, []),
}

_lib = None


def load_library():
    """dlopen libthor_b200.so (built in-tree by paper_1607_05535_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ThorError(THOR_ECUDA, "%s is missing: run `python -m paper_1607_05535_b200.build` "
                                        "(there is no CPU fallback)" % LIB_PATH)
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(code):
    if code != THOR_OK:
        raise ThorError(code, load_library().thor_last_error().decode())


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != tuple(shape):
        raise ThorError(THOR_EINVAL, "expected shape %s, got %s" % (tuple(shape), a.shape))
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_D)


# ---------------------------------------------------------------------------------------------
# the C entry points, same names
# ---------------------------------------------------------------------------------------------
def thor_grid_create(level, n_layers, planet):
    P = thor_planet(**{k: float(planet[k]) for k in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")})
    h = _V()
    _check(load_library().thor_grid_create(int(level), int(n_layers), ctypes.byref(P), ctypes.byref(h)))
    return h


def thor_grid_create_vertical(level, n_layers, planet, z_interfaces=None, order_k=1):
    P = thor_planet(**{k: float(planet[k]) for k in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")})
    z = None if z_interfaces is None else _f64(z_interfaces, (int(n_layers) + 1,))
    h = _V()
    _check(load_library().thor_grid_create_vertical(int(level), int(n_layers), ctypes.byref(P), _ptr(z), int(order_k),
                                                    ctypes.byref(h)))
    return h


def thor_grid_create_shallow(level, n_layers, planet, z_interfaces=None):
    P = thor_planet(**{k: float(planet[k]) for k in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")})
    z = None if z_interfaces is None else _f64(z_interfaces, (int(n_layers) + 1,))
    h = _V()
    _check(load_library().thor_grid_create_shallow(int(level), int(n_layers), ctypes.byref(P), _ptr(z), ctypes.byref(h)))
    return h


def thor_grid_create_device(level, n_layers, planet, z_interfaces=None, order_k=1):
    P = thor_planet(**{k: float(planet[k]) for k in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")})
    z = None if z_interfaces is None else _f64(z_interfaces, (int(n_layers) + 1,))
    h = _V()
    _check(load_library().thor_grid_create_device(int(level), int(n_layers), ctypes.byref(P), _ptr(z), int(order_k),
                                                  ctypes.byref(h)))
    return h


def thor_grid_get(grid):
    v = thor_grid_view()
    _check(load_library().thor_grid_get(grid, ctypes.byref(v)))
    N = v.n_cols
    as_np = np.ctypeslib.as_array
    return dict(level=v.level, n_cols=N, n_layers=v.n_layers, spring_iterations=v.spring_iterations,
                xyz=as_np(v.xyz, (N, 3)).copy(), nbr=as_np(v.nbr, (N, 6)).copy(),
                cv_vertex=as_np(v.cv_vertex, (N, 6, 3)).copy(), area=as_np(v.area, (N,)).copy(),
                edge_len=as_np(v.edge_len, (N, 6)).copy(), edge_nrm=as_np(v.edge_nrm, (N, 6, 3)).copy(),
                device_order=as_np(v.device_order, (N,)).copy())


def thor_grid_destroy(grid):
    load_library().thor_grid_destroy(grid)


def thor_state_init(grid, rho, mom_h, W, p, cuda_stream=None):
    h = _V()
    _check(load_library().thor_state_init(grid, _ptr(rho), _ptr(mom_h), _ptr(W), _ptr(p), _V(cuda_stream or 0),
                                          ctypes.byref(h)))
    return h


def thor_state_set(state, rho, mom_h, W, p):
    _check(load_library().thor_state_set(state, _ptr(rho), _ptr(mom_h), _ptr(W), _ptr(p)))


def thor_state_get(state, rho, mom_h, W, p):
    _check(load_library().thor_state_get(state, _ptr(rho), _ptr(mom_h), _ptr(W), _ptr(p)))


def thor_state_destroy(state):
    load_library().thor_state_destroy(state)


def thor_step(state, n_large, dt, n_acoustic_substeps, forcing=None):
    _check(load_library().thor_step(state, int(n_large), float(dt), int(n_acoustic_substeps),
                                    None if forcing is None else ctypes.byref(forcing)))


def thor_state_set_diffusion(state, D_hyper, D_div):
    _check(load_library().thor_state_set_diffusion(state, float(D_hyper), float(D_div)))


def thor_state_set_energy_fixer(state, on):
    _check(load_library().thor_state_set_energy_fixer(state, int(bool(on))))


def thor_state_set_held_suarez(state, hs):
    """hs: dict with the fields of thor_held_suarez, or None to switch the evolving-sigma forcing off."""
    if hs is None:
        _check(load_library().thor_state_set_held_suarez(state, None))
        return
    H = thor_held_suarez(**{k: float(hs[k]) for k, _ in thor_held_suarez._fields_})
    _check(load_library().thor_state_set_held_suarez(state, ctypes.byref(H)))


def thor_state_set_hot_jupiter(state, hj):
    if hj is None:
        _check(load_library().thor_state_set_hot_jupiter(state, None))
        return
    J = thor_hot_jupiter(**{k: float(hj[k]) for k, _ in thor_hot_jupiter._fields_})
    _check(load_library().thor_state_set_hot_jupiter(state, ctypes.byref(J)))


def thor_acoustic_substeps(state, n_substeps, delta, which=3):
    _check(load_library().thor_acoustic_substeps(state, int(n_substeps), float(delta), int(which)))


def thor_diagnostics(state):
    d = thor_diag()
    _check(load_library().thor_diagnostics(state, ctypes.byref(d)))
    return d.total_mass, d.total_energy


def thor_diagnostics_noalloc(state):
    d = thor_diag()
    _check(load_library().thor_diagnostics_noalloc(state, ctypes.byref(d)))
    return d.total_mass, d.total_energy


def thor_apply_div(grid, vec, out):
    _check(load_library().thor_apply_div(grid, _ptr(vec), _ptr(out)))


def thor_apply_grad(grid, s, out):
    _check(load_library().thor_apply_grad(grid, _ptr(s), _ptr(out)))


def thor_apply_div_device(grid, vx, vy, vz, out, cuda_stream=None):
    """vx, vy, vz, out: integer DEVICE addresses of [n_cols][n_layers] arrays in device column order."""
    _check(load_library().thor_apply_div_device(grid, _V(vx), _V(vy), _V(vz), _V(out), _V(cuda_stream or 0)))


def thor_apply_grad_device(grid, s, gx, gy, gz, cuda_stream=None):
    _check(load_library().thor_apply_grad_device(grid, _V(s), _V(gx), _V(gy), _V(gz), _V(cuda_stream or 0)))


def thor_apply_lap(grid, s, out):
    _check(load_library().thor_apply_lap(grid, _ptr(s), _ptr(out)))


def thor_apply_lap_device(grid, s, out, cuda_stream=None):
    _check(load_library().thor_apply_lap_device(grid, _V(s), _V(out), _V(cuda_stream or 0)))


def thor_launch_count():
    return int(load_library().thor_launch_count())


def thor_last_error():
    return load_library().thor_last_error().decode()


# ---------------------------------------------------------------------------------------------
# conveniences (ownership + shapes); still no arithmetic
# ---------------------------------------------------------------------------------------------
class Grid:
    def __init__(self, level, n_layers, planet, z_interfaces=None, order_k=1, on_device=False, shallow=False):
        self.planet = dict(planet)
        if shallow:
            if order_k != 1 or on_device:
                raise ThorError(THOR_EINVAL, "shallow-atmosphere grids: linear vertical interpolation, host generator")
            self._h = thor_grid_create_shallow(level, n_layers, planet, z_interfaces)
        elif on_device:
            self._h = thor_grid_create_device(level, n_layers, planet, z_interfaces, order_k)
        elif z_interfaces is None and order_k == 1:
            self._h = thor_grid_create(level, n_layers, planet)
        else:
            self._h = thor_grid_create_vertical(level, n_layers, planet, z_interfaces, order_k)
        self.view = thor_grid_get(self._h)
        self.n_cols, self.n_layers, self.level = self.view["n_cols"], self.view["n_layers"], self.view["level"]

    @property
    def handle(self):
        return self._h

    def apply_div(self, vec):
        vec = _f64(vec, (self.n_cols, self.n_layers, 3))
        out = np.empty((self.n_cols, self.n_layers))
        thor_apply_div(self._h, vec, out)
        return out

    def apply_grad(self, s):
        s = _f64(s, (self.n_cols, self.n_layers))
        out = np.empty((self.n_cols, self.n_layers, 3))
        thor_apply_grad(self._h, s, out)
        return out

    def apply_lap(self, s):
        s = _f64(s, (self.n_cols, self.n_layers))
        out = np.empty((self.n_cols, self.n_layers))
        thor_apply_lap(self._h, s, out)
        return out

    def close(self):
        if self._h is not None:
            thor_grid_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class State:
    def __init__(self, grid, rho, mom_h, W, p, cuda_stream=None):
        self.grid = grid
        N, nv = grid.n_cols, grid.n_layers
        self._shapes = ((N, nv), (N, nv, 3), (N, nv + 1), (N, nv))
        arrs = [_f64(a, s) for a, s in zip((rho, mom_h, W, p), self._shapes)]
        self._h = thor_state_init(grid.handle, *arrs, cuda_stream=cuda_stream)
        self._forcing = None
        self._forcing_keep = None

    @property
    def handle(self):
        return self._h

    def set(self, rho, mom_h, W, p):
        thor_state_set(self._h, *[_f64(a, s) for a, s in zip((rho, mom_h, W, p), self._shapes)])

    def get(self, out=None):
        """out: four caller-owned C-contiguous float64 arrays of the state's shapes (checked: the library writes
        through their raw pointers), or None for fresh ones."""
        if out is None:
            out = tuple(np.empty(s) for s in self._shapes)
        else:
            out = tuple(out)
            if len(out) != 4:
                raise ThorError(THOR_EINVAL, "State.get: need four output arrays (rho, mom_h, W, p)")
            for a, shp in zip(out, self._shapes):
                if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.shape == tuple(shp)
                        and a.flags["C_CONTIGUOUS"] and a.flags["WRITEABLE"]):
                    raise ThorError(THOR_EINVAL, "State.get: output arrays must be writeable C-contiguous float64 of shape %s" % (tuple(shp),))
        thor_state_get(self._h, *out)
        return out

    def step(self, n_large, dt, n_acoustic_substeps, forcing=None):
        """forcing: None, or dict(T_eq=, k_T=, k_v=) of host arrays (uploaded on first use and kept
        resident while the same dict object is passed again)."""
        f = None
        if forcing is not None:
            if forcing is self._forcing_keep:
                f = self._forcing
                f.resident = 1
            else:
                N, nv = self.grid.n_cols, self.grid.n_layers
                arrs = {k: (None if forcing.get(k) is None else _f64(forcing[k], (N, nv))) for k in ("T_eq", "k_T", "k_v")}
                f = thor_forcing(_ptr(arrs["T_eq"]), _ptr(arrs["k_T"]), _ptr(arrs["k_v"]), 0)
                self._forcing, self._forcing_keep, self._forcing_arrays = f, forcing, arrs
        thor_step(self._h, n_large, dt, n_acoustic_substeps, f)

    def set_diffusion(self, D_hyper, D_div=None):
        """NEXT-1: hyper-diffusion and divergence damping parameter D of Eq. 49 (D_div defaults to D_hyper, L367)."""
        thor_state_set_diffusion(self._h, D_hyper, D_hyper if D_div is None else D_div)

    def set_energy_fixer(self, on=True):
        """NEXT-4: the energy fixer of L215 (reading RE1) for the following steps."""
        thor_state_set_energy_fixer(self._h, on)

    def set_held_suarez(self, hs):
        thor_state_set_held_suarez(self._h, hs)

    def set_hot_jupiter(self, hj):
        thor_state_set_hot_jupiter(self._h, hj)

    def acoustic_substeps(self, n_substeps, delta, which=3):
        thor_acoustic_substeps(self._h, n_substeps, delta, which)

    def diagnostics(self):
        return thor_diagnostics(self._h)

    def diagnostics_noalloc(self):
        """thor_diagnostics without any allocation (static device scratch; at most 65 536 columns)."""
        return thor_diagnostics_noalloc(self._h)

    def close(self):
        if self._h is not None:
            thor_state_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
