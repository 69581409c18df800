"""oracle/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain CPU oracle of the THOR HE-VI large step (arXiv 1607.05535), written from PAPER.md with the
readings of SURVEY.md 8(c) / DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never imports
paper_1607_05535_b200 and shares no code with it.

This file is argument marshalling only (ctypes around oracle/thor_oracle.c); grid_oracle.py is the
independent numpy grid generator.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "thor_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
# The SAME source compiled with FMA contraction allowed (a flag, not new arithmetic): the distance between
# the two builds' answers is what a legal change of rounding does to this algorithm on these inputs -- the
# yardstick of the parity tolerance.  Never the reference: parity is against _LIB.
_LIB_FMA = os.path.join(_HERE, "liboracle_fma.so")
# -ffp-contract=off: no FMA contraction, so the oracle's rounding is the plain IEEE one
_CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c99"]
_CFLAGS_FMA = ["-O2", "-ffp-contract=fast", "-mfma", "-fopenmp", "-shared", "-fPIC", "-std=c99"]

_lib = None
_lib_fma = None


def _compile(lib, flags, force):
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        tmp = lib + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc"] + flags + [_SRC, "-o", tmp, "-lm"])
        os.replace(tmp, lib)
    return lib


def build(force=False):
    """Compile thor_oracle.c with gcc (building the checker is not using it): the oracle proper and
    its FMA-contracted twin."""
    _compile(_LIB_FMA, _CFLAGS_FMA, force)
    return _compile(_LIB, _CFLAGS, force)


_D = ctypes.POINTER(ctypes.c_double)
_I = ctypes.POINTER(ctypes.c_int)


class _Planet(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")]


def have_fma():
    """The FMA twin needs a host CPU with the fma instruction set."""
    try:
        with open("/proc/cpuinfo") as f:
            return " fma " in f.read().replace("\n", " ")
    except OSError:
        return False


def _load(fma=False):
    global _lib, _lib_fma
    if fma:
        if _lib_fma is None:
            if not have_fma():
                raise RuntimeError("oracle: the FMA-contracted twin needs a CPU with fma")
            build()
            _lib_fma = _declare(ctypes.CDLL(_LIB_FMA))
        return _lib_fma
    if _lib is None:
        _lib = _declare(ctypes.CDLL(build()))
    return _lib


def _declare(L):
    L.orc_geom_build.restype = ctypes.c_void_p
    L.orc_geom_build.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(_Planet), _D, _I, _D]
    L.orc_geom_free.argtypes = [ctypes.c_void_p]
    L.orc_vertical_ops.argtypes = [ctypes.c_void_p, ctypes.c_int, _D, _D, _D, _D, _D, _D]
    L.orc_geom_set_vertical.restype = ctypes.c_int
    L.orc_geom_set_vertical.argtypes = [ctypes.c_void_p, _D, ctypes.c_int]
    for name in ("Ac", "len", "nrm", "C", "bary"):
        f = getattr(L, "orc_geom_" + name)
        f.restype = _D
        f.argtypes = [ctypes.c_void_p]
    L.orc_geom_deg.restype = _I
    L.orc_geom_deg.argtypes = [ctypes.c_void_p]
    L.orc_hdiv.argtypes = [ctypes.c_void_p, _D, _D]
    L.orc_hgrad.argtypes = [ctypes.c_void_p, _D, _D]
    L.orc_hlap.argtypes = [ctypes.c_void_p, _D, _D]
    for name, nargs in (("orc_dbar", None), ("orc_kd", None), ("orc_tau_d", None)):
        getattr(L, name).restype = ctypes.c_double
    L.orc_dbar.argtypes = [ctypes.c_double, ctypes.c_int]
    L.orc_kd.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_double]
    L.orc_tau_d.argtypes = [ctypes.c_double, ctypes.c_double]
    L.orc_thomas.argtypes = [ctypes.c_int, _D, _D, _D, _D, _D]
    L.orc_centroid_eq13.argtypes = [_D, ctypes.c_int, _D]
    L.orc_step.argtypes = [ctypes.c_void_p, _D, _D, _D, _D, ctypes.c_int, ctypes.c_double, ctypes.c_int, _D, _D, _D]
    L.orc_step_diffusion.argtypes = [ctypes.c_void_p, _D, _D, _D, _D, ctypes.c_int, ctypes.c_double, ctypes.c_int, _D, _D, _D,
                                     ctypes.c_double, ctypes.c_double]
    L.orc_diagnostics.argtypes = [ctypes.c_void_p, _D, _D, _D, _D, _D, _D]
    L.orc_tridiag_coefficients.argtypes = [ctypes.c_void_p, ctypes.c_double, _D, _D, _D, _D, _D]
    L.orc_slow_terms.argtypes = [ctypes.c_void_p] + [_D] * 12
    L.orc_substep.argtypes = [ctypes.c_void_p, ctypes.c_double] + [_D] * 14
    L.orc_diffusion_fluxes.argtypes = [ctypes.c_void_p, _D, _D, _D, _D, ctypes.c_double, _D, _D, _D, _D, _D]
    L.orc_divergence_damping.argtypes = [ctypes.c_void_p, _D, _D, ctypes.c_double, _D]
    L.orc_step_held_suarez.argtypes = [ctypes.c_void_p, _D, _D, _D, _D, ctypes.c_int, ctypes.c_double, ctypes.c_int, _D,
                                       ctypes.c_double, ctypes.c_double]
    L.orc_forcing_held_suarez.argtypes = [ctypes.c_void_p, ctypes.c_double, _D, _D, _D, _D]
    L.orc_step_hot_jupiter.argtypes = [ctypes.c_void_p, _D, _D, _D, _D, ctypes.c_int, ctypes.c_double, ctypes.c_int, _D,
                                       ctypes.c_double, ctypes.c_double]
    L.orc_forcing_hot_jupiter.argtypes = [ctypes.c_void_p, ctypes.c_double, _D, _D, _D]
    L.orc_set_energy_fixer.argtypes = [ctypes.c_int]
    L.orc_geom_set_shallow.argtypes = [ctypes.c_void_p, ctypes.c_int]
    L.orc_num_threads.restype = ctypes.c_int
    L.orc_set_num_threads.argtypes = [ctypes.c_int]
    return L


def _p(a):
    return None if a is None else a.ctypes.data_as(_D)


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return int(_load().orc_num_threads())


def set_num_threads(n):
    """OpenMP threads of the following oracle calls (both builds); results do not depend on it."""
    _load().orc_set_num_threads(int(n))
    if _lib_fma is not None:
        _lib_fma.orc_set_num_threads(int(n))


class Geometry:
    """All geometric coefficients recomputed from the grid description (O2): positions xyz [N][3],
    neighbour lists nbr [N][6] and control-volume vertices C [N][6][3] (None: triangle centroids
    of xyz).  fma=True: the FMA-contracted build of the same source (a rounding yardstick, never the reference).
    NEXT-3: z_interfaces = nv+1 increasing interface altitudes from 0 to z_top (None: uniform layers, R6);
    vert_order = the k of Eq. 8-9 (odd; 1 = linear, the paper's choice)."""

    def __init__(self, xyz, nbr, nv, planet, C=None, fma=False, z_interfaces=None, vert_order=1, shallow=False):
        L = self._L = _load(fma)
        self.xyz = _c(xyz)
        self.nbr = np.ascontiguousarray(nbr, dtype=np.int32)
        self.N = int(self.xyz.shape[0])
        self.nv = int(nv)
        self.planet = dict(planet)
        self._P = _Planet(**{k: float(planet[k]) for k in ("radius", "omega", "gravity", "Rd", "Cp", "p_ref", "z_top")})
        Cin = None if C is None else _c(C)
        assert Cin is None or Cin.shape == (self.N, 6, 3)
        self._h = L.orc_geom_build(self.N, self.nv, ctypes.byref(self._P), _p(self.xyz),
                                   self.nbr.ctypes.data_as(_I), _p(Cin))
        N = self.N
        self.Ac = np.ctypeslib.as_array(L.orc_geom_Ac(self._h), (N,)).copy()
        self.len = np.ctypeslib.as_array(L.orc_geom_len(self._h), (N, 6)).copy()
        self.nrm = np.ctypeslib.as_array(L.orc_geom_nrm(self._h), (N, 6, 3)).copy()
        self.C = np.ctypeslib.as_array(L.orc_geom_C(self._h), (N, 6, 3)).copy()
        self.bary = np.ctypeslib.as_array(L.orc_geom_bary(self._h), (N, 6, 3)).copy()
        self.deg = np.ctypeslib.as_array(L.orc_geom_deg(self._h), (N,)).copy()
        self.dz = planet["z_top"] / nv
        self.z_c = (np.arange(nv) + 0.5) * self.dz
        self.z_h = np.arange(nv + 1) * self.dz
        self.vert_order = int(vert_order)
        if z_interfaces is not None or vert_order != 1:
            zi = None if z_interfaces is None else _c(z_interfaces)
            assert zi is None or zi.shape == (nv + 1,)
            if L.orc_geom_set_vertical(self._h, _p(zi), int(vert_order)) != 0:
                raise ValueError("oracle: bad z_interfaces / vert_order")
            if zi is not None:
                self.z_h = zi.copy()
                self.z_c = 0.5 * (zi[:-1] + zi[1:])
        self.r_c = planet["radius"] + self.z_c
        self.r_h = planet["radius"] + self.z_h
        self.shallow = bool(shallow)
        if self.shallow:                      # NEXT-4, reading RS1: every radius is the planetary radius
            L.orc_geom_set_shallow(self._h, 1)
            self.r_c = np.full(nv, float(planet["radius"]))
            self.r_h = np.full(nv + 1, float(planet["radius"]))

    def __del__(self):
        try:
            if self._h:
                self._L.orc_geom_free(self._h)
                self._h = None
        except Exception:
            pass

    # Eq. 4-6: horizontal divergence of vec [N][nv][3] at radius r_k -> [N][nv]
    def hdiv(self, vec):
        vec = _c(vec)
        assert vec.shape == (self.N, self.nv, 3)
        out = np.empty((self.N, self.nv))
        self._L.orc_hdiv(self._h, _p(vec), _p(out))
        return out

    # Eq. 7 (difference form, projected): horizontal gradient of s [N][nv] -> [N][nv][3]
    def hgrad(self, s):
        s = _c(s)
        assert s.shape == (self.N, self.nv)
        out = np.empty((self.N, self.nv, 3))
        self._L.orc_hgrad(self._h, _p(s), _p(out))
        return out

    # L369-L371: horizontal Laplacian (gradient on the triangles, then Eq. 6) of s [N][nv] at radius r_k
    def hlap(self, s):
        s = _c(s)
        assert s.shape == (self.N, self.nv)
        out = np.empty((self.N, self.nv))
        self._L.orc_hlap(self._h, _p(s), _p(out))
        return out

    def step(self, rho, V, W, p, n_large, dt, n_sub, forcing=None, D_hyp=0.0, D_div=0.0, energy_fixer=False):
        """n_large large steps; returns new (rho, V, W, p); inputs are not modified.  D_hyp, D_div:
        non-dimensional diffusion parameter of Eq. 49 for the hyper-diffusion / divergence damping
        (NEXT-1; 0 = off = the base path).  energy_fixer: NEXT-4, reading RE1 (L215)."""
        if energy_fixer:
            self._L.orc_set_energy_fixer(1)
            try:
                return self.step(rho, V, W, p, n_large, dt, n_sub, forcing, D_hyp, D_div)
            finally:
                self._L.orc_set_energy_fixer(0)
        rho, V, W, p = (_c(x).copy() for x in (rho, V, W, p))
        assert rho.shape == (self.N, self.nv) and V.shape == (self.N, self.nv, 3)
        assert W.shape == (self.N, self.nv + 1) and p.shape == (self.N, self.nv)
        assert n_sub >= 2 and n_sub % 2 == 0
        T_eq = k_T = k_v = None
        if forcing is not None:
            T_eq = None if forcing.get("T_eq") is None else _c(forcing["T_eq"])
            k_T = None if forcing.get("k_T") is None else _c(forcing["k_T"])
            k_v = None if forcing.get("k_v") is None else _c(forcing["k_v"])
        if D_hyp == 0.0 and D_div == 0.0:
            self._L.orc_step(self._h, _p(rho), _p(V), _p(W), _p(p), int(n_large), float(dt), int(n_sub),
                             _p(T_eq), _p(k_T), _p(k_v))
        else:
            self._L.orc_step_diffusion(self._h, _p(rho), _p(V), _p(W), _p(p), int(n_large), float(dt), int(n_sub),
                                       _p(T_eq), _p(k_T), _p(k_v), float(D_hyp), float(D_div))
        return rho, V, W, p

    # NEXT-1 (Eq. 43-48): hyper-diffusion fluxes of a state, and the divergence-damping flux of a momentum field
    def diffusion_fluxes(self, rho, V, W, p, Kd):
        rho, V, W, p = (_c(x) for x in (rho, V, W, p))
        N, nv = self.N, self.nv
        Frho, FV, FW, Fp, Frt = np.empty((N, nv)), np.empty((N, nv, 3)), np.empty((N, nv + 1)), np.empty((N, nv)), np.empty((N, nv))
        self._L.orc_diffusion_fluxes(self._h, _p(rho), _p(V), _p(W), _p(p), float(Kd), _p(Frho), _p(FV), _p(FW), _p(Fp), _p(Frt))
        return Frho, FV, FW, Fp, Frt

    def divergence_damping(self, V, W, Kd):
        V, W = _c(V), _c(W)
        out = np.empty((self.N, self.nv, 3))
        self._L.orc_divergence_damping(self._h, _p(V), _p(W), float(Kd), _p(out))
        return out

    # NEXT-2: Held-Suarez forcing from the evolving sigma (Eq. 51-55); hs = HELD_SUAREZ-like dict
    def step_held_suarez(self, rho, V, W, p, n_large, dt, n_sub, hs, D_hyp=0.0, D_div=0.0):
        rho, V, W, p = (_c(x).copy() for x in (rho, V, W, p))
        h = _c(hs_array(hs))
        self._L.orc_step_held_suarez(self._h, _p(rho), _p(V), _p(W), _p(p), int(n_large), float(dt), int(n_sub), _p(h),
                                     float(D_hyp), float(D_div))
        return rho, V, W, p

    def forcing_held_suarez(self, rho, V, p, dt, hs):
        rho, V, p = (_c(x).copy() for x in (rho, V, p))
        h = _c(hs_array(hs))
        self._L.orc_forcing_held_suarez(self._h, float(dt), _p(rho), _p(V), _p(p), _p(h))
        return V, p

    # NEXT-2, hot Jupiter (Eq. 59-61); hj: dict with HJ_KEYS
    def step_hot_jupiter(self, rho, V, W, p, n_large, dt, n_sub, hj, D_hyp=0.0, D_div=0.0):
        rho, V, W, p = (_c(x).copy() for x in (rho, V, W, p))
        h = _c(np.array([float(hj[k]) for k in HJ_KEYS]))
        self._L.orc_step_hot_jupiter(self._h, _p(rho), _p(V), _p(W), _p(p), int(n_large), float(dt), int(n_sub), _p(h),
                                     float(D_hyp), float(D_div))
        return rho, V, W, p

    def forcing_hot_jupiter(self, rho, p, dt, hj):
        rho, p = _c(rho).copy(), _c(p).copy()
        h = _c(np.array([float(hj[k]) for k in HJ_KEYS]))
        self._L.orc_forcing_hot_jupiter(self._h, float(dt), _p(rho), _p(p), _p(h))
        return p

    def vertical_ops(self, Yc, Xh, order_k=True):
        """NEXT-3 pins: (I_h[Yc], G_h[Yc], I_c[Xh], D_c[Xh]) of one column; order_k: Eq. 8-9 at the order of the
        run, else the linear interpolations of the acoustic system."""
        Yc, Xh = _c(Yc), _c(Xh)
        assert Yc.shape == (self.nv,) and Xh.shape == (self.nv + 1,)
        Ih, Gh, Ic, Dc = np.empty(self.nv + 1), np.empty(self.nv + 1), np.empty(self.nv), np.empty(self.nv)
        self._L.orc_vertical_ops(self._h, int(bool(order_k)), _p(Yc), _p(Xh), _p(Ih), _p(Gh), _p(Ic), _p(Dc))
        return Ih, Gh, Ic, Dc

    def diagnostics(self, rho, V, W, p):
        rho, V, W, p = (_c(x) for x in (rho, V, W, p))
        m = ctypes.c_double()
        e = ctypes.c_double()
        self._L.orc_diagnostics(self._h, _p(rho), _p(V), _p(W), _p(p), ctypes.byref(m), ctypes.byref(e))
        return m.value, e.value

    def tridiag_coefficients(self, delta, h, gt):
        h, gt = _c(h), _c(gt)
        a, b, c = (np.zeros(self.nv + 1) for _ in range(3))
        self._L.orc_tridiag_coefficients(self._h, float(delta), _p(h), _p(gt), _p(a), _p(b), _p(c))
        return a, b, c

    def slow_terms(self, rho, V, W, p):
        rho, V, W, p = (_c(x) for x in (rho, V, W, p))
        N, nv = self.N, self.nv
        out = dict(slowV=np.zeros((N, nv, 3)), slowrho=np.zeros((N, nv)), Svr=np.zeros((N, nv + 1)),
                   slowp=np.zeros((N, nv)), slowrt=np.zeros((N, nv)), h=np.zeros((N, nv)),
                   th=np.zeros((N, nv)), gt=np.zeros((N, nv + 1)))
        self._L.orc_slow_terms(self._h, _p(rho), _p(V), _p(W), _p(p), *[_p(out[k]) for k in
                               ("slowV", "slowrho", "Svr", "slowp", "slowrt", "h", "th", "gt")])
        return out

    def substep(self, delta, stage, dev):
        """One acoustic substep.  stage: dict(h, th, gt, p_t, slowV, slowrho, Svr, slowp, slowrt);
        dev: dict(rho_s, V_s, W_s, p_s, rt).  Returns the updated dev (copies)."""
        st = {k: _c(v) for k, v in stage.items()}
        dv = {k: _c(v).copy() for k, v in dev.items()}
        self._L.orc_substep(self._h, float(delta), _p(st["h"]), _p(st["th"]), _p(st["gt"]), _p(st["p_t"]),
                            _p(st["slowV"]), _p(st["slowrho"]), _p(st["Svr"]), _p(st["slowp"]), _p(st["slowrt"]),
                            _p(dv["rho_s"]), _p(dv["V_s"]), _p(dv["W_s"]), _p(dv["p_s"]), _p(dv["rt"]))
        return dv


def thomas(a, b, c, d):
    """Thomas algorithm on arrays indexed 1..n (index 0 unused)."""
    a, b, c, d = (_c(x) for x in (a, b, c, d))
    n = len(b) - 1
    x = np.zeros(n + 2)
    a2, b2, c2, d2 = (np.concatenate([v, [0.0]]) for v in (a, b, c, d))
    _load().orc_thomas(n, _p(a2), _p(b2), _p(c2), _p(d2), _p(x))
    return x[: n + 1]


def centroid_eq13(r):
    r = _c(r)
    out = np.zeros(3)
    _load().orc_centroid_eq13(_p(r), int(r.shape[0]), _p(out))
    return out


# Eq. 2, 49, 50 (L55, L373-L381)
def dbar(radius, level):
    return float(_load().orc_dbar(float(radius), int(level)))


def kd(D, dbar_, dt):
    return float(_load().orc_kd(float(D), float(dbar_), float(dt)))


def tau_d(dbar_, kd_):
    return float(_load().orc_tau_d(float(dbar_), float(kd_)))


HJ_KEYS = ("T_surf", "Gamma", "dT_stra", "z_stra", "sigma_stra", "dT_EP", "tau_rad")
HS_KEYS = ("T_surf", "dT_y", "dth_z", "T_min", "k_a", "k_s", "k_f", "sigma_b", "p_star")


def hs_array(hs):
    return np.array([float(hs[k]) for k in HS_KEYS])
