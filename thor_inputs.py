"""thor_inputs.py -- seeded synthetic inputs shared by the oracle and the CUDA library.

This module holds NONE of the method's arithmetic (no stencil, no solve, no time stepping): only
the five workload configurations of BASELINE.json, the seeded initial states and forcing tables
(recipes of SURVEY.md 8(d), restated in DESIGN.md), and closed-form test fields with their exact
derivatives.  All arrays are numpy float64 in CANONICAL order: column index = the grid generator's
numbering, layer fastest; rho,p [N][nv]; V [N][nv][3] (Cartesian, tangent to the sphere);
W [N][nv+1] on interfaces with both ends zero.

The paper's workloads are analytic forcings on a rest state (Held-Suarez, and
a tidally locked hot Jupiter, L508-L529), not data sets; the configs below take their shapes
(g-level, layer count, constants, dt/n, forcing form) and stand in for them.
"""
import math

import numpy as np

SEED0 = 160705535

EARTH = dict(radius=6.371e6, omega=7.292e-5, gravity=9.8, Rd=287.0, Cp=1005.0, p_ref=1.0e5, z_top=36.0e3)
_HJ_H = 3779.0 * 1500.0 / 9.42                       # scale height Rd T0 / g
HOT_JUPITER = dict(radius=9.44e7, omega=2.06e-5, gravity=9.42, Rd=3779.0, Cp=13226.0, p_ref=1.0e5,
                   z_top=_HJ_H * math.log(1.0e7 / 1.0e5))

# Held-Suarez forcing parameters (Eq. 53-55): k_f = 1/day, sigma_b = 0.7, k_a = 1/40 d,
# k_s = 1/4 d, (Delta T)_y = 60 K, 315 K, 200 K are printed; (Delta theta)_z and p* are not (G14): the
# benchmark's published 10 K and the reference pressure 1e5 Pa are used.
HELD_SUAREZ = dict(T_surf=315.0, dT_y=60.0, dth_z=10.0, T_min=200.0, k_a=1.0 / (40 * 86400.0), k_s=1.0 / (4 * 86400.0),
                   k_f=1.0 / 86400.0, sigma_b=0.7, p_star=1.0e5)

# Hot-Jupiter benchmark of the paper (Table 1): forcing parameters of Eq. 59-61 and the
# planet; the surface pressure is not printed (1e5 Pa, the reference pressure, is used).
HOT_JUPITER_FORCING = dict(T_surf=1600.0, Gamma=2.0e-4, dT_stra=10.0, z_stra=2.0e6, sigma_stra=0.12, dT_EP=300.0, tau_rad=1.5e5)
PAPER_HOT_JUPITER = dict(radius=1.0e8, omega=2.1e-5, gravity=8.0, Rd=3779.0, Cp=13226.5, p_ref=1.0e5, z_top=4.875e6)

# BASELINE.json configs (index = config number).  n_large is the run length used for parity.
CONFIGS = {
    0: dict(name="cfg0_level4x8_earth", level=4, nv=8, planet=EARTH, p_s=1.0e5, T0=300.0,
            dt=1800.0, n_sub=4, n_large=10, forcing=None, init="perturbed"),
    1: dict(name="cfg1_operator_sweep", levels=(5, 6, 7), nv=32, planet=EARTH),
    2: dict(name="cfg2_level5x32_earth", level=5, nv=32, planet=EARTH, p_s=1.0e5, T0=300.0,
            dt=1200.0, n_sub=6, n_large=500, forcing="earth", init="noise_T", noise=0.1),
    3: dict(name="cfg3_level6x32_hotjupiter", level=6, nv=32, planet=HOT_JUPITER, p_s=1.0e7, T0=1500.0,
            dt=300.0, n_sub=8, n_large=100, forcing="hotjupiter", init="noise_rel", noise=1.0e-4),
    4: dict(name="cfg4_level7x64_hotjupiter", level=7, nv=64, planet=HOT_JUPITER, p_s=1.0e7, T0=1500.0,
            dt=150.0, n_sub=10, n_large=50, forcing="hotjupiter", init="noise_rel", noise=1.0e-4),
}


def n_columns(level):
    """Eq. 1."""
    return 2 + 10 * 4 ** level


def substeps_per_large_step(n_sub):
    """1 + n/2 + n acoustic substeps are executed per large step."""
    return 1 + n_sub // 2 + n_sub


def vertical_grid(planet, nv):
    dz = planet["z_top"] / nv
    z_c = (np.arange(nv) + 0.5) * dz
    z_h = np.arange(nv + 1) * dz
    return dz, z_c, z_h


def hydrostatic_isothermal(planet, nv, p_s, T0):
    """Pressure column of an isothermal atmosphere in DISCRETE hydrostatic balance (pin P12):
    (p_k - p_k-1)/dz + g (rho_k-1 + rho_k)/2 = 0 with rho = p/(Rd T0)."""
    dz, z_c, _ = vertical_grid(planet, nv)
    g, Rd = planet["gravity"], planet["Rd"]
    q = g * dz / (2.0 * Rd * T0)
    p = np.empty(nv)
    p[0] = p_s * math.exp(-g * z_c[0] / (Rd * T0))
    for k in range(1, nv):
        p[k] = p[k - 1] * (1.0 - q) / (1.0 + q)
    return p


def stretched_interfaces(planet, nv, ratio):
    """nv+1 interface altitudes from 0 to z_top whose layer thickness grows geometrically, top/bottom = ratio
    (NEXT-3 workloads: thin layers near the surface)."""
    t = ratio ** (np.arange(nv) / max(nv - 1, 1))
    z = np.concatenate([[0.0], np.cumsum(t)])
    z *= planet["z_top"] / z[-1]
    z[-1] = planet["z_top"]
    return z


def hydrostatic_column(planet, z_h, p_s, T_c):
    """Pressure column in DISCRETE hydrostatic balance for layer-centre temperatures T_c on layers bounded by
    z_h (centres at the midpoints): (p_k - p_k-1)/(z_k - z_k-1) + g (wl rho_k-1 + wu rho_k) = 0 with
    rho = p/(Rd T) and the linear weights of the interface between the two centres; p_0 from the surface
    pressure with the lowest layer's temperature.  Uniform layers and constant T: hydrostatic_isothermal."""
    z_h = np.asarray(z_h, dtype=np.float64)
    z_c = 0.5 * (z_h[:-1] + z_h[1:])
    g, Rd = planet["gravity"], planet["Rd"]
    nv = z_c.size
    p = np.empty(nv)
    p[0] = p_s * math.exp(-g * z_c[0] / (Rd * T_c[0]))
    for k in range(1, nv):
        s = z_c[k] - z_c[k - 1]
        wl, wu = (z_c[k] - z_h[k]) / s, (z_h[k] - z_c[k - 1]) / s
        p[k] = p[k - 1] * (1.0 / s - g * wl / (Rd * T_c[k - 1])) / (1.0 / s + g * wu / (Rd * T_c[k]))
    return p


def benchmark_column(planet, z_h, p_s, T_of):
    """Initial column of the paper's Earth benchmark ("the same temperature profile in every column
    taken from the function T_eq at the equator in hydrostatic equilibrium"): layer-centre temperatures
    T_k = T_of(z_k, p_k, p_s) with the pressure in DISCRETE hydrostatic balance (hydrostatic_column).
    T_eq depends on the pressure itself (Eq. 54), so the pair is found by fixed-point iteration (a contraction:
    the profile moves p by O(dT/T) per sweep); returns (p, T)."""
    z_h = np.asarray(z_h, dtype=np.float64)
    z_c = 0.5 * (z_h[:-1] + z_h[1:])
    T = np.full(z_c.size, T_of(z_c[:1], np.array([p_s]), p_s)[0])
    p = hydrostatic_column(planet, z_h, p_s, T)
    for _ in range(200):
        T_new = T_of(z_c, p, p_s)
        p_new = hydrostatic_column(planet, z_h, p_s, T_new)
        done = np.abs(p_new - p).max() <= 1e-14 * p_s
        p, T = p_new, T_new
        if done:
            break
    return p, T


def held_suarez_equator_profile(planet, hs):
    """T_eq of Eq. 54 at the equator (latitude 0) as a function of pressure: the initial profile of L452."""
    kappa = planet["Rd"] / planet["Cp"]

    def T_of(z, p, p_s):
        pr = p / hs["p_star"]
        return np.maximum(hs["T_min"], (hs["T_surf"] - hs["dth_z"] * np.log(pr)) * pr ** kappa)
    return T_of


def rest_state(planet, nv, n_cols, p_s, T0):
    p_col = hydrostatic_isothermal(planet, nv, p_s, T0)
    p = np.tile(p_col, (n_cols, 1))
    rho = p / (planet["Rd"] * T0)
    V = np.zeros((n_cols, nv, 3))
    W = np.zeros((n_cols, nv + 1))
    return rho, V, W, p


def initial_state(cfg_id, xyz):
    """Seeded initial state of config `cfg_id` on the columns at unit vectors xyz [N][3]."""
    cfg = CONFIGS[cfg_id]
    planet, nv = cfg["planet"], cfg["nv"]
    N = xyz.shape[0]
    rng = np.random.default_rng(SEED0 + cfg_id)
    rho, V, W, p = rest_state(planet, nv, N, cfg["p_s"], cfg["T0"])
    Rd = planet["Rd"]
    if cfg["init"] == "perturbed":
        eps = rng.uniform(-1e-3, 1e-3, size=(N, nv))
        T = cfg["T0"] * (1.0 + eps)
        rho = p / (Rd * T)
        vel = rng.uniform(-0.1, 0.1, size=(N, nv, 3))
        rhat = xyz[:, None, :]
        vel = vel - np.sum(vel * rhat, axis=-1, keepdims=True) * rhat      # tangent plane
        V = rho[..., None] * vel
        w = rng.uniform(-0.1, 0.1, size=(N, nv + 1))
        w[:, 0] = 0.0
        w[:, nv] = 0.0
        W = np.zeros((N, nv + 1))
        W[:, 1:nv] = 0.5 * (rho[:, :-1] + rho[:, 1:]) * w[:, 1:nv]
    elif cfg["init"] == "noise_T":
        T = cfg["T0"] + rng.uniform(-cfg["noise"], cfg["noise"], size=(N, nv))
        rho = p / (Rd * T)
    elif cfg["init"] == "noise_rel":
        T = cfg["T0"] * (1.0 + rng.uniform(-cfg["noise"], cfg["noise"], size=(N, nv)))
        rho = p / (Rd * T)
    else:
        raise ValueError(cfg["init"])
    return (np.ascontiguousarray(rho), np.ascontiguousarray(V), np.ascontiguousarray(W), np.ascontiguousarray(p))


def forcing_tables(cfg_id, xyz):
    """Per-cell forcing tables T_eq, k_T, k_v ([N][nv] each, or None), fixed in time (reading R9),
    built from the initial hydrostatic pressure column.  None for configs without forcing."""
    cfg = CONFIGS[cfg_id]
    if cfg.get("forcing") is None:
        return None
    planet, nv = cfg["planet"], cfg["nv"]
    N = xyz.shape[0]
    rng = np.random.default_rng(SEED0 + 1000 + cfg_id)
    p_col = hydrostatic_isothermal(planet, nv, cfg["p_s"], cfg["T0"])
    p = np.tile(p_col, (N, 1))
    lat = np.arcsin(np.clip(xyz[:, 2], -1.0, 1.0))[:, None]
    lon = np.arctan2(xyz[:, 1], xyz[:, 0])[:, None]
    day = 86400.0
    if cfg["forcing"] == "earth":
        # forms of Eq. 53-55 (restored per G14); (Delta theta)_z is seeded
        dTy = 60.0
        dthz = rng.uniform(5.0, 15.0)
        kappa = planet["Rd"] / planet["Cp"]
        sigma = p / cfg["p_s"]
        pr = p / planet["p_ref"]
        T_eq = np.maximum(200.0, (315.0 - dTy * np.sin(lat) ** 2 - dthz * np.log(pr) * np.cos(lat) ** 2) * pr ** kappa)
        ramp = np.maximum(0.0, (sigma - 0.7) / 0.3)
        k_a, k_s, k_f = 1.0 / (40 * day), 1.0 / (4 * day), 1.0 / day
        k_T = k_a + (k_s - k_a) * ramp * np.cos(lat) ** 4
        k_v = k_f * ramp * np.ones_like(lat)
        return dict(T_eq=np.ascontiguousarray(T_eq), k_T=np.ascontiguousarray(k_T), k_v=np.ascontiguousarray(k_v))
    if cfg["forcing"] == "hotjupiter":
        # day-night form of Eq. 59; K_v = 0 (L512)
        lon0 = rng.uniform(0.0, 2 * np.pi)
        lp = np.log10(p)
        wgt = np.clip((7.0 - lp) / 2.0, 0.0, 1.0)
        T_eq = 1300.0 + 500.0 * wgt * np.cos(lon - lon0) * np.cos(lat)
        tau = 10.0 ** np.clip(4.0 + 1.5 * (lp - 5.0), 4.0, 7.0)
        k_T = 1.0 / tau
        return dict(T_eq=np.ascontiguousarray(T_eq), k_T=np.ascontiguousarray(k_T), k_v=None)
    raise ValueError(cfg["forcing"])


# --------------------------------------------------------------------------------------------
# Closed-form test fields on the unit sphere
# --------------------------------------------------------------------------------------------

def _legendre_derivative_coefficients(l, m):
    """q_j with r^(l-m) P_l^(m)(z/r) = sum_j q_j z^(l-m-2j) (r^2)^j  (m-th derivative of P_l)."""
    q = []
    for j in range(l // 2 + 1):
        n = l - 2 * j
        if n - m < 0:
            break
        c = (-1) ** j * math.comb(l, j) * math.comb(2 * l - 2 * j, l) / 2.0 ** l
        c *= math.factorial(n) / math.factorial(n - m)
        q.append(c)
    return q


def _xy_powers(x, y, mmax):
    """A_m + i B_m = (x + i y)^m for m = 0..mmax."""
    zc = x + 1j * y
    out = [np.ones_like(zc)]
    for _ in range(mmax):
        out.append(out[-1] * zc)
    return out


def real_sph_harm(xyz, lmax):
    """Real orthonormal spherical harmonics Y_lm on unit vectors xyz [N][3], evaluated as
    homogeneous harmonic polynomials H(x,y,z) so that the poles need no special case.
    Returns (Y [N][K], gradY [N][K][3], ell [K]) with K = (lmax+1)^2 and gradY the tangential
    gradient on the unit sphere: grad_h Y = grad H - l H r  (Euler's theorem)."""
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    pw = _xy_powers(x, y, lmax)
    N = xyz.shape[0]
    Ys, Gs, ells = [], [], []
    for l in range(lmax + 1):
        for m in range(0, l + 1):
            q = _legendre_derivative_coefficients(l, m)
            Q = np.zeros(N)
            Qz = np.zeros(N)
            Qr = np.zeros(N)
            for j, c in enumerate(q):
                e = l - m - 2 * j
                Q += c * z ** e
                if e > 0:
                    Qz += c * e * z ** (e - 1)
                Qr += c * j * z ** e
            norm = math.sqrt((2 * l + 1) / (4 * math.pi) * math.factorial(l - m) / math.factorial(l + m))
            if m > 0:
                norm *= math.sqrt(2.0)
            gQ = np.stack([2 * x * Qr, 2 * y * Qr, Qz + 2 * z * Qr], axis=-1)
            kinds = ("c",) if m == 0 else ("c", "s")
            for kind in kinds:
                if kind == "c":
                    Am = pw[m].real
                    dAx = m * pw[m - 1].real if m > 0 else np.zeros(N)
                    dAy = -m * pw[m - 1].imag if m > 0 else np.zeros(N)
                else:
                    Am = pw[m].imag
                    dAx = m * pw[m - 1].imag
                    dAy = m * pw[m - 1].real
                H = norm * Am * Q
                gH = norm * (np.stack([dAx * Q, dAy * Q, np.zeros(N)], axis=-1) + Am[:, None] * gQ)
                Ys.append(H)
                Gs.append(gH - l * H[:, None] * xyz)
                ells.append(l)
    return np.stack(Ys, axis=1), np.stack(Gs, axis=1), np.array(ells)


def harmonic_test_fields(xyz, planet, nv, seed, lmax=8):
    """Config 1 fields: scalar s = f(z) sum a Y, vector v = f(z)(grad_h chi + r x grad_h psi),
    with N(0,1) coefficients and f(z) = 1 + z/z_top, and their exact horizontal gradient /
    divergence at radius r_k (unit-sphere result / r_k).  All [N][nv]([3])."""
    rng = np.random.default_rng(seed)
    Y, gY, ell = real_sph_harm(xyz, lmax)
    K = Y.shape[1]
    a, b, c = rng.standard_normal(K), rng.standard_normal(K), rng.standard_normal(K)
    dz, z_c, _ = vertical_grid(planet, nv)
    f = 1.0 + z_c / planet["z_top"]
    r_c = planet["radius"] + z_c
    s1 = Y @ a
    gs1 = np.einsum("nkd,k->nd", gY, a)
    gchi = np.einsum("nkd,k->nd", gY, b)
    gpsi = np.einsum("nkd,k->nd", gY, c)
    v1 = gchi + np.cross(xyz, gpsi)
    lap_chi = -(Y * (ell * (ell + 1))[None, :]) @ b
    s = s1[:, None] * f[None, :]
    v = v1[:, None, :] * f[None, :, None]
    grad_exact = gs1[:, None, :] * (f / r_c)[None, :, None]
    div_exact = lap_chi[:, None] * (f / r_c)[None, :]
    return dict(s=np.ascontiguousarray(s), v=np.ascontiguousarray(v),
                grad_exact=np.ascontiguousarray(grad_exact), div_exact=np.ascontiguousarray(div_exact))


def heikes_randall_fields(xyz, m, n):
    """Test functions of Eq. 14-16 (with G16): alpha = sin(lon),
    beta = cos(m lon) cos^4(n lat), v = alpha grad beta, on the unit sphere.  Returns beta [N],
    v [N][3], exact grad beta [N][3] and exact div v [N].  The two polar columns (cos lat = 0)
    take the limit value 0 of every term that carries 1/cos(lat) (n odd)."""
    lat = np.arcsin(np.clip(xyz[:, 2], -1.0, 1.0))
    lon = np.arctan2(xyz[:, 1], xyz[:, 0])
    cl = np.cos(lat)
    pole = cl < 1e-12
    icl = np.where(pole, 0.0, 1.0 / np.where(pole, 1.0, cl))
    c, s = np.cos(n * lat), np.sin(n * lat)
    e_lon = np.stack([-np.sin(lon), np.cos(lon), np.zeros_like(lon)], axis=-1)
    e_lat = np.stack([-np.sin(lat) * np.cos(lon), -np.sin(lat) * np.sin(lon), np.cos(lat)], axis=-1)
    beta = np.cos(m * lon) * c ** 4
    db_dlon = -m * np.sin(m * lon) * c ** 4
    db_dlat = -4 * n * np.cos(m * lon) * c ** 3 * s
    grad_beta = (db_dlon * icl)[:, None] * e_lon + db_dlat[:, None] * e_lat
    alpha = np.sin(lon)
    v = alpha[:, None] * grad_beta
    lap_beta = (-m * m * np.cos(m * lon) * c ** 4 * icl ** 2
                - 4 * n * np.cos(m * lon) * (-np.sin(lat) * icl * c ** 3 * s + n * (c ** 4 - 3 * c ** 2 * s ** 2)))
    galpha_gbeta = np.cos(lon) * db_dlon * icl ** 2
    div_v = galpha_gbeta + alpha * lap_beta
    return dict(beta=beta, v=v, grad_beta=grad_beta, div_v=div_v)
