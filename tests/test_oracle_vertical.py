"""NEXT-3 pins of the oracle (Eq. 8-9): layers of unequal thickness and
Lagrange interpolation of order k between layer centres and interfaces.  Readings RV1-RV3 of DESIGN.md.
Grids come from the oracle's own generator; nothing comes from the CUDA path."""
import numpy as np
import pytest

import oracle
import thor_inputs as ti
from test_oracle_dynamics import _dense_column_solve


def _column_geometry(nv, planet, z_h=None, order=1):
    """The smallest closed grid (the icosahedron itself, 12 columns): the vertical operators do not look at it."""
    from oracle import grid_oracle
    xyz, nbr, C, _ = grid_oracle.build(0, smooth=False)
    return oracle.Geometry(xyz, nbr, nv, planet, C, z_interfaces=z_h, vert_order=order)


def _random_interfaces(rng, nv, z_top):
    t = rng.uniform(0.4, 1.6, size=nv)
    z = np.concatenate([[0.0], np.cumsum(t)])
    z *= z_top / z[-1]
    z[-1] = z_top
    return z


# --------------------------------------------------------------------------- Eq. 8-9 as such
@pytest.mark.parametrize("order", [1, 3, 5])
def test_lagrange_interpolation_reproduces_polynomials_of_its_degree(order):
    """Eq. 8-9 with k+1 nodes is exact for polynomials of degree <= k.  Away from the ends of the column every
    interface has (k+1)/2 centres on each side; at the first and last (k-1)/2 interior interfaces the window is
    cut by the boundary and the degree falls by one per missing node (RV1)."""
    rng = np.random.default_rng(order)
    nv, planet = 14, dict(ti.EARTH)
    z_h = _random_interfaces(rng, nv, planet["z_top"])
    G = _column_geometry(nv, planet, z_h, order)
    z_c = 0.5 * (z_h[:-1] + z_h[1:])
    assert np.allclose(G.z_c, z_c, rtol=0, atol=0)
    s = planet["z_top"]
    half = (order + 1) // 2
    for deg in range(0, order + 2):
        coef = rng.standard_normal(deg + 1)
        f = lambda z: np.polyval(coef, z / s)
        Ih, _, Ic, _ = G.vertical_ops(f(z_c), f(z_h))
        err_h = np.abs(Ih[1:nv] - f(z_h[1:nv])) / np.abs(coef).sum()
        err_c = np.abs(Ic - f(z_c)) / np.abs(coef).sum()
        for k in range(1, nv):                                   # interface k: centres k-half .. k+half-1 inside 0..nv-1
            nodes = min(k + half - 1, nv - 1) - max(k - half, 0) + 1
            if deg <= nodes - 1:
                assert err_h[k - 1] < 1e-13, (order, deg, k)
        for k in range(nv):                                      # centre k: interfaces k+1-half .. k+half inside 0..nv
            nodes = min(k + half, nv) - max(k + 1 - half, 0) + 1
            if deg <= nodes - 1:
                assert err_c[k] < 1e-13, (order, deg, k)
        if deg == order + 1:                                     # one degree more is NOT reproduced: the order is k, not more
            assert err_h[half:nv - 1 - half].min() > 1e-10
            assert err_c[half:nv - half].min() > 1e-10


def test_interpolation_error_falls_with_the_order():
    """Error of I_h on a smooth profile: ~dz^2 for k = 1, ~dz^4 for k = 3 (interior interfaces)."""
    planet = dict(ti.EARTH)
    f = lambda z: np.exp(-z / 8.0e3) * np.cos(z / 5.0e3)
    err = {}
    for order in (1, 3):
        for nv in (16, 32, 64):
            z_h = ti.stretched_interfaces(planet, nv, 3.0)
            G = _column_geometry(nv, planet, z_h, order)
            Ih, _, _, _ = G.vertical_ops(f(G.z_c), np.zeros(nv + 1))
            err[order, nv] = np.abs(Ih[3:nv - 2] - f(z_h[3:nv - 2])).max()
    for order, rate in ((1, 2.0), (3, 4.0)):
        o1 = np.log2(err[order, 16] / err[order, 32])
        o2 = np.log2(err[order, 32] / err[order, 64])
        assert rate - 0.4 < o1 < rate + 0.6 and rate - 0.3 < o2 < rate + 0.4, (order, o1, o2)
    assert err[3, 64] < 1e-2 * err[1, 64]


def test_gradient_and_divergence_on_unequal_layers_closed_forms():
    """G_h of a linear profile is its slope exactly; D_c[X] with X = c/r_h^2 is exactly 0 (the radial flux
    r^2 X is constant, Eq. 27), and D_c telescopes under the weight r_k^2 dz_k (mass conservation, L339)."""
    rng = np.random.default_rng(3)
    nv, planet = 11, dict(ti.EARTH)
    z_h = _random_interfaces(rng, nv, planet["z_top"])
    G = _column_geometry(nv, planet, z_h, 1)
    _, Gh, _, Dc = G.vertical_ops(3.0 - 2.5e-4 * G.z_c, 7.0 / G.r_h ** 2)
    assert np.abs(Gh[1:nv] + 2.5e-4).max() < 1e-16 + 1e-12 * 2.5e-4
    assert np.abs(Dc).max() < 1e-13 * (7.0 / G.r_h[0] ** 2) / np.diff(z_h).min()
    X = rng.standard_normal(nv + 1)
    X[0] = X[nv] = 0.0
    _, _, _, Dc = G.vertical_ops(np.zeros(nv), X)
    tot = np.sum(Dc * G.r_c ** 2 * np.diff(z_h))
    assert abs(tot) < 1e-12 * np.sum(np.abs(Dc) * G.r_c ** 2 * np.diff(z_h))


# ------------------------------------------------------------------ the step on unequal layers
def _hydrostatic_rest_column(G, planet, p_s, T0, order):
    """Isothermal column with G_h[p]_k + g I[rho]_k = 0 at every interior interface for the interpolation of
    the given order (RV1 window), rho = p/(Rd T0): one linear solve for p_1..p_nv-1 given p_0."""
    nv, g, Rd = G.nv, planet["gravity"], planet["Rd"]
    z_c, z_h = G.z_c, G.z_h
    half = (order + 1) // 2
    A = np.zeros((nv, nv))
    b = np.zeros(nv)
    A[0, 0] = 1.0
    b[0] = p_s * np.exp(-g * z_c[0] / (Rd * T0))
    for k in range(1, nv):
        s = z_c[k] - z_c[k - 1]
        A[k, k] += 1.0 / s
        A[k, k - 1] -= 1.0 / s
        lo, hi = max(k - half, 0), min(k + half - 1, nv - 1)
        nodes = np.arange(lo, hi + 1)
        for j in nodes:
            L = 1.0
            for i in nodes:
                if i != j:
                    L *= (z_h[k] - z_c[i]) / (z_c[j] - z_c[i])
            A[k, j] += g * L / (Rd * T0)
    return np.linalg.solve(A, b)


@pytest.mark.parametrize("order", [1, 3])
def test_rest_state_and_mass_on_stretched_layers(ogrid, order):
    """P12 and P11 on layers of unequal thickness: the discretely hydrostatic isothermal column (balanced with the
    interpolation of the run's order) stays at rest to round-off, and a perturbed state conserves total mass."""
    planet = dict(ti.EARTH)
    nv = 10
    xyz, nbr, C = ogrid(2, True)
    z_h = ti.stretched_interfaces(planet, nv, 4.0)
    G = oracle.Geometry(xyz, nbr, nv, planet, C, z_interfaces=z_h, vert_order=order)
    p_col = _hydrostatic_rest_column(G, planet, 1.0e5, 300.0, order)
    if order == 1:                                                           # the input recipe is the same column
        assert np.abs(p_col - ti.hydrostatic_column(planet, z_h, 1.0e5, np.full(nv, 300.0))).max() < 1e-9
    p = np.tile(p_col, (G.N, 1))
    rho = p / (planet["Rd"] * 300.0)
    V, W = np.zeros((G.N, nv, 3)), np.zeros((G.N, nv + 1))
    r2, V2, W2, p2 = G.step(rho, V, W, p, 5, 600.0, 4)
    assert np.abs(W2).max() < 1e-9 and np.abs(V2).max() < 1e-9
    assert np.abs(r2 - rho).max() < 1e-13 * rho.max() and np.abs(p2 - p).max() < 1e-13 * p.max()
    rng = np.random.default_rng(7 + order)
    T = 300.0 * (1 + rng.uniform(-1e-2, 1e-2, size=rho.shape))
    rho = p / (planet["Rd"] * T)
    vel = rng.uniform(-3, 3, size=V.shape)
    vel -= np.sum(vel * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    W[:, 1:nv] = rng.uniform(-0.2, 0.2, size=(G.N, nv - 1))
    state = (rho, rho[..., None] * vel, W, p)
    m0, e0 = G.diagnostics(*state)
    assert abs(m0 - np.sum(rho * G.Ac[:, None] * (G.r_c ** 2 * np.diff(z_h))[None, :])) < 1e-12 * m0
    new = G.step(*state, 4, 600.0, 4)
    m1, e1 = G.diagnostics(*new)
    assert abs(m1 - m0) < 1e-14 * m0
    assert abs(e1 - e0) < 1e-5 * abs(e0)


def test_uniform_layers_given_explicitly_are_the_uniform_path(ogrid):
    """z_interfaces = k z_top/nv takes the general branch (Lagrange weights, per-layer thickness); it must agree
    with the uniform path (R6) to rounding, and order 1 given explicitly IS the default path bit for bit."""
    cfg = ti.CONFIGS[0]
    xyz, nbr, C = ogrid(2, True)
    nv = cfg["nv"]
    G0 = oracle.Geometry(xyz, nbr, nv, cfg["planet"], C)
    G1 = oracle.Geometry(xyz, nbr, nv, cfg["planet"], C, z_interfaces=np.arange(nv + 1) * (cfg["planet"]["z_top"] / nv))
    G2 = oracle.Geometry(xyz, nbr, nv, cfg["planet"], C, vert_order=1)
    state = ti.initial_state(0, xyz)
    a, b, c = (G.step(*state, 2, cfg["dt"], cfg["n_sub"]) for G in (G0, G1, G2))
    for x, y, z in zip(a, b, c):
        assert np.array_equal(x, z)
    assert np.abs(a[0] - b[0]).max() < 1e-13 * np.abs(a[0]).max() and np.abs(a[3] - b[3]).max() < 1e-13 * np.abs(a[3]).max()
    assert np.abs(a[1] - b[1]).max() < 1e-9 * np.abs(a[1]).max() and np.abs(a[2] - b[2]).max() < 1e-9 * np.abs(a[2]).max()


def test_p10_substep_on_stretched_layers_matches_the_dense_solve(ogrid):
    """P10 on unequal layers: the tridiagonal elimination (R8) against a dense solve of the three fast equations
    written with the per-layer thickness, the centre spacing and the linear weights of the interface."""
    planet = dict(ti.EARTH)
    xyz, nbr, C = ogrid(2, True)
    nv = 7
    z_h = ti.stretched_interfaces(planet, nv, 5.0)
    G = oracle.Geometry(xyz, nbr, nv, planet, C, z_interfaces=z_h, vert_order=3)
    rng = np.random.default_rng(21)
    p = np.tile(ti.hydrostatic_column(planet, z_h, 1.0e5, np.full(nv, 300.0)), (G.N, 1))
    T = 300.0 * (1 + rng.uniform(-2e-2, 2e-2, size=p.shape))
    rho = p / (287.0 * T)
    vel = rng.uniform(-5, 5, size=(G.N, nv, 3))
    vel -= np.sum(vel * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    V = rho[..., None] * vel
    W = np.zeros((G.N, nv + 1))
    W[:, 1:nv] = rng.uniform(-0.5, 0.5, size=(G.N, nv - 1))
    st = G.slow_terms(rho, V, W, p)
    stage = dict(st, p_t=p)
    dev = dict(rho_s=rng.uniform(-1e-3, 1e-3, size=rho.shape), V_s=rng.uniform(-1, 1, size=V.shape),
               W_s=np.zeros_like(W), p_s=rng.uniform(-50, 50, size=p.shape),
               rt=(1e5 / 287.0) * (p / 1e5) ** (1 - 287.0 / 1005.0))
    dev["V_s"] -= np.sum(dev["V_s"] * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    dev["W_s"][:, 1:nv] = rng.uniform(-0.1, 0.1, size=(G.N, nv - 1))
    delta = 200.0
    new = G.substep(delta, stage, dev)
    divV = G.hdiv(new["V_s"])
    divhV = G.hdiv(st["h"][..., None] * new["V_s"])
    for col in (0, 5, G.N - 1):
        Wd, rd, _ = _dense_column_solve(G, delta, col, stage, dev, divV, divhV)
        assert np.abs(new["W_s"][col, 1:nv] - Wd).max() < 1e-11 * np.abs(Wd).max()
        assert np.abs(new["rho_s"][col] - rd).max() < 1e-11 * np.abs(rd).max()
    # g~ is the acoustic system's coefficient: linear interpolation whatever the order of the run (RV2)
    s = np.diff(G.z_c)
    wl, wu = (G.z_c[1:] - z_h[1:nv]) / s, (z_h[1:nv] - G.z_c[:-1]) / s
    gt = (p[0, 1:] - p[0, :-1]) / s / (wl * rho[0, :-1] + wu * rho[0, 1:])
    assert np.abs(st["gt"][0, 1:nv] - gt).max() < 1e-13 * np.abs(gt).max()


def test_higher_order_changes_the_slow_terms_only_where_it_should(ogrid):
    """RV2: order k enters the explicit slow terms (vertical fluxes of u, h, theta; rho and F_r in S_vr; I_c[W] in
    u and the Coriolis term); on a state whose profiles are LINEAR in z and on equal layers, cubic and linear
    interpolation coincide away from nothing at all -- so the slow terms must agree to rounding; on a curved
    profile they differ at second order."""
    planet = dict(ti.EARTH)
    xyz, nbr, C = ogrid(2, True)
    nv = 12
    G1 = oracle.Geometry(xyz, nbr, nv, planet, C, vert_order=1)
    G3 = oracle.Geometry(xyz, nbr, nv, planet, C, vert_order=3)
    z = G1.z_c
    rho = np.tile(1.2 - 2.0e-5 * z, (G1.N, 1))
    p = np.tile(1.0e5 - 2.2 * z, (G1.N, 1))
    V = np.zeros((G1.N, nv, 3))
    W = np.zeros((G1.N, nv + 1))
    a, b = G1.slow_terms(rho, V, W, p), G3.slow_terms(rho, V, W, p)
    assert np.abs(a["Svr"] - b["Svr"]).max() < 1e-12 * np.abs(a["Svr"]).max()
    rho2 = np.tile(1.2 * np.exp(-z / 8.0e3), (G1.N, 1))
    a, b = G1.slow_terms(rho2, V, W, p), G3.slow_terms(rho2, V, W, p)
    d = np.abs(a["Svr"] - b["Svr"])[0, 2:nv - 1]
    # linear interpolation error of rho at the interface: rho''(z_h) dz^2 / 8, times g
    est = planet["gravity"] * 1.2 / 8.0e3 ** 2 * np.exp(-G1.z_h[2:nv - 1] / 8.0e3) * G1.dz ** 2 / 8.0
    assert np.all(np.abs(d / est - 1.0) < 0.1)
