"""NEXT-4 pins of the oracle: the shallow-atmosphere approximation (reading RS1 of DESIGN.md).
The paper prints no equations for it; these pins fix what the reading claims: radii -> A in every operator,
Coriolis from the radial component of Omega only, no metric coupling between horizontal and vertical motion,
and the invariants the deep path has (mass, rest state).  Grids come from the oracle's own generator."""
import math

import numpy as np
import pytest

import oracle
import thor_inputs as ti


def _geo(ogrid, level, nv, planet, **kw):
    xyz, nbr, C = ogrid(level, True)
    return oracle.Geometry(xyz, nbr, nv, planet, C, **kw), xyz


def test_operators_use_the_planetary_radius_at_every_layer(ogrid):
    """RS1 (i): div, grad and the Laplacian are the unit-sphere operators over A (A^2), the same in every layer; the
    deep operators over r_k differ by the factor r_k/A.  D_c loses its r^2 factors: D_c[X] = (X_k+1 - X_k)/dz."""
    planet = dict(ti.EARTH, z_top=600.0e3)                   # a deep shell, so that r_k/A is far from 1 (up to 1.09)
    nv = 5
    Gs, xyz = _geo(ogrid, 2, nv, planet, shallow=True)
    Gd, _ = _geo(ogrid, 2, nv, planet)
    rng = np.random.default_rng(3)
    s = np.tile(rng.standard_normal((Gs.N, 1)), (1, nv))      # the same horizontal pattern in every layer
    v = np.tile(rng.standard_normal((Gs.N, 1, 3)), (1, nv, 1))
    A = planet["radius"]
    for op, arg, power in ((Gs.hdiv, v, 1), (Gs.hgrad, s, 1), (Gs.hlap, s, 2)):
        out = op(arg)
        deep = getattr(Gd, op.__name__)(arg)
        for k in range(nv):
            assert np.array_equal(out[:, k], out[:, 0])       # layer-independent, bit for bit
            ratio = (Gd.r_c[k] / A) ** power
            assert np.abs(out[:, k] - deep[:, k] * ratio).max() <= 1e-13 * np.abs(out[:, k]).max()
    X = rng.standard_normal(nv + 1)
    _, _, _, Dc = Gs.vertical_ops(np.zeros(nv), X, order_k=False)
    assert np.abs(Dc - np.diff(X) / (planet["z_top"] / nv)).max() <= 1e-15 * np.abs(Dc).max()


def test_coriolis_is_f_r_cross_v_and_does_no_work(ogrid):
    """RS1 (ii): slowV of a state with uniform p, no gravity and a flow too slow to advect is -f r x V with
    f = 2 Omega sin(lat); it is tangent, perpendicular to V, and W neither feels nor causes a Coriolis force."""
    planet = dict(ti.EARTH, gravity=0.0)
    nv = 4
    G, xyz = _geo(ogrid, 3, nv, planet, shallow=True)
    rng = np.random.default_rng(5)
    rho = np.full((G.N, nv), 1.1)
    p = np.full((G.N, nv), 9.0e4)
    u = 1e-3 * rng.standard_normal((G.N, nv, 3))              # Rossby number ~ 1e-6: advection is negligible
    u -= np.sum(u * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    V = rho[..., None] * u
    W = np.zeros((G.N, nv + 1))
    W[:, 1:nv] = 1e-6 * rng.standard_normal((G.N, nv - 1))     # and too weak a W to advect them vertically
    st = G.slow_terms(rho, V, W, p)
    f = 2.0 * planet["omega"] * xyz[:, 2]
    expect = -f[:, None, None] * np.cross(xyz[:, None, :], V)
    scale = np.abs(expect).max()
    assert np.abs(st["slowV"] - expect).max() < 1e-4 * scale                      # what is left is the advection
    assert np.abs(np.sum(expect * V, axis=-1)).max() <= 1e-15 * scale * np.abs(V).max()
    # W sees no Coriolis force: S_vr is the same with and without rotation (deep: the 2 Omega cos(lat) u term differs)
    G0, _ = _geo(ogrid, 3, nv, dict(planet, omega=0.0), shallow=True)
    st0 = G0.slow_terms(rho, V, W, p)
    assert np.array_equal(st["Svr"], st0["Svr"])
    # and W causes none: slowV does not change with W beyond its advection (second order in the amplitudes)
    stW = G.slow_terms(rho, V, 0.0 * W, p)
    assert np.abs(stW["slowV"] - st["slowV"]).max() < 1e-4 * scale
    Gd, _ = _geo(ogrid, 3, nv, planet)                        # the deep equations do have a vertical Coriolis force
    Gd0, _ = _geo(ogrid, 3, nv, dict(planet, omega=0.0))
    assert np.abs(Gd.slow_terms(rho, V, W, p)["Svr"] - Gd0.slow_terms(rho, V, W, p)["Svr"]).max() > 0.0


def test_solid_body_rotation_keeps_the_horizontal_curvature_term_and_drops_the_radial_one(ogrid):
    """RS1 (iii): for u = w x (A r) the horizontal momentum advection is the tangential part of the centripetal vector
    -rho w^2 s s_hat with s on the sphere of radius A (the u^2 tan(lat)/A metric term), second order in the grid; the
    vertical equation gets NO -rho |v_h|^2/r term: S_vr = 0 where the deep equations have it."""
    planet = dict(ti.EARTH, omega=0.0, gravity=0.0)
    wrot, nv = 2e-5, 4
    errs = []
    for lvl in (2, 3):
        G, xyz = _geo(ogrid, lvl, nv, planet, shallow=True)
        rho = np.tile(1.2 * np.exp(-G.z_c / 8000.0), (G.N, 1))
        p = np.full((G.N, nv), 1e5)
        r = planet["radius"] * np.tile(xyz[:, None, :], (1, nv, 1))
        u = wrot * np.stack([-r[..., 1], r[..., 0], np.zeros_like(r[..., 0])], axis=-1)
        V = rho[..., None] * u
        W = np.zeros((G.N, nv + 1))
        st = G.slow_terms(rho, V, W, p)
        A_exact = -rho[..., None] * wrot ** 2 * np.stack([r[..., 0], r[..., 1], np.zeros_like(r[..., 0])], axis=-1)
        Ah = A_exact - np.sum(A_exact * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
        scale = np.abs(A_exact).max()
        wgt = (G.Ac / G.Ac.sum())[:, None]
        d_h = np.linalg.norm(-st["slowV"] - Ah, axis=-1) / scale
        errs.append(math.sqrt(np.sum(wgt * d_h ** 2)))
        assert np.abs(st["Svr"]).max() == 0.0                  # W = 0, p uniform, g = 0, no metric term: exactly nothing
        Gd, _ = _geo(ogrid, lvl, nv, planet)
        assert np.abs(Gd.slow_terms(rho, V, W, p)["Svr"][:, 1:nv]).max() > 0.3 * scale   # the deep path has it
    assert errs[1] < 0.35 * errs[0] and errs[1] < 0.005


def test_vertical_velocity_is_advected_as_a_scalar(ogrid):
    """RS1 (iii): with a horizontally uniform w = W/rho_h carried by a non-divergent horizontal flow, the scalar advection
    div_h(V w) + D_c[W I_h[w]] reduces to w div_h(V) + (vertical part); for W uniform in the horizontal and V = 0 it is
    the closed form D_c[W I_h[I_c[W]/rho]] interpolated to the interfaces, and the horizontal momentum feels nothing."""
    planet = dict(ti.EARTH, omega=0.0, gravity=0.0)
    nv = 6
    G, xyz = _geo(ogrid, 2, nv, planet, shallow=True)
    dz = planet["z_top"] / nv
    rho = np.full((G.N, nv), 0.9)
    p = np.full((G.N, nv), 5.0e4)
    Wcol = np.zeros(nv + 1)
    Wcol[1:nv] = np.array([0.3, -0.2, 0.5, 0.1, -0.4])
    W = np.tile(Wcol, (G.N, 1))
    V = np.zeros((G.N, nv, 3))
    st = G.slow_terms(rho, V, W, p)
    wc = 0.5 * (Wcol[:-1] + Wcol[1:]) / 0.9                     # I_c[W]/rho
    X = np.zeros(nv + 1)
    X[1:nv] = Wcol[1:nv] * 0.5 * (wc[:-1] + wc[1:])             # W I_h[w]
    Aw = np.diff(X) / dz                                        # D_c without r^2 factors
    expect = -0.5 * (Aw[:-1] + Aw[1:])                          # S_vr = -I_h[F_r], p uniform, g = 0
    assert np.abs(st["Svr"][:, 1:nv] - expect[None, :]).max() <= 1e-14 * np.abs(expect).max()
    assert np.abs(st["slowV"]).max() == 0.0                     # no rho v_h v_r / r coupling, and V = 0


@pytest.mark.parametrize("forced", [False, True])
def test_rest_state_and_mass_in_the_shallow_atmosphere(ogrid, forced):
    """The invariants of the deep path hold: the discretely hydrostatic isothermal column stays at rest, total mass
    (now sum rho A_c A^2 dz) is conserved to round-off by a perturbed run with and without NEXT-1."""
    planet = ti.EARTH
    nv, n, dt = 8, 4, 900.0
    G, xyz = _geo(ogrid, 2, nv, planet, shallow=True)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1e5, 300.0)
    out = G.step(rho, V, W, p, 3, dt, n)
    assert np.abs(out[1]).max() < 1e-9 and np.abs(out[2]).max() < 1e-9
    assert np.abs(out[0] - rho).max() < 1e-12 * rho.max()
    m_exact = float(np.sum(rho * G.Ac[:, None])) * planet["radius"] ** 2 * (planet["z_top"] / nv)
    m0, _ = G.diagnostics(rho, V, W, p)
    assert abs(m0 - m_exact) <= 1e-13 * m_exact                 # volume element A_c A^2 dz
    x, y, z = xyz[:, 0:1], xyz[:, 1:2], xyz[:, 2:3]
    rho2 = p / (planet["Rd"] * 300.0 * (1 + 0.01 * x * z + 0.005 * y))
    vel = 10.0 * np.cross(np.array([0.3, 0.2, 1.0]), xyz)[:, None, :] * np.ones((1, nv, 1))
    D = 0.004837 if forced else 0.0
    s0 = (rho2, rho2[..., None] * vel, W, p)
    m0, _ = G.diagnostics(*s0)
    run = G.step(*s0, 10, dt, n, None, D, D)
    m1, _ = G.diagnostics(*run)
    assert np.all(np.isfinite(run[3]))
    assert abs(m1 - m0) <= 1e-13 * m0
    # and the approximation is an approximation: the deep run differs from it at the order z_top / A
    Gd, _ = _geo(ogrid, 2, nv, planet)
    deep = Gd.step(*s0, 10, dt, n, None, D, D)
    diff = np.abs(deep[3] - run[3]).max() / np.abs(run[3] - s0[3]).max()
    assert 1e-4 < diff < 0.2
