"""Pins P10-P15 of the oracle's time step plus closed-form checks of the slow
terms.  Grids come from the oracle's own generator; nothing comes from the CUDA path."""
import math

import numpy as np
import pytest

import oracle
import thor_inputs as ti


def _geom(ogrid, level, nv, planet):
    xyz, nbr, C = ogrid(level, True)
    return oracle.Geometry(xyz, nbr, nv, planet, C)


# ------------------------------------------------------------------------------------------ P10
def test_p10_thomas_matches_dense_lu():
    rng = np.random.default_rng(10)
    for n in (1, 2, 5, 7):
        a, b, c, d = (rng.standard_normal(n + 1) for _ in range(4))
        b = b + 4.0 * np.sign(b)                                   # diagonally dominant
        x = oracle.thomas(a, b, c, d)
        A = np.zeros((n, n))
        for k in range(1, n + 1):
            A[k - 1, k - 1] = b[k]
            if k > 1:
                A[k - 1, k - 2] = a[k]
            if k < n:
                A[k - 1, k] = c[k]
        ref = np.linalg.solve(A, d[1:])
        assert np.abs(x[1:] - ref).max() < 1e-13 * max(1.0, np.abs(ref).max())


def _dense_column_solve(G, delta, col, stage, dev, divV, divhV):
    """Solve the THREE discrete fast equations of one column as one dense linear system in the
    unknowns (W'_1..nv-1, rho*'_0..nv-1, p'_lin_0..nv-1), written out directly from Eq. 32, the
    linearised pressure equation and Eq. 34 (no elimination)."""
    nv = G.nv
    P = G.planet
    kv = P["Rd"] / (P["Cp"] - P["Rd"])
    g = P["gravity"]
    rc, rh = G.r_c, G.r_h
    # layer thickness t_j, centre spacing s_k and the linear (Eq. 8-9, k = 1) weights of interface k between the
    # centres k-1 and k; equal layers: t = s = dz, weights 1/2
    t = np.diff(G.z_h)
    sp = np.concatenate([[1.0], np.diff(G.z_c)])
    wl = np.concatenate([[0.0], (G.z_c[1:] - G.z_h[1:nv]) / np.diff(G.z_c)])
    wu = np.concatenate([[0.0], (G.z_h[1:nv] - G.z_c[:-1]) / np.diff(G.z_c)])
    h, gt = stage["h"][col], stage["gt"][col]
    hh = np.zeros(nv + 1)
    hh[1:nv] = wl[1:] * h[:-1] + wu[1:] * h[1:]
    nW = nv - 1
    n = nW + 2 * nv
    A = np.zeros((n, n))
    b = np.zeros(n)
    iW = lambda k: k - 1            # interface k = 1..nv-1
    iR = lambda j: nW + j
    iP = lambda j: nW + nv + j
    S_rho = stage["slowrho"][col] - divV[col]
    S_p = stage["slowp"][col] - kv * divhV[col]
    for j in range(nv):
        # Eq. 32: rho' + delta * D_c[W'] = rho* + delta S_rho
        A[iR(j), iR(j)] = 1.0
        if j + 1 <= nv - 1:
            A[iR(j), iW(j + 1)] += delta * rh[j + 1] ** 2 / (rc[j] ** 2 * t[j])
        if j >= 1:
            A[iR(j), iW(j)] -= delta * rh[j] ** 2 / (rc[j] ** 2 * t[j])
        b[iR(j)] = dev["rho_s"][col, j] + delta * S_rho[j]
        # pressure: p' + delta kv (D_c[h_h W'] - I_c[g~ W']) = p* + delta S_p
        A[iP(j), iP(j)] = 1.0
        if j + 1 <= nv - 1:
            A[iP(j), iW(j + 1)] += delta * kv * (rh[j + 1] ** 2 * hh[j + 1] / (rc[j] ** 2 * t[j]) - 0.5 * gt[j + 1])
        if j >= 1:
            A[iP(j), iW(j)] += delta * kv * (-rh[j] ** 2 * hh[j] / (rc[j] ** 2 * t[j]) - 0.5 * gt[j])
        b[iP(j)] = dev["p_s"][col, j] + delta * S_p[j]
    for k in range(1, nv):
        # Eq. 34: (W' - W*)/delta + G_h[p'] + g I_h[rho'] = S_vr
        A[iW(k), iW(k)] = 1.0 / delta
        A[iW(k), iP(k)] += 1.0 / sp[k]
        A[iW(k), iP(k - 1)] -= 1.0 / sp[k]
        A[iW(k), iR(k)] += wu[k] * g
        A[iW(k), iR(k - 1)] += wl[k] * g
        b[iW(k)] = stage["Svr"][col, k] + dev["W_s"][col, k] / delta
    x = np.linalg.solve(A, b)
    return x[:nW], x[nW:nW + nv], x[nW + nv:]


def test_p10_substep_matches_dense_solve_of_the_three_fast_equations(ogrid):
    cfg = ti.CONFIGS[0]
    xyz, nbr, C = ogrid(2, True)
    nv = 6
    G = oracle.Geometry(xyz, nbr, nv, cfg["planet"], C)
    rng = np.random.default_rng(11)
    rho, V, W, p = ti.rest_state(cfg["planet"], nv, G.N, 1e5, 300.0)
    T = 300.0 * (1 + rng.uniform(-2e-2, 2e-2, size=rho.shape))
    rho = p / (287.0 * T)
    vel = rng.uniform(-5, 5, size=V.shape)
    vel -= np.sum(vel * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    V = rho[..., None] * vel
    W[:, 1:nv] = rng.uniform(-0.5, 0.5, size=(G.N, nv - 1))
    st = G.slow_terms(rho, V, W, p)
    stage = dict(st, p_t=p)
    dev = dict(rho_s=rng.uniform(-1e-3, 1e-3, size=rho.shape), V_s=rng.uniform(-1, 1, size=V.shape),
               W_s=np.zeros_like(W), p_s=rng.uniform(-50, 50, size=p.shape),
               rt=p / 287.0 * (1e5 / p) ** (287.0 / 1005.0) * 0 + (1e5 / 287.0) * (p / 1e5) ** (1 - 287.0 / 1005.0))
    dev["V_s"] -= np.sum(dev["V_s"] * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    dev["W_s"][:, 1:nv] = rng.uniform(-0.1, 0.1, size=(G.N, nv - 1))
    delta = 300.0
    new = G.substep(delta, stage, dev)
    # Eq. 33 by hand from the (separately pinned) gradient operator
    Vexp = dev["V_s"] + delta * (-G.hgrad(dev["p_s"]) + st["slowV"])
    assert np.abs(new["V_s"] - Vexp).max() < 1e-12 * np.abs(Vexp).max()
    divV = G.hdiv(new["V_s"])
    divhV = G.hdiv(st["h"][..., None] * new["V_s"])
    divtV = G.hdiv(st["th"][..., None] * new["V_s"])
    for col in (0, 3, 77, G.N - 1):
        Wd, rd, pl = _dense_column_solve(G, delta, col, stage, dev, divV, divhV)
        assert np.abs(new["W_s"][col, 1:nv] - Wd).max() < 1e-11 * np.abs(Wd).max()
        assert np.abs(new["rho_s"][col] - rd).max() < 1e-11 * np.abs(rd).max()
        assert new["W_s"][col, 0] == 0.0 and new["W_s"][col, nv] == 0.0          # rigid lid, L339
        # Eq. 35 (G7) and Eq. 36 from the dense W'
        Wn = np.concatenate([[0.0], Wd, [0.0]])
        thh = np.zeros(nv + 1)
        thh[1:nv] = 0.5 * (st["th"][col, :-1] + st["th"][col, 1:])
        X = thh * Wn
        Dc = (G.r_h[1:] ** 2 * X[1:] - G.r_h[:-1] ** 2 * X[:-1]) / (G.r_c ** 2 * G.dz)
        rt_exp = dev["rt"][col] + delta * (st["slowrt"][col] - divtV[col] - Dc)
        assert np.abs(new["rt"][col] - rt_exp).max() < 1e-12 * np.abs(rt_exp).max()
        gam = 1005.0 / (1005.0 - 287.0)
        p_exp = 1e5 * (287.0 * rt_exp / 1e5) ** gam - p[col]
        assert np.abs(new["p_s"][col] - p_exp).max() < 1e-9
    # tridiagonal is diagonally dominant enough for Thomas without pivoting
    a, b, c = G.tridiag_coefficients(delta, st["h"][5], st["gt"][5])
    assert np.all(np.abs(b[1:nv]) > 0.9 * (np.abs(a[1:nv]) + np.abs(c[1:nv])))


# ------------------------------------------------------------------------------------- P11, P12
def test_p12_resting_isothermal_atmosphere_stays_at_rest(ogrid):
    cfg = ti.CONFIGS[0]
    G = _geom(ogrid, 3, cfg["nv"], cfg["planet"])
    rho, V, W, p = ti.rest_state(cfg["planet"], cfg["nv"], G.N, cfg["p_s"], cfg["T0"])
    r2, V2, W2, p2 = G.step(rho, V, W, p, 10, cfg["dt"], cfg["n_sub"])
    w = W2[:, 1:-1] / (0.5 * (r2[:, 1:] + r2[:, :-1]))
    assert np.abs(w).max() < 1e-9                                     # m/s
    assert np.abs(V2 / r2[..., None]).max() < 1e-9
    assert np.abs(r2 - rho).max() < 1e-13 * rho.max()
    assert np.abs(p2 - p).max() < 1e-13 * p.max()
    # an analytically exponential profile is NOT at rest discretely (O(dz^2) residual): sanity
    z = G.z_c
    p_exp = np.tile(1e5 * np.exp(-9.8 * z / (287.0 * 300.0)), (G.N, 1))
    r3, V3, W3, p3 = G.step(p_exp / (287.0 * 300.0), V, W, p_exp, 1, cfg["dt"], cfg["n_sub"])
    assert np.abs(W3).max() > 1e-6


@pytest.mark.parametrize("forced", [False, True])
def test_p11_total_mass_is_conserved_to_roundoff(ogrid, forced):
    cfg = ti.CONFIGS[0]
    xyz, nbr, C = ogrid(3, True)
    G = oracle.Geometry(xyz, nbr, cfg["nv"], cfg["planet"], C)
    state = ti.initial_state(0, xyz)
    forcing = None
    if forced:
        rng = np.random.default_rng(5)
        forcing = dict(T_eq=300 + rng.uniform(-20, 20, size=state[0].shape),
                       k_T=np.full(state[0].shape, 1e-5), k_v=np.full(state[0].shape, 2e-5))
    m0, e0 = G.diagnostics(*state)
    new = G.step(*state, 5, cfg["dt"], cfg["n_sub"], forcing)
    m1, e1 = G.diagnostics(*new)
    assert abs(m1 - m0) < 1e-14 * m0
    # closed form of the initial mass: sum over layers of rho * shell weight; rho is known
    assert abs(m0 - np.sum(state[0] * G.Ac[:, None] * (G.r_c ** 2 * G.dz)[None, :])) < 1e-12 * m0
    if not forced:                                                    # P15 (soft)
        assert abs(e1 - e0) < 1e-6 * abs(e0)


# ------------------------------------------------------------------------- slow-term closed forms
def test_p13_coriolis_closed_form_and_no_work(ogrid):
    cfg = ti.CONFIGS[0]
    xyz, nbr, C = ogrid(3, True)
    nv = 4
    rot = dict(cfg["planet"])
    norot = dict(cfg["planet"], omega=0.0)
    G1, G0 = oracle.Geometry(xyz, nbr, nv, rot, C), oracle.Geometry(xyz, nbr, nv, norot, C)
    rng = np.random.default_rng(13)
    rho, V, W, p = ti.rest_state(rot, nv, G1.N, 1e5, 300.0)
    vel = rng.uniform(-10, 10, size=V.shape)
    vel -= np.sum(vel * xyz[:, None, :], axis=-1, keepdims=True) * xyz[:, None, :]
    V = rho[..., None] * vel
    s1, s0 = G1.slow_terms(rho, V, W, p), G0.slow_terms(rho, V, W, p)
    Ch = -(s1["slowV"] - s0["slowV"])                      # horizontal Coriolis term C_h
    f = 2 * rot["omega"] * xyz[:, 2]                       # 2 Omega sin(lat)
    expect = f[:, None, None] * np.cross(np.broadcast_to(xyz[:, None, :], V.shape), V)
    assert np.abs(Ch - expect).max() < 1e-12 * np.abs(expect).max()
    assert np.abs(np.sum(Ch * V, axis=-1)).max() < 1e-12 * np.abs(expect).max() * np.abs(V).max()
    # radial part: C_r = 2 Omega (z x V).r, averaged to interfaces, enters S_vr with a minus sign
    Cr = 2 * rot["omega"] * (-V[..., 1] * xyz[:, None, 0] + V[..., 0] * xyz[:, None, 1])
    dS = -(s1["Svr"] - s0["Svr"])[:, 1:nv]
    assert np.abs(dS - 0.5 * (Cr[:, :-1] + Cr[:, 1:])).max() < 1e-12 * np.abs(Cr).max()


def test_advection_of_solid_body_rotation_is_centripetal(ogrid):
    """For u = w x r with rho = rho(r): div(rho u u) = rho w x (w x r) exactly, i.e.
    A = -rho w^2 s s_hat (s = distance from the axis).  The discrete A (reading R7) must converge
    to it at second order; its horizontal part shows up in slowV, its radial part in S_vr."""
    cfg = ti.CONFIGS[0]
    planet = dict(cfg["planet"], omega=0.0, gravity=0.0)
    errs = []
    wrot = 2e-5
    for lvl in (2, 3):
        xyz, nbr, C = ogrid(lvl, True)
        nv = 4
        G = oracle.Geometry(xyz, nbr, nv, planet, C)
        rho = np.tile(1.2 * np.exp(-G.z_c / 8000.0), (G.N, 1))
        p = np.full((G.N, nv), 1e5)                        # uniform p, g = 0: no other force
        r = G.r_c[None, :, None] * xyz[:, None, :]
        u = wrot * np.stack([-r[..., 1], r[..., 0], np.zeros_like(r[..., 0])], axis=-1)
        V = rho[..., None] * u
        W = np.zeros((G.N, nv + 1))
        st = G.slow_terms(rho, V, W, p)
        A_exact = -rho[..., None] * wrot ** 2 * np.stack([r[..., 0], r[..., 1], np.zeros_like(r[..., 0])], axis=-1)
        Ar = np.sum(A_exact * xyz[:, None, :], axis=-1)
        Ah = A_exact - Ar[..., None] * xyz[:, None, :]
        scale = np.abs(A_exact).max()
        wgt = (G.Ac / G.Ac.sum())[:, None]
        d_h = np.linalg.norm(-st["slowV"] - Ah, axis=-1) / scale
        d_r = np.abs(-st["Svr"][:, 1:nv] - 0.5 * (Ar[:, :-1] + Ar[:, 1:])) / scale
        errs.append((math.sqrt(np.sum(wgt * d_h ** 2)), math.sqrt(np.sum(wgt * d_r ** 2)), d_h.max(), d_r.max()))
        # mass tendency of a divergence-free flow: second-order small
        assert np.abs(st["slowrho"]).max() < 0.05 * np.abs(rho * wrot).max()
    # l2 (Eq. 17) second order; l_inf slower (hexagons next to the pentagons), as in L154
    assert errs[1][0] < 0.35 * errs[0][0] and errs[1][0] < 0.005
    assert errs[1][1] < 0.35 * errs[0][1] and errs[1][1] < 0.005
    assert errs[1][2] < 0.7 * errs[0][2] and errs[1][3] < 0.7 * errs[0][3]


def test_pressure_and_entropy_tendencies_are_consistent(ogrid):
    """dp/dt = (gamma p / (rho theta)) d(rho theta)/dt (Eq. 24): the slow part of the pressure
    equation (Eq. 40 with the signs of G10) and of Eq. 35 discretise the same quantity; their
    mismatch is a truncation error that shrinks with resolution, for a smooth state."""
    cfg = ti.CONFIGS[0]
    planet = dict(cfg["planet"])
    gam = planet["Cp"] / (planet["Cp"] - planet["Rd"])
    mism = []
    for lvl, nv in ((2, 8), (3, 16)):
        xyz, nbr, C = ogrid(lvl, True)
        G = oracle.Geometry(xyz, nbr, nv, planet, C)
        x, y, z = xyz[:, 0:1], xyz[:, 1:2], xyz[:, 2:3]
        zc = G.z_c[None, :]
        T = 280.0 + 15.0 * x * y + 10.0 * z - 3e-4 * zc
        p = 1e5 * np.exp(-zc / 8000.0) * (1 + 0.01 * (x - 0.5 * z * y))
        rho = p / (planet["Rd"] * T)
        hr = ti.heikes_randall_fields(xyz, 1, 1)
        vel = 20.0 * hr["v"][:, None, :] * (1 + zc[..., None] / 36e3)
        V = rho[..., None] * vel
        W = np.zeros((G.N, nv + 1))
        W[:, 1:nv] = 0.02 * (0.5 * (rho[:, 1:] + rho[:, :-1])) * (x + z) * np.sin(np.pi * G.r_h[None, 1:nv] / 1.0 % 1.0 * 0 + np.pi * np.arange(1, nv)[None, :] / nv)
        st = G.slow_terms(rho, V, W, p)
        rt = planet["p_ref"] / planet["Rd"] * (p / planet["p_ref"]) ** (1 / gam)
        lhs = st["slowp"]
        rhs = gam * p / rt * st["slowrt"]
        mism.append(np.abs(lhs - rhs)[:, 1:-1].max() / np.abs(rhs).max())
    assert mism[1] < 0.5 * mism[0] and mism[1] < 0.05, mism


def test_vertical_slow_term_is_second_order_hydrostatic_residual(ogrid):
    """S_vr of an analytic hydrostatic isothermal column is an O(dz^2) residual (Eq. 42)."""
    cfg = ti.CONFIGS[0]
    planet = dict(cfg["planet"], omega=0.0)
    xyz, nbr, C = ogrid(1, True)
    res = []
    for nv in (16, 32):
        G = oracle.Geometry(xyz, nbr, nv, planet, C)
        H = 287.0 * 300.0 / 9.8
        p = np.tile(1e5 * np.exp(-G.z_c / H), (G.N, 1))
        rho = p / (287.0 * 300.0)
        st = G.slow_terms(rho, np.zeros((G.N, nv, 3)), np.zeros((G.N, nv + 1)), p)
        res.append(np.abs(st["Svr"][:, 1:nv]).max())
        assert np.all(st["slowV"] == 0.0)
    assert 3.5 < res[0] / res[1] < 4.5


# ------------------------------------------------------------------------------------------ P14
def test_p14_rk3_stage_weights_give_third_order_on_rotation_dominated_flow(ogrid):
    """Pin of reading R1 (stage reference state, the 1/3, 1/2, 1 weights and the restart from t_n of
    Eq. 30-31).  Three step sizes against a much finer reference, observed order asserted
    for V and for p separately.

    The HE-VI coupling of the fast modes (forward-backward in the horizontal, backward Euler in the
    vertical, Eq. 33-37) is first order in the substep delta BY CONSTRUCTION; a flow dominated by
    acoustic/gravity-wave adjustment therefore shows order ~1 at fixed n whatever the stage weights
    are (measured: 1.04-1.10 on a warm anomaly at rest), which is why this pin uses a flow whose
    evolution is carried by the SLOW terms: solid-body rotation about a tilted axis on a fast
    rotator (Omega = 3e-4 1/s, inertial period ~3 h, Coriolis and advection in slowV), many substeps
    (n = 32) so that the first-order fast-mode error is far below the Runge-Kutta error.  Eq. 30 is
    then a three-stage Runge-Kutta scheme on a nearly linear slow operator: third order.  A wrong
    second-stage weight or restart gives order 1, a wrong first-stage weight order 2 (both outside
    the asserted windows); L243 claims second order at least."""
    xyz, nbr, C = ogrid(2, True)
    nv, n, Ttot = 6, 32, 7200.0
    planet = dict(ti.EARTH, omega=3.0e-4)
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1e5, 300.0)
    vel = 10.0 * np.cross(np.array([0.3, 0.2, 1.0]), xyz)[:, None, :] * np.ones((1, nv, 1))
    V = rho[..., None] * vel
    ref = G.step(rho, V, W, p, 64, Ttot / 64, n)
    eV, ep = [], []
    for k in (2, 4, 8):
        out = G.step(rho, V, W, p, k, Ttot / k, n)
        eV.append(np.abs(out[1] - ref[1]).max())
        ep.append(np.abs(out[3] - ref[3]).max())
    assert eV[0] > 0.1 * np.abs(ref[1] - V).max()                # the coarse run is far from converged: a real test
    oV = [math.log2(eV[i] / eV[i + 1]) for i in range(2)]
    op = [math.log2(ep[i] / ep[i + 1]) for i in range(2)]
    assert all(2.6 < o < 3.3 for o in oV), (oV, eV)
    assert all(2.0 < o < 3.0 for o in op), (op, ep)


def test_p14b_fast_mode_coupling_is_first_order_in_the_substep(ogrid):
    """The complement of P14, stated so that nobody reads L243's "second-order accuracy" into the whole
    scheme: on an adjustment problem (warm anomaly at rest, Earth rotation, n = 4) the error falls
    ~2x per halving of dt -- the backward-Euler vertical solve and the forward-backward horizontal
    coupling of Eq. 33-37 are first order in delta = dt/n."""
    xyz, nbr, C = ogrid(2, True)
    nv, n, Ttot = 6, 4, 3600.0
    planet = ti.EARTH
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1e5, 300.0)
    x, y, z = xyz[:, 0:1], xyz[:, 1:2], xyz[:, 2:3]
    rho = p / (287.0 * 300.0 * (1 + 0.01 * x * z + 0.005 * y))
    ref = G.step(rho, V, W, p, 64, Ttot / 64, n)
    e = [np.abs(G.step(rho, V, W, p, k, Ttot / k, n)[1] - ref[1]).max() for k in (2, 4, 8)]
    o = [math.log2(e[i] / e[i + 1]) for i in range(2)]
    assert all(0.8 < x < 1.4 for x in o), (o, e)


# ------------------------------------------------------------------------------------------ R10
def test_total_energy_closed_forms(ogrid):
    """Pin of the energy half of orc_diagnostics (R10: E = sum (Cv p/Rd + (|V|^2 + I_c[W]^2)/(2 rho)
    + rho g z_c) A_c r_c^2 dz; L215, L339 only name "total energy").  Four states whose energy is a
    one-line closed form, each isolating one term, so that Cp for Cv, a missing 1/2, z_h for z_c,
    r_h for r_c or a wrong I_c fails one of them.  The expected values are written out here with
    math.fsum from the layer tables; sum(A_c) = 4 pi is pin P2."""
    xyz, nbr, C = ogrid(2, True)
    nv = 5
    planet = dict(ti.EARTH, z_top=20.0e3)
    Rd, Cp, g, A = planet["Rd"], planet["Cp"], planet["gravity"], planet["radius"]
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    N = G.N
    dz = planet["z_top"] / nv
    zc = [(k + 0.5) * dz for k in range(nv)]
    rc = [A + zk for zk in zc]
    area = math.fsum(G.Ac)
    assert abs(area - 4 * math.pi) < 1e-12
    pk = ti.hydrostatic_isothermal(planet, nv, 1.0e5, 250.0)           # the P12 recurrence
    rk = [float(x) / (Rd * 250.0) for x in pk]
    rho, p = np.tile(np.array(rk), (N, 1)), np.tile(pk, (N, 1))
    V0, W0 = np.zeros((N, nv, 3)), np.zeros((N, nv + 1))
    # (a) internal + potential energy of the discretely hydrostatic isothermal rest column
    E_int = area * math.fsum((Cp - Rd) * float(pk[k]) / Rd * rc[k] ** 2 * dz for k in range(nv))
    E_pot = area * math.fsum(rk[k] * g * zc[k] * rc[k] ** 2 * dz for k in range(nv))
    _, E = G.diagnostics(rho, V0, W0, p)
    assert abs(E - (E_int + E_pot)) <= 1e-13 * (E_int + E_pot)
    # (b) no gravity: the internal term alone (Cv, not Cp: they differ by 40 %)
    G0 = oracle.Geometry(xyz, nbr, nv, dict(planet, gravity=0.0), C)
    _, E = G0.diagnostics(rho, V0, W0, p)
    assert abs(E - E_int) <= 1e-13 * E_int
    assert abs(E_pot) > 0.05 * E_int                                    # (a) did test the potential term
    # (c) horizontal kinetic energy of solid-body rotation in ONE layer: 1/2 rho |w x r|^2, |w x r|^2 = w^2 r^2 (1 - z^2)
    k0, wrot = 3, 2.0e-6
    V = V0.copy()
    V[:, k0, :] = rk[k0] * wrot * rc[k0] * np.cross(np.array([0.0, 0.0, 1.0]), xyz)
    S = math.fsum(float(a) * (1.0 - float(zz) ** 2) for a, zz in zip(G.Ac, xyz[:, 2]))
    E_kh = 0.5 * rk[k0] * (wrot * rc[k0]) ** 2 * S * rc[k0] ** 2 * dz
    _, E = G0.diagnostics(rho, V, W0, p)
    assert abs((E - E_int) - E_kh) <= 1e-9 * E_kh                      # E_kh ~ 1e-6 E_int: 1e-9 of it is the rounding of the sum
    # (d) vertical kinetic energy of W on ONE interface k1: I_c[W] = W/2 in the layers below and above it
    k1, Wv = 2, 0.7
    W = W0.copy()
    W[:, k1] = Wv
    E_kv = area * 0.5 * (0.5 * Wv) ** 2 * (rc[k1 - 1] ** 2 / rk[k1 - 1] + rc[k1] ** 2 / rk[k1]) * dz
    _, E = G0.diagnostics(rho, V0, W, p)
    assert abs((E - E_int) - E_kv) <= 1e-8 * E_kv


# ------------------------------------------------------------------------------------- energy fixer RE1
def test_energy_fixer_restores_total_energy_by_one_uniform_temperature_increment(ogrid):
    """NEXT-4, reading RE1 (L215, "globally uniform adjusts the internal energy at all grid points"): with the fixer
    on, an unforced run keeps the total energy of R10 (pinned by test_total_energy_closed_forms) to round-off while
    the same run without it drifts by orders of magnitude more; the adjustment of one step is ONE temperature
    increment dT = (E - E')/(Cv M) for every cell, density untouched; off is the base path bit for bit."""
    xyz, nbr, C = ogrid(2, True)
    nv, n, dt = 6, 4, 900.0
    planet = ti.EARTH
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1e5, 300.0)
    x, y, z = xyz[:, 0:1], xyz[:, 1:2], xyz[:, 2:3]
    rho = p / (planet["Rd"] * 300.0 * (1 + 0.01 * x * z + 0.005 * y))
    vel = 15.0 * np.cross(np.array([0.3, 0.2, 1.0]), xyz)[:, None, :] * np.ones((1, nv, 1))
    s0 = (rho, rho[..., None] * vel, W, p)
    m0, e0 = G.diagnostics(*s0)
    plain = G.step(*s0, 1, dt, n)
    fixed = G.step(*s0, 1, dt, n, energy_fixer=True)
    m1, e1 = G.diagnostics(*plain)
    mf, ef = G.diagnostics(*fixed)
    assert abs(e1 - e0) > 1e-9 * e0                                   # the dynamics alone do change E: a real test
    assert abs(ef - e0) <= 2e-15 * e0
    assert np.array_equal(fixed[0], plain[0]) and np.array_equal(fixed[1], plain[1]) and np.array_equal(fixed[2], plain[2])
    dT = (fixed[3] - plain[3]) / (plain[0] * planet["Rd"])
    expect = (e0 - e1) / ((planet["Cp"] - planet["Rd"]) * m1)
    assert np.abs(dT - expect).max() <= 1e-6 * abs(expect) + 1e-12     # uniform; p - p' itself is rounded at ulp(p)
    # many steps: E stays, mass stays
    run = G.step(*s0, 20, dt, n, energy_fixer=True)
    mr, er = G.diagnostics(*run)
    m20, e20 = G.diagnostics(*G.step(*s0, 20, dt, n))
    assert abs(er - e0) <= 1e-14 * e0 and abs(mr - m0) <= 1e-13 * m0
    assert abs(e20 - e0) > 100 * abs(er - e0)
    # off = the base path
    again = G.step(*s0, 1, dt, n, energy_fixer=False)
    assert all(np.array_equal(a, b) for a, b in zip(again, plain))


# ------------------------------------------------------------------------------------- forcing R9
def test_forcing_limits(ogrid):
    cfg = ti.CONFIGS[0]
    xyz, nbr, C = ogrid(2, True)
    nv = cfg["nv"]
    G = oracle.Geometry(xyz, nbr, nv, cfg["planet"], C)
    rho, V, W, p = ti.rest_state(cfg["planet"], nv, G.N, 1e5, 300.0)
    shape = rho.shape
    # k = 0: nothing happens; T_eq = T: nothing happens
    for F in (dict(T_eq=np.full(shape, 250.0), k_T=np.zeros(shape), k_v=np.zeros(shape)),
              dict(T_eq=np.full(shape, 300.0), k_T=np.full(shape, 1e-3), k_v=np.full(shape, 1e-3))):
        out = G.step(rho, V, W, p, 1, 600.0, 2, F)
        assert np.abs(out[3] - p).max() < 1e-9 and np.abs(out[0] - rho).max() < 1e-15
    # k -> infinity: T -> T_eq exactly, rho untouched (L200), p = rho Rd T_eq
    Teq = 250.0 + 10 * xyz[:, 2:3] * np.ones(shape)
    out = G.step(rho, V, W, p, 1, 600.0, 2, dict(T_eq=Teq, k_T=np.full(shape, 1e12), k_v=None))
    assert np.abs(out[3] / (out[0] * 287.0) - Teq).max() < 1e-6
    # Rayleigh drag divides the horizontal momentum by (1 + k dt) and leaves W alone (Eq. 51)
    state = ti.initial_state(0, ogrid(2, True)[0])
    a = G.step(*state, 1, 600.0, 2, None)
    b = G.step(*state, 1, 600.0, 2, dict(T_eq=None, k_T=None, k_v=np.full(shape, 1e-3)))
    assert np.abs(b[1] * 1.6 - a[1]).max() < 1e-12 * np.abs(a[1]).max()
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[0], b[0]) and np.array_equal(a[3], b[3])


# --------------------------------------------------------------------------------------------
# NEXT-1: hyper-diffusion and divergence damping (Eq. 43-50; readings RD1-RD5 of DESIGN.md)
# --------------------------------------------------------------------------------------------
def test_diffusion_off_is_the_base_path_bit_for_bit(ogrid):
    cfg = ti.CONFIGS[0]
    G = _geom(ogrid, 2, cfg["nv"], cfg["planet"])
    state = ti.initial_state(0, G.xyz)
    a = G.step(*state, 2, cfg["dt"], cfg["n_sub"])
    b = G.step(*state, 2, cfg["dt"], cfg["n_sub"], None, 0.0, 0.0)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))


def test_diffusion_conserves_mass_and_keeps_the_rest_state(ogrid):
    cfg = ti.CONFIGS[0]
    planet, nv = cfg["planet"], cfg["nv"]
    G = _geom(ogrid, 3, nv, planet)
    D = 0.004837                                     # the paper's Earth value (Table 1 with dt = 1000 s)
    state = ti.initial_state(0, G.xyz)
    m0, _ = G.diagnostics(*state)
    out = G.step(*state, 5, cfg["dt"], cfg["n_sub"], None, D, D)
    m1, _ = G.diagnostics(*out)
    assert abs(m1 - m0) <= 1e-14 * m0                # the Laplacian is in flux form: F_rho integrates to zero
    assert not np.array_equal(out[0], G.step(*state, 5, cfg["dt"], cfg["n_sub"])[0])
    rest = ti.rest_state(planet, nv, G.N, cfg["p_s"], cfg["T0"])
    a = G.step(*rest, 3, cfg["dt"], cfg["n_sub"], None, D, D)
    b = G.step(*rest, 3, cfg["dt"], cfg["n_sub"])
    assert np.abs(a[1]).max() < 1e-9 and np.abs(a[2]).max() < 1e-9      # still at rest (P12)
    assert np.abs(a[0] - b[0]).max() <= 1e-13 * np.abs(b[0]).max()     # horizontally uniform fields: lap = 0


def test_hyper_diffusion_fluxes_closed_forms(ogrid):
    """On a horizontally uniform density: solid-body rotation v = w x r has Cartesian components that
    are degree-1 harmonics, lap v_j = -2 v_j / r^2, so F_vh = -K_d lap(rho lap v) = -4 K_d rho v / r^4
    (tangent already); T = T0 + a Y_l gives F_p = -Rd K_d rho [l(l+1)]^2 a Y_l / r^4, and the same
    pattern on rho gives F_rho.  F_rt follows F_p through Eq. 24."""
    import oracle
    planet, nv = dict(ti.EARTH), 3
    planet["z_top"] = 9000.0
    xyz, nbr, C = ogrid(4, True)
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1.0e5, 280.0)
    Kd = 1.0e16
    om = np.array([0.3, -0.2, 1.0]) * 1e-5
    vel = np.cross(om[None, None, :], xyz[:, None, :] * G.r_c[None, :, None])
    V = rho[..., None] * vel
    Y, _, ell = ti.real_sph_harm(xyz, 3)
    k = int(np.where(ell == 3)[0][2])
    T = 280.0 + 2.0 * Y[:, k][:, None] * np.ones(nv)[None, :]
    p = rho * planet["Rd"] * T
    Frho, FV, FW, Fp, Frt = G.diffusion_fluxes(rho, V, W, p, Kd)
    exact_V = -4.0 * Kd * V / G.r_c[None, :, None] ** 4
    # A biharmonic operator built from two 7-point Laplacians is not pointwise consistent on an irregular
    # grid (the second Laplacian differentiates the first one's O(h^2) error twice): the pins are the median
    # and the 90th percentile away from the twelve pentagons, not the maximum
    far = np.ones(G.N, dtype=bool)
    ring = np.where(G.deg == 5)[0]
    for _ in range(3):
        far[ring] = False
        ring = np.unique(G.nbr[ring][G.nbr[ring] >= 0])
    assert np.median(np.abs(FV - exact_V)) < 0.01 * np.abs(exact_V).max()
    assert np.percentile(np.abs(FV - exact_V)[far], 90) < 0.05 * np.abs(exact_V).max()
    exact_p = -planet["Rd"] * Kd * rho * 144.0 * (T - 280.0) / G.r_c[None, :] ** 4
    assert np.median(np.abs(Fp - exact_p)) < 0.02 * np.abs(exact_p).max()
    assert np.percentile(np.abs(Fp - exact_p)[far], 90) < 0.1 * np.abs(exact_p).max()
    assert np.all(Frho == 0.0) and np.all(FW == 0.0)                   # uniform rho, W = 0
    gam = planet["Cp"] / (planet["Cp"] - planet["Rd"])
    rt = planet["p_ref"] / planet["Rd"] * (p / planet["p_ref"]) ** (1.0 / gam)
    assert np.allclose(Frt, Fp * rt / (gam * p), rtol=1e-12, atol=0)
    # density pattern and vertical velocity pattern: same operator, same eigenvalue
    rho2 = rho * (1.0 + 1e-3 * Y[:, k][:, None])
    W2 = np.zeros_like(W)
    W2[:, 1:nv] = 0.5 * (rho[:, 1:] + rho[:, :-1]) * 0.01 * Y[:, k][:, None]
    Frho2, _, FW2, _, _ = G.diffusion_fluxes(rho2, np.zeros_like(V), W2, rho2 * planet["Rd"] * 280.0, Kd)
    ex_rho = -Kd * 144.0 * (rho2 - rho) / G.r_c[None, :] ** 4
    assert np.median(np.abs(Frho2 - ex_rho)) < 0.02 * np.abs(ex_rho).max()
    ex_W = -Kd * 144.0 * W2[:, 1:nv] / G.r_h[None, 1:nv] ** 4
    assert np.median(np.abs(FW2[:, 1:nv] - ex_W)) < 0.03 * np.abs(ex_W).max()
    assert np.all(FW2[:, 0] == 0.0) and np.all(FW2[:, nv] == 0.0)


def test_divergence_damping_acts_on_divergence_only(ogrid):
    """F_dd = -K_d lap(grad D3): tangent; (nearly) zero for a non-divergent flow; for a divergent flow
    it opposes the divergence pattern (div F_dd anti-correlated with D3)."""
    import oracle
    planet, nv = dict(ti.EARTH), 2
    planet["z_top"] = 6000.0
    xyz, nbr, C = ogrid(4, True)
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1.0e5, 280.0)
    Y, gY, ell = ti.real_sph_harm(xyz, 4)
    a = np.random.default_rng(3).standard_normal(Y.shape[1])
    a[0] = 0.0
    gchi = np.einsum("nkd,k->nd", gY, a)
    Vdiv = rho[..., None] * gchi[:, None, :]
    Vrot = rho[..., None] * np.cross(xyz, gchi)[:, None, :]
    Kd = 1.0e16
    Fd, Fr = G.divergence_damping(Vdiv, W, Kd), G.divergence_damping(Vrot, W, Kd)
    assert np.abs(np.sum(Fd * xyz[:, None, :], axis=-1)).max() <= 1e-12 * np.abs(Fd).max()
    assert np.median(np.linalg.norm(Fr, axis=-1)) < 0.02 * np.median(np.linalg.norm(Fd, axis=-1))   # (spikes at the pentagons only)
    D3 = G.hdiv(Vdiv)
    w = G.Ac[:, None]
    corr = (w * G.hdiv(Fd) * D3).sum() / np.sqrt((w * G.hdiv(Fd) ** 2).sum() * (w * D3 ** 2).sum())
    assert corr < -0.7


# --------------------------------------------------------------------------------------------
# NEXT-2: Held-Suarez forcing from the evolving sigma (Eq. 51-55)
# --------------------------------------------------------------------------------------------
def test_held_suarez_forcing_closed_forms(ogrid):
    """Eq. 53-55 evaluated by hand on an isothermal hydrostatic column: the extrapolated surface pressure
    is the column's p_s exactly (L390), so sigma = p/p_s; drag only below sigma_b = 0.7 (Eq. 53); T_eq =
    315 K at the equator's surface pressure, 255 K at the poles', 200 K aloft (Eq. 54); with a huge
    step the backward-Euler update lands on T_eq and on zero wind (Eq. 51-52)."""
    import oracle
    planet, nv = dict(ti.EARTH), 16
    xyz, nbr, C = ogrid(2, True)
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    ps, T0 = 1.0e5, 280.0
    rho, V, W, p = ti.rest_state(planet, nv, G.N, ps, T0)
    V = rho[..., None] * np.cross(np.array([0.0, 0.0, 1.0e-6])[None, None, :], xyz[:, None, :] * G.r_c[None, :, None])
    hs = dict(ti.HELD_SUAREZ)
    sigma = p / ps
    lat_s = xyz[:, 2][:, None]
    c2 = 1.0 - lat_s ** 2
    kappa = planet["Rd"] / planet["Cp"]
    Teq = np.maximum(200.0, (315.0 - 60.0 * lat_s ** 2 - hs["dth_z"] * np.log(p / 1e5) * c2) * (p / 1e5) ** kappa)
    ramp = np.maximum(0.0, (sigma - 0.7) / 0.3)
    KT = hs["k_a"] + (hs["k_s"] - hs["k_a"]) * ramp * c2 ** 2
    Kv = hs["k_f"] * ramp
    dt = 1200.0
    Vn, pn = G.forcing_held_suarez(rho, V, p, dt, hs)
    T = p / (rho * planet["Rd"])
    Tn = (T + KT * dt * Teq) / (1.0 + KT * dt)
    assert np.allclose(pn, rho * planet["Rd"] * Tn, rtol=1e-13, atol=0)
    assert np.allclose(Vn, V / (1.0 + Kv * dt)[..., None], rtol=1e-13, atol=1e-300)
    assert np.all(Vn[sigma < 0.7] == V[sigma < 0.7])                       # no drag above the boundary layer
    # the printed landmarks of Eq. 54, on a column whose lowest layer centre sits at p = p*: with a huge step the
    # update lands on T_eq: 315 K at the equator, 315 - 60 = 255 K at the poles, 200 K aloft; and on zero wind
    ps2 = 1.0e5 * np.exp(planet["gravity"] * G.z_c[0] / (planet["Rd"] * T0))
    rho2, _, _, p2 = ti.rest_state(planet, nv, G.N, ps2, T0)
    assert abs(p2[0, 0] - 1.0e5) < 1e-6
    eq, pole = int(np.argmin(np.abs(xyz[:, 2]))), int(np.argmax(xyz[:, 2]))
    Vbig, pbig = G.forcing_held_suarez(rho2, V, p2, 1.0e13, hs)
    Tbig = pbig / (rho2 * planet["Rd"])
    assert abs(Tbig[pole, 0] - 255.0) < 1e-3
    assert abs(Tbig[eq, 0] - (315.0 - 60.0 * xyz[eq, 2] ** 2)) < 1e-3
    assert np.all(np.abs(Tbig[:, -1] - 200.0) < 1e-3)                                # clipped aloft (top at 36 km)
    assert np.abs(Vbig[p2 / ps2 > 0.75]).max() < 1e-6 * np.abs(V).max()


def test_hot_jupiter_forcing_closed_forms(ogrid):
    """Eq. 59-61 by hand (G15: the second branch of T_vert is z > z_stra): with a huge step T lands on T_eq;
    at the substellar point's lowest layer T_eq = T_vert + beta dT_EP with beta -> sin(pi/2 (sigma - 0.12)/0.88),
    on the terminator (x = 0) T_eq = T_vert exactly, on the night side the contrast changes sign, above
    z_stra = 2000 km T_eq = 1600 - 2e-4 * 2e6 + 10 = 1210 K everywhere; T_vert is continuous at z_stra."""
    import oracle
    planet, nv = dict(ti.PAPER_HOT_JUPITER), 37
    xyz, nbr, C = ogrid(2, True)
    G = oracle.Geometry(xyz, nbr, nv, planet, C)
    hj = dict(ti.HOT_JUPITER_FORCING)
    rho, V, W, p = ti.rest_state(planet, nv, G.N, 1.0e5, 1600.0)
    pn = G.forcing_hot_jupiter(rho, p, 1.0e14, hj)
    T = pn / (rho * planet["Rd"])
    z, sigma = G.z_c, p[0] / 1.0e5                                   # isothermal hydrostatic column: p_s extrapolates to 1e5 exactly
    hz = 0.5 * hj["Gamma"] * (z - hj["z_stra"])
    Tvert = np.where(z <= hj["z_stra"], hj["T_surf"] - hj["Gamma"] * (hj["z_stra"] + 0.5 * (z - hj["z_stra"])) + np.sqrt(hz ** 2 + hj["dT_stra"] ** 2),
                     hj["T_surf"] - hj["Gamma"] * hj["z_stra"] + hj["dT_stra"])
    beta = np.where((z <= hj["z_stra"]) & (sigma > hj["sigma_stra"]), np.sin(np.pi * (sigma - hj["sigma_stra"]) / (2 * (1 - hj["sigma_stra"]))), 0.0)
    Teq = Tvert[None, :] + beta[None, :] * hj["dT_EP"] * xyz[:, 0][:, None]
    assert np.abs(T - Teq).max() < 1e-6
    assert np.all(np.abs(T[:, z > hj["z_stra"]] - 1210.0) < 1e-6)
    sub, anti = int(np.argmax(xyz[:, 0])), int(np.argmin(xyz[:, 0]))
    assert T[sub, 0] > Tvert[0] + 250.0 and T[anti, 0] < Tvert[0] - 250.0     # ~ +-300 K day-night contrast at depth
    k = int(np.searchsorted(z, hj["z_stra"]))
    assert abs(Tvert[k] - Tvert[k - 1]) < 2.0 * hj["Gamma"] * G.dz            # continuous across z_stra
    # finite step: Eq. 52 with K_T = 1/tau_rad
    dt = 600.0
    p2 = G.forcing_hot_jupiter(rho, p, dt, hj)
    KT = 1.0 / hj["tau_rad"]
    assert np.allclose(p2 / (rho * planet["Rd"]), (1600.0 + KT * dt * Teq) / (1.0 + KT * dt), rtol=1e-13, atol=0)
