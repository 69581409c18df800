"""Pins P1-P9 of the oracle's grid, geometry and horizontal operators.

Everything here runs on grids from the ORACLE's own generator (oracle/grid_oracle.py) and compares
the oracle with what the paper and the mathematics fix: printed values, closed forms, identities,
convergence order.  Nothing comes from the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import oracle
import thor_inputs as ti
from oracle import grid_oracle

NV = 3
PLANET = dict(ti.EARTH)


def _golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 2:
                out[line[0]] = float(line[1])
    return out


def _geom(ogrid, level, smooth=True, nv=NV):
    xyz, nbr, C = ogrid(level, smooth)
    return oracle.Geometry(xyz, nbr, nv, PLANET, C)


def test_p1_resolution_formulas_match_printed_values():
    g = _golden()
    assert ti.n_columns(5) == g["n_vertices_glevel5"]                        # Eq. 1
    dbar = math.sqrt(2 * math.pi / 5) * 7.0e7 / 2 ** 5                        # Eq. 2
    assert abs(dbar / 1e3 - g["dbar_km_A70000km_g5"]) < 1.0
    theta = math.degrees(math.sqrt(2 * math.pi / 5) / 2 ** 5)                # Eq. 3
    assert abs(theta - g["thetabar_deg_g5"]) < 0.05


def test_icosahedron_is_regular_and_counter_clockwise():
    g = _golden()
    pts, tris = grid_oracle.icosahedron()
    assert len(pts) == g["icosahedron_vertices"] and len(tris) == g["icosahedron_faces"]
    assert np.allclose(np.linalg.norm(pts, axis=1), 1.0)
    assert np.allclose(pts[0], [0, 0, 1]) and np.allclose(pts[11], [0, 0, -1])     # L45: poles
    e = np.linalg.norm(pts[tris] - pts[np.roll(tris, 1, axis=1)], axis=-1)
    assert np.allclose(e, e[0, 0])                                                  # 30 equal edges
    a, b, c = pts[tris[:, 0]], pts[tris[:, 1]], pts[tris[:, 2]]
    assert np.all(np.einsum("ij,ij->i", a, np.cross(b, c)) > 0)                     # CCW from outside


@pytest.mark.parametrize("level", [1, 3])
def test_p2_topology(ogrid, level):
    xyz, nbr, C = ogrid(level)
    N = len(xyz)
    assert N == ti.n_columns(level)
    deg = (nbr >= 0).sum(axis=1)
    assert (deg == 5).sum() == 12 and (deg == 6).sum() == N - 12
    assert deg.sum() == 2 * (3 * N - 6)                                     # 3N-6 edges
    for i in range(N):                                                     # symmetric relation
        for j in nbr[i, : deg[i]]:
            assert i in nbr[j, : deg[j]]
    G = oracle.Geometry(xyz, nbr, NV, PLANET, C)
    assert abs(G.Ac.sum() - 4 * math.pi) < 1e-12                           # areas tile the sphere
    # counter-clockwise ordering seen from outside
    for i in range(0, N, 7):
        m = deg[i]
        for k in range(m):
            a, b = xyz[nbr[i, k]], xyz[nbr[i, (k + 1) % m]]
            assert np.dot(xyz[i], np.cross(a, b)) > 0


def test_geometry_vectors_are_unit_outward_tangent(ogrid):
    G = _geom(ogrid, 3)
    for i in range(0, G.N, 5):
        m = G.deg[i]
        for k in range(m):
            n = G.nrm[i, k]
            c0, c1 = G.C[i, k], G.C[i, (k + 1) % m]
            assert abs(np.linalg.norm(n) - 1) < 1e-14
            assert abs(np.dot(n, c0)) < 1e-14 and abs(np.dot(n, c1)) < 1e-14      # normal to the arc plane
            mid = c0 + c1
            assert np.dot(n, mid / np.linalg.norm(mid) - G.xyz[i]) > 0            # outward (L67)
            assert abs(G.len[i, k] - math.acos(np.clip(np.dot(c0, c1), -1, 1))) < 1e-9
        assert np.allclose(G.bary[i, :m].sum(axis=1), 1.0, atol=1e-15)            # Eq. 5 weights sum to 1
        assert np.all(G.bary[i, :m] > 0.2) and np.all(G.bary[i, :m] < 0.5)        # near-centroid corners


def _integral_rhat(poly, nsub=80):
    """Brute-force quadrature of int r dA over a small convex spherical polygon: fan of planar
    triangles (c, a, b), each cut into nsub^2 small triangles whose centroids are projected to the
    sphere; solid-angle element = planar area * (plane normal . x) / |x|^3."""
    c = poly.mean(axis=0)
    tot = np.zeros(3)
    m = len(poly)
    uv = []
    for i in range(nsub):
        for j in range(nsub - i):
            uv.append(((i + 1 / 3) / nsub, (j + 1 / 3) / nsub))
            if i + j < nsub - 1:
                uv.append(((i + 2 / 3) / nsub, (j + 2 / 3) / nsub))
    uv = np.array(uv)
    assert len(uv) == nsub * nsub
    for k in range(m):
        a, b = poly[k], poly[(k + 1) % m]
        nvec = np.cross(a - c, b - c)
        x = c[None, :] + uv[:, :1] * (a - c)[None, :] + uv[:, 1:] * (b - c)[None, :]
        r = np.linalg.norm(x, axis=1)
        dA = np.abs(x @ nvec) / (2 * nsub ** 2) / r ** 3
        tot += ((x / r[:, None]) * dA[:, None]).sum(axis=0)
    return tot


def test_p4_eq13_centroid_identity(ogrid):
    """-sum l_k n_k = 2 int r dA, and it is parallel to the Eq. 13 centroid of the polygon (G4)."""
    G = _geom(ogrid, 2)
    for i in (0, 5, 17, 40):
        m = G.deg[i]
        s = -(G.len[i, :m, None] * G.nrm[i, :m]).sum(axis=0)
        cen = oracle.centroid_eq13(G.C[i, :m])
        assert np.linalg.norm(np.cross(s / np.linalg.norm(s), cen)) < 1e-13
        quad = 2 * _integral_rhat(G.C[i, :m])
        assert np.linalg.norm(s - quad) < 2e-3 * np.linalg.norm(s)
    # L120: the grid points sit exactly on the Eq. 13 centroids of their control volumes
    d = [np.linalg.norm(np.cross(oracle.centroid_eq13(G.C[i, : G.deg[i]]), G.xyz[i])) for i in range(G.N)]
    assert max(d) < 1e-13


def _l2(G, err):
    return math.sqrt(np.sum(G.Ac * err ** 2) / np.sum(G.Ac))              # Eq. 17


def _hr_errors(G, m, n):
    hr = ti.heikes_randall_fields(G.xyz, m, n)
    r = G.r_c[None, :]
    div = G.hdiv(np.repeat(hr["v"][:, None, :], G.nv, axis=1)) * r
    grad = G.hgrad(np.repeat(hr["beta"][:, None], G.nv, axis=1)) * r[..., None]
    ed = div[:, 1] - hr["div_v"]
    eg = np.linalg.norm(grad[:, 1] - hr["grad_beta"], axis=-1)
    return _l2(G, ed), np.abs(ed).max(), _l2(G, eg), eg.max()


def test_p5_operator_accuracy_second_order_on_modified_grid(ogrid):
    """Heikes-Randall fields (Eq. 14-18): l2 falls ~4x per g-level on the modified grid (L154),
    and the unmodified grid is visibly worse (Fig. 3-5)."""
    for (m, n) in ((1, 1), (3, 3)):
        e = {lvl: _hr_errors(_geom(ogrid, lvl), m, n) for lvl in (2, 3, 4)}
        for q in (0, 2):                                                    # l2 of div, l2 of grad
            order = math.log2(e[3][q] / e[4][q])
            assert 1.7 < order < 2.4, (m, n, q, order)
        for q in (1, 3):                                                    # l_inf, "slightly slower"
            order = math.log2(e[3][q] / e[4][q])
            assert 1.3 < order < 2.5, (m, n, q, order)
        # unmodified grid: larger errors and a visibly lower l_inf order (L148, Fig. 3-5)
        raw3 = _hr_errors(_geom(ogrid, 3, smooth=False), m, n)
        raw4 = _hr_errors(_geom(ogrid, 4, smooth=False), m, n)
        assert raw4[1] > (1.5 if m == 1 else 1.1) * e[4][1]
        assert raw4[3] > 1.1 * e[4][3]
        assert math.log2(raw3[1] / raw4[1]) < math.log2(e[3][1] / e[4][1]) - 0.2


def test_p6_gradient_of_constant_is_exactly_zero(ogrid):
    G = _geom(ogrid, 3)
    s = np.full((G.N, G.nv), 12345.678)
    assert np.all(G.hgrad(s) == 0.0)                                        # L86


def test_p7_divergence_of_constant_vector(ogrid):
    """div of a constant Cartesian vector c = c . sum l_k n_k / A_c exactly (Eq. 5 reproduces
    constants) and -> -2 c.r as the grid is refined."""
    c = np.array([0.3, -1.1, 0.7])
    errs = []
    for lvl in (2, 3):
        G = _geom(ogrid, lvl)
        d = G.hdiv(np.tile(c, (G.N, G.nv, 1))) * G.r_c[None, :]
        expect = np.array([np.dot(c, (G.len[i, : G.deg[i], None] * G.nrm[i, : G.deg[i]]).sum(axis=0)) / G.Ac[i]
                           for i in range(G.N)])
        assert np.abs(d[:, 0] - expect).max() < 1e-13
        errs.append(np.abs(d[:, 0] + 2 * G.xyz @ c).max())
    assert errs[1] < 0.3 * errs[0] and errs[1] < 0.01        # second order: P_0 is the centroid (L120)


def test_p8_spherical_harmonic_fields_converge(ogrid):
    """Config 1 fields: grad s vs analytic grad_h s, div v vs -f sum l(l+1) b Y / r (laplacian of
    spherical harmonics); observed order ~2."""
    e = {}
    for lvl in (3, 4):
        G = _geom(ogrid, lvl, nv=4)
        f = ti.harmonic_test_fields(G.xyz, PLANET, 4, seed=ti.SEED0 + 1)
        ed = (G.hdiv(f["v"]) - f["div_exact"])
        eg = np.linalg.norm(G.hgrad(f["s"]) - f["grad_exact"], axis=-1)
        e[lvl] = (_l2(G, ed[:, 2]) / _l2(G, f["div_exact"][:, 2]),
                  _l2(G, eg[:, 2]) / _l2(G, np.linalg.norm(f["grad_exact"][:, 2], axis=-1)))
    for q in (0, 1):
        assert 1.6 < math.log2(e[3][q] / e[4][q]) < 2.4, e
        assert e[4][q] < 0.08


def test_harmonic_fields_are_eigenfunctions():
    """Independent check of thor_inputs.real_sph_harm: orthonormality by quadrature on a
    lat-lon Gauss grid and tangency of the gradients."""
    nlat, nlon = 24, 48
    mu, w = np.polynomial.legendre.leggauss(nlat)
    lon = 2 * np.pi * np.arange(nlon) / nlon
    MU, LON = np.meshgrid(mu, lon, indexing="ij")
    xyz = np.stack([np.sqrt(1 - MU ** 2) * np.cos(LON), np.sqrt(1 - MU ** 2) * np.sin(LON), MU], axis=-1).reshape(-1, 3)
    W = np.repeat(w, nlon) * (2 * np.pi / nlon)
    Y, gY, ell = ti.real_sph_harm(xyz, 8)
    gram = (Y * W[:, None]).T @ Y
    assert np.abs(gram - np.eye(81)).max() < 1e-12
    assert np.abs(np.einsum("nkd,nd->nk", gY, xyz)).max() < 1e-12           # tangent
    # int |grad Y|^2 dA = l(l+1)
    g2 = np.einsum("nkd,nkd,n->k", gY, gY, W)
    assert np.abs(g2 - ell * (ell + 1)).max() < 1e-10


def test_p9_flux_antisymmetry(ogrid):
    """sum_i A_c,i div_i(Phi) = 0 to round-off for any Phi (each edge flux is shared, L190)."""
    G = _geom(ogrid, 3)
    rng = np.random.default_rng(3)
    vec = rng.standard_normal((G.N, G.nv, 3))
    d = G.hdiv(vec) * G.r_c[None, :]
    tot = (G.Ac[:, None] * d).sum(axis=0)
    scale = (G.Ac[:, None] * np.abs(d)).sum(axis=0)
    assert np.all(np.abs(tot) < 1e-14 * scale)


def test_p3_spring_dynamics_reduces_distortion(ogrid):
    """L100-L102: spring dynamics evens out the control-volume areas and the neighbour distances
    (the jumps next to the original icosahedron's edges)."""
    def spread(level, smooth):
        xyz, nbr, C = ogrid(level, smooth)
        G = oracle.Geometry(xyz, nbr, NV, PLANET, C)
        d = np.array([np.linalg.norm(xyz[i] - xyz[j]) for i in range(len(xyz)) for j in nbr[i][nbr[i] >= 0]])
        hexa = G.Ac[G.deg == 6]
        return d.std() / d.mean(), hexa.max() / hexa.min()
    raw, smooth = spread(3, False), spread(3, True)
    assert smooth[0] < 0.8 * raw[0]
    assert smooth[1] - 1 < 0.6 * (raw[1] - 1)


# --------------------------------------------------------------------------------------------
# NEXT-1 building block: the horizontal Laplacian of L369-L371 and the diffusion coefficient
# --------------------------------------------------------------------------------------------
def _lap_setup(ogrid, level, nv=2, lmax=4, seed=0):
    import oracle
    xyz, nbr, C = ogrid(level)
    G = oracle.Geometry(xyz, nbr, nv, ti.EARTH, C)
    Y, _, ell = ti.real_sph_harm(xyz, lmax)
    a = np.random.default_rng(seed).standard_normal(Y.shape[1])
    a[0] = 0.0
    s1 = Y @ a
    exact = -(Y * (ell * (ell + 1))[None, :]) @ a            # Laplace-Beltrami eigenfunctions on the unit sphere
    return G, np.repeat(s1[:, None], nv, axis=1), exact


def test_laplacian_of_a_constant_is_exactly_zero_and_it_is_in_flux_form(ogrid):
    G, s, _ = _lap_setup(ogrid, 3)
    assert np.all(G.hlap(np.full_like(s, 3.7)) == 0.0)
    lap = G.hlap(s)
    # Eq. 6 structure: every edge flux is shared by two control volumes with opposite normals and the
    # bit-identical corner vectors, so the area integral telescopes to round-off
    assert abs((G.Ac * lap[:, 0]).sum()) <= 1e-13 * (G.Ac * np.abs(lap[:, 0])).sum()
    # deep atmosphere: the same unit-sphere operator over r_k^2 in every layer
    assert np.allclose(lap[:, 0] * G.r_c[0] ** 2, lap[:, 1] * G.r_c[1] ** 2, rtol=1e-14, atol=0)


def test_laplacian_converges_on_spherical_harmonics(ogrid):
    """lap Y_lm = -l(l+1) Y_lm.  Second order in the bulk of the grid (median error falls ~4x per
    level), l2 falls every level; the twelve pentagons keep an O(1) error, as for any such stencil on
    a hexagonal-pentagonal grid, so l_inf is not asserted.  At these levels it beats div(grad)
    composed from Eq. 6 and Eq. 7 in l2 -- the reason the paper gives for the construction (L369)."""
    med, l2, l2_dg = {}, {}, {}
    for level in (2, 3, 4):
        G, s, exact = _lap_setup(ogrid, level)
        r2 = G.r_c[0] ** 2
        lap = G.hlap(s)[:, 0] * r2
        dg = G.hdiv(G.hgrad(s))[:, 0] * r2
        w = G.Ac / G.Ac.sum()
        scale = np.abs(exact).max()
        med[level] = np.median(np.abs(lap - exact)) / scale
        l2[level] = np.sqrt((w * (lap - exact) ** 2).sum() / (w * exact ** 2).sum())
        l2_dg[level] = np.sqrt((w * (dg - exact) ** 2).sum() / (w * exact ** 2).sum())
        hexagons = G.deg == 6
        assert np.abs(lap - exact)[hexagons].max() / scale < 0.12
    assert med[2] / med[3] > 3.0 and med[3] / med[4] > 3.0
    assert l2[2] > 2.0 * l2[3] and l2[3] > 2.0 * l2[4]
    assert all(l2[k] < l2_dg[k] for k in (2, 3, 4))


def test_diffusion_coefficient_formulas_and_table1_timescales():
    """Eq. 49-50 (L373-L381): K_d = D dbar^4/dt and tau_d = dbar^4/(2^5 K_d), so tau_d = dt/(32 D)
    whatever the resolution; with Table 1's timescales and the runs' time steps this gives the
    non-dimensional D the paper used (0.004837 Earth, 0.01992 hot Jupiter)."""
    import oracle
    gold = _golden()
    assert abs(oracle.dbar(7.0e7, 5) / 1e3 - gold["dbar_km_A70000km_g5"]) < 1.0          # Eq. 2
    for key, dt, radius, D_expect in (("tau_d_earth_s", 1000.0, 6.371e6, 0.004837), ("tau_d_hotjupiter_s", 600.0, 1.0e8, 0.01992)):
        tau = gold[key]
        D = dt / (32.0 * tau)
        assert abs(D - D_expect) < 5e-6
        for level in (4, 5, 6):
            db = oracle.dbar(radius, level)
            K = oracle.kd(D, db, dt)
            assert abs(oracle.tau_d(db, K) - tau) <= 1e-12 * tau
            assert abs(K - D * db ** 4 / dt) <= 1e-15 * K
