"""Host grid generator of the library (thor_grid_create) against the oracle's independent
generator (pin P3) and the oracle's geometry.  Host only: runs without a GPU."""
import math

import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle
import paper_1607_05535_b200 as thor
import thor_inputs as ti
from oracle import grid_oracle


@pytest.fixture(scope="module")
def lib_grid3():
    return thor.Grid(3, 4, ti.EARTH)


def test_p3_library_grid_matches_the_oracle_generator(lib_grid3):
    v = lib_grid3.view
    xyz, nbr, C, _ = grid_oracle.build(3, tol=1e-9)
    assert v["n_cols"] == len(xyz) == ti.n_columns(3)
    dist, idx = cKDTree(xyz).query(v["xyz"])
    assert len(set(idx)) == len(idx)                       # one-to-one
    assert dist.max() < 2e-6                               # both converged to the same equilibrium
    # same topology under that matching
    for i in range(0, v["n_cols"], 3):
        mine = {idx[j] for j in v["nbr"][i] if j >= 0}
        theirs = {j for j in nbr[idx[i]] if j >= 0}
        assert mine == theirs
    # control-volume vertices agree too (triangle centroids of the pre-move grid)
    dC, _ = cKDTree(C[:, :5].reshape(-1, 3)).query(v["cv_vertex"][:, :5].reshape(-1, 3))
    assert dC.max() < 2e-6


def test_exported_geometry_matches_the_oracle_recomputation(lib_grid3):
    v = lib_grid3.view
    G = oracle.Geometry(v["xyz"], v["nbr"], 4, ti.EARTH, v["cv_vertex"])
    assert np.abs(G.Ac - v["area"]).max() < 1e-15
    assert np.abs(G.len - v["edge_len"]).max() < 1e-15
    assert np.abs(G.nrm - v["edge_nrm"]).max() < 1e-14
    assert abs(v["area"].sum() - 4 * math.pi) < 1e-12
    # L120: every point is the Eq. 13 centroid of its control volume
    deg = (v["nbr"] >= 0).sum(axis=1)
    d = [np.linalg.norm(np.cross(oracle.centroid_eq13(v["cv_vertex"][i, : deg[i]]), v["xyz"][i])) for i in range(v["n_cols"])]
    assert max(d) < 1e-13


@pytest.mark.parametrize("level", [0, 1, 5])
def test_topology_and_device_order(level):
    g = thor.Grid(level, 2, ti.EARTH)
    v = g.view
    N = v["n_cols"]
    assert N == ti.n_columns(level)
    deg = (v["nbr"] >= 0).sum(axis=1)
    assert (deg == 5).sum() == 12 and deg.sum() == 2 * (3 * N - 6)
    assert sorted(v["device_order"]) == list(range(N))                      # a permutation
    assert np.allclose(np.linalg.norm(v["xyz"], axis=1), 1.0, atol=1e-15)
    if level >= 5:
        # device order = rhombus by rhombus along the Morton curve of the lattice: every aligned run of
        # 4 / 8 / 16 columns is a 2x2 / 2x4 / 4x4 patch, whose halo (distinct neighbours outside the run)
        # is the minimum 10 / 14 / 18 columns; and neighbours sit close in memory
        rank = np.empty(N, dtype=np.int64)
        rank[v["device_order"]] = np.arange(N)
        dn = np.where(v["nbr"] >= 0, rank[np.where(v["nbr"] >= 0, v["nbr"], 0)], -1)[v["device_order"]]
        for tc, hmax in ((4, 10), (8, 14), (16, 18)):
            halos = []
            for t in range(0, N - tc + 1, tc):
                own = set(range(t, t + tc))
                halos.append(len({int(x) for x in dn[t:t + tc].ravel() if x >= 0} - own))
            assert max(halos) <= hmax and np.mean(halos) > hmax - 1
        gaps = np.abs(dn - np.arange(N)[:, None])[dn >= 0]
        assert np.median(gaps) < 64


def test_operator_accuracy_on_library_grids():
    """P5 on the library's own grids, through the oracle's operators: second order 4 -> 5."""
    e = {}
    for lvl in (4, 5):
        v = thor.Grid(lvl, 2, ti.EARTH).view
        G = oracle.Geometry(v["xyz"], v["nbr"], 2, ti.EARTH, v["cv_vertex"])
        hr = ti.heikes_randall_fields(v["xyz"], 1, 1)
        d = G.hdiv(np.repeat(hr["v"][:, None, :], 2, axis=1)) * G.r_c[None, :]
        err = d[:, 0] - hr["div_v"]
        e[lvl] = (math.sqrt(np.sum(G.Ac * err ** 2) / G.Ac.sum()), np.abs(err).max())
    assert 1.8 < math.log2(e[4][0] / e[5][0]) < 2.2
    assert 1.7 < math.log2(e[4][1] / e[5][1]) < 2.3


@pytest.mark.parametrize("level", [2, 3, 4])
def test_interior_lattice_points_have_the_six_fixed_neighbour_offsets(level):
    """What the kernels' computed neighbour indices rest on (thor_kernels.cuh: neighbours()): the device order is
    rhombus by rhombus along the Morton curve of (I, J-1), and a lattice point that is not on the rim of its rhombus has
    its six neighbours in the same rhombus at the offsets (1,0), (0,1), (-1,1), (-1,0), (0,-1), (1,-1), counter-clockwise."""
    g = thor.Grid(level, 4, ti.EARTH)
    v = g.view
    n, N = 1 << level, g.n_cols
    order, nbr = v["device_order"], v["nbr"]
    rank = np.empty(N, dtype=np.int64)
    rank[order] = np.arange(N)

    def lattice(m):
        I = sum(((m >> (2 * b + 1)) & 1) << b for b in range(16))
        J = sum(((m >> (2 * b)) & 1) << b for b in range(16))
        return I, J

    want = [(1, 0), (0, 1), (-1, 1), (-1, 0), (0, -1), (1, -1)]
    seen = 0
    for d in range(10 * n * n):
        r, m = divmod(d, n * n)
        I, J = lattice(m)
        if not (1 <= I <= n - 2 and 1 <= J <= n - 2):
            continue
        offs = []
        for k in range(6):
            rn, mn = divmod(int(rank[nbr[order[d], k]]), n * n)
            assert rn == r
            In, Jn = lattice(mn)
            offs.append((In - I, Jn - J))
        i0 = offs.index((1, 0))
        assert offs[i0:] + offs[:i0] == want, (d, offs)
        seen += 1
    assert seen == 10 * (n - 2) ** 2
    g.close()
