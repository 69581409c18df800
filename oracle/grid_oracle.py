"""oracle/grid_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Independent, literal numpy statement of the paper's grid construction:
icosahedron with two polar vertices -> g rounds of edge bisection projected to the unit sphere
(L45-L49) -> spring dynamics (Eq. 10-12) -> centroid relocation (Eq. 13).
It is used (a) to run the oracle's geometry pins on a grid that does not come from the CUDA
library and (b) to cross-check the library's own generator (pin P3).  It shares no code with
paper_1607_05535_b200/.

Readings: G2 spring constant k = 1; G3 the stopping test is the
largest per-step displacement on the unit sphere, `tol` (paper: 1e-5; callers may tighten it);
G4 Eq. 13 uses the arc atan2(|a x b|, a.b) and the result is normalised; R4 (as revised in
DESIGN.md): the control-volume vertices C_k stay where L120 puts them (centroids of the triangles
of the PRE-move positions) and are part of the grid description next to the positions.
Orientation convention shared with the library (the paper only says "two of the twelve vertices
are placed at each pole", L45): north pole +z, upper ring at longitudes 72 deg * j, lower ring at
36 deg + 72 deg * j, latitude +-atan(1/2).
"""
import numpy as np


def icosahedron():
    """12 vertices, 20 counter-clockwise (seen from outside) triangles."""
    lat = np.arctan(0.5)
    pts = [(0.0, 0.0, 1.0)]
    for j in range(5):
        lon = 2 * np.pi * j / 5
        pts.append((np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), np.sin(lat)))
    for j in range(5):
        lon = 2 * np.pi * (j + 0.5) / 5
        pts.append((np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), -np.sin(lat)))
    pts.append((0.0, 0.0, -1.0))
    tris = []
    for j in range(5):
        u0, u1 = 1 + j, 1 + (j + 1) % 5
        l0, l1 = 6 + j, 6 + (j + 1) % 5
        tris.append((0, u0, u1))        # north cap
        tris.append((u0, l0, u1))       # upper band
        tris.append((u1, l0, l1))       # lower band
        tris.append((11, l1, l0))       # south cap
    return np.array(pts, dtype=np.float64), np.array(tris, dtype=np.int64)


def bisect(pts, tris):
    """One refinement: bisect every edge, project the midpoints to the sphere (L45, Fig. 1)."""
    pts = [tuple(p) for p in pts]
    mid = {}

    def midpoint(a, b):
        key = (a, b) if a < b else (b, a)
        if key not in mid:
            m = np.array(pts[a]) + np.array(pts[b])
            m /= np.linalg.norm(m)
            mid[key] = len(pts)
            pts.append(tuple(m))
        return mid[key]

    out = []
    for a, b, c in tris:
        ab, bc, ca = midpoint(a, b), midpoint(b, c), midpoint(c, a)
        out += [(a, ab, ca), (ab, b, bc), (ca, bc, c), (ab, bc, ca)]
    return np.array(pts, dtype=np.float64), np.array(out, dtype=np.int64)


def neighbour_table(pts, tris):
    """[N][6] neighbours in counter-clockwise order seen from outside; pentagons end with -1."""
    n = len(pts)
    nxt = [dict() for _ in range(n)]          # around vertex v: neighbour a is followed by b
    for a, b, c in tris:
        nxt[a][b] = c
        nxt[b][c] = a
        nxt[c][a] = b
    nbr = -np.ones((n, 6), dtype=np.int32)
    for v in range(n):
        start = min(nxt[v].keys())
        ring = [start]
        while True:
            w = nxt[v][ring[-1]]
            if w == start:
                break
            ring.append(w)
        assert len(ring) in (5, 6) and len(ring) == len(nxt[v])
        nbr[v, : len(ring)] = ring
    return nbr


def _arc(a, b):
    c = np.cross(a, b)
    return np.arctan2(np.linalg.norm(c, axis=-1), np.sum(a * b, axis=-1))


def spring_dynamics(pts, nbr, level, beta=1.15, alpha=1.0, k=1.0, dt=0.01, tol=1e-5, max_iter=2000000):
    """Eq. 10-12 (L104-L118).  The 12 pentagon centres stay fixed (L109)."""
    x = pts.copy()
    n = len(x)
    deg6 = nbr[:, 5] >= 0
    nb = nbr.copy()
    nb[~deg6, 5] = nb[~deg6, 0]               # placeholder, masked below
    mask = np.ones((n, 6))
    mask[~deg6, 5] = 0.0
    d_spr = beta * 2 * np.pi / (10 * 2 ** (level - 1))      # Eq. 12 with A = 1
    v = np.zeros_like(x)
    it = 0
    for it in range(max_iter):
        xn = x[nb]                                           # [n][6][3]
        x0 = x[:, None, :]
        d = _arc(np.broadcast_to(x0, xn.shape), xn)          # arc length d_i
        t = xn - np.sum(xn * x0, axis=-1, keepdims=True) * x0
        t /= np.linalg.norm(t, axis=-1, keepdims=True)       # unit tangent e_i at P_0 towards P_i
        force = np.sum((k * (d - d_spr) * mask)[..., None] * t, axis=1) - alpha * v   # Eq. 10
        v = v + dt * force
        v[~deg6] = 0.0
        xnew = x + dt * v                                    # Eq. 11
        xnew /= np.linalg.norm(xnew, axis=-1, keepdims=True)
        move = np.max(np.linalg.norm(xnew - x, axis=-1))
        x = xnew
        v = v - np.sum(v * x, axis=-1, keepdims=True) * x    # keep the velocity tangent
        if move < tol:
            break
    return x, it + 1


def _centroid_eq13(r):
    """Eq. 13 (G4) for a batch of polygons r[..., n, 3] (all n vertices valid)."""
    a = r
    b = np.roll(r, -1, axis=-2)
    c = np.cross(a, b)
    l = np.linalg.norm(c, axis=-1, keepdims=True)
    ang = np.arctan2(l[..., 0], np.sum(a * b, axis=-1))[..., None]
    s = np.sum(c / l * ang, axis=-2)
    return s / np.linalg.norm(s, axis=-1, keepdims=True)


def triangle_centroids(pts, nbr):
    """C [N][6][3]: Eq. 13 centroid (n = 3) of the triangle (P_0, P_k, P_k+1) for every corner k.
    The three vertices are taken in a canonical rotation (smallest index first, orientation kept)
    so that the three columns sharing a triangle hold bit-identical copies.  Pentagons: C[i][5] = 0."""
    n = len(pts)
    C = np.zeros((n, 6, 3))
    for m in (5, 6):
        idx = np.where((nbr[:, 5] >= 0) == (m == 6))[0]
        nb = nbr[idx, :m]
        tri = np.stack([np.broadcast_to(idx[:, None], nb.shape), nb, np.roll(nb, -1, axis=1)], axis=-1)
        rot = np.argmin(tri, axis=-1)[..., None]
        tri = np.take_along_axis(tri, (rot + np.arange(3)) % 3, axis=-1)           # [.., m, 3]
        C[idx[:, None], np.arange(m)[None, :]] = _centroid_eq13(pts[tri])
    return C


def centroid_relocation(pts, nbr):
    """L120: C_k -> centroids of the triangles; then, C fixed, P_i -> Eq. 13 centroid of its
    polygon of C points.  Returns (new positions, C)."""
    C = triangle_centroids(pts, nbr)
    out = pts.copy()
    for m in (5, 6):
        idx = np.where((nbr[:, 5] >= 0) == (m == 6))[0]
        out[idx] = _centroid_eq13(C[idx, :m])
    return out, C


def build(level, smooth=True, tol=1e-5, max_iter=2000000):
    """Return (xyz [N][3], nbr [N][6] int32, C [N][6][3] control-volume vertices, iterations)."""
    pts, tris = icosahedron()
    for _ in range(level):
        pts, tris = bisect(pts, tris)
    nbr = neighbour_table(pts, tris)
    its = 0
    if smooth:
        pts, its = spring_dynamics(pts, nbr, level, tol=tol, max_iter=max_iter)
        pts, C = centroid_relocation(pts, nbr)
    else:
        C = triangle_centroids(pts, nbr)
    return np.ascontiguousarray(pts), nbr, np.ascontiguousarray(C), its
