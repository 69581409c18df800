// Host icosahedral grid generator + finite-volume stencil weights.
//
//   icosahedron, two vertices on the poles
//   -> recursive edge bisection, new points projected to the unit sphere (L45-L49, Fig. 1)
//   -> spring dynamics (Eq. 10-12; beta = 1.15, alpha = 1, k = 1 (G2), dt = 0.01)
//   -> centroid move (Eq. 13 with reading G4, L120-L125): C_k to the triangle centroids, then,
//      C fixed, P_i to the centroid of its control volume
//   -> stencil weights of Eq. 4-7 expanded per neighbour, device column order.
//
// Design choices that differ from a literal reading ("grid generator"):
//   * The relaxation is hierarchical: every refinement level is relaxed before it is bisected
//     again, so the finer level starts next to its equilibrium and only its short wavelengths
//     have to decay.  The equilibrium of Eq. 10 does not depend on where the iteration starts.
//   * G3: the paper's stopping test (no point moves more than 1e-5 in a step) is met by the very
//     first step of a grid that starts at rest; here the iteration runs until the largest
//     per-step displacement stays below kSpringTol after the initial transient.
#include "grid_host.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <unordered_map>

namespace thor {
namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr double kBeta = 1.15;       // L118
constexpr double kAlpha = 1.0;       // L118
constexpr double kSpringK = 1.0;     // G2
constexpr double kSpringDt = 0.01;   // L118
constexpr double kSpringTol = 1e-9;  // G3 (per-step displacement on the unit sphere)
constexpr double kSpringTolGrowth = 4.0;   // per level above 4; measured: no effect on the operator errors
constexpr int kSpringMinIter = 200;
constexpr int kSpringMaxIter = 60000;

struct V3 {
    double x, y, z;
};
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double norm(V3 a) { return std::sqrt(dot(a, a)); }
inline V3 unit(V3 a) { return (1.0 / norm(a)) * a; }
inline double arc(V3 a, V3 b) { return std::atan2(norm(cross(a, b)), dot(a, b)); }

// A triangle and, for the device column order, the position of its corners on the lattice of the
// rhombus it belongs to: the 20 faces pair into 10 rhombi (L45 "ten rhombuses"), each an n x n
// lattice (n = 2^level) with corners (0,0), (n,0), (0,n), (n,n) and the shared face edge on the
// short diagonal (n,0)-(0,n).
struct Tri {
    int a, b, c;
    int r = 0;                       // rhombus 0..9
    int ia = 0, ja = 0, ib = 0, jb = 0, ic = 0, jc = 0;
};

void icosahedron(std::vector<V3>& pts, std::vector<Tri>& tris, int n) {
    const double lat = std::atan(0.5);
    pts.clear();
    tris.clear();
    pts.push_back({0, 0, 1});
    for (int j = 0; j < 5; ++j) {
        double lon = 2 * kPi * j / 5;
        pts.push_back({std::cos(lat) * std::cos(lon), std::cos(lat) * std::sin(lon), std::sin(lat)});
    }
    for (int j = 0; j < 5; ++j) {
        double lon = 2 * kPi * (j + 0.5) / 5;
        pts.push_back({std::cos(lat) * std::cos(lon), std::cos(lat) * std::sin(lon), -std::sin(lat)});
    }
    pts.push_back({0, 0, -1});
    // five north-to-south strips of four faces; counter-clockwise seen from outside
    for (int j = 0; j < 5; ++j) {
        int u0 = 1 + j, u1 = 1 + (j + 1) % 5, l0 = 6 + j, l1 = 6 + (j + 1) % 5;
        tris.push_back({0, u0, u1, 2 * j, 0, 0, n, 0, 0, n});
        tris.push_back({u0, l0, u1, 2 * j, n, 0, n, n, 0, n});
        tris.push_back({u1, l0, l1, 2 * j + 1, 0, 0, n, 0, 0, n});
        tris.push_back({11, l1, l0, 2 * j + 1, n, n, 0, n, n, 0});
    }
}

// One refinement (L45): children of triangle t are stored at 4t..4t+3, so the triangle list stays
// in quadtree (depth-first) order -- the device column order below relies on that.
void bisect(std::vector<V3>& pts, std::vector<Tri>& tris) {
    std::unordered_map<uint64_t, int> mid;
    mid.reserve(tris.size() * 2);
    auto midpoint = [&](int a, int b) {
        uint64_t key = a < b ? (uint64_t(a) << 32) | uint32_t(b) : (uint64_t(b) << 32) | uint32_t(a);
        auto it = mid.find(key);
        if (it != mid.end()) return it->second;
        int id = int(pts.size());
        pts.push_back(unit(pts[a] + pts[b]));
        mid.emplace(key, id);
        return id;
    };
    std::vector<Tri> out;
    out.reserve(tris.size() * 4);
    for (const Tri& t : tris) {
        int ab = midpoint(t.a, t.b), bc = midpoint(t.b, t.c), ca = midpoint(t.c, t.a);
        const int iab = (t.ia + t.ib) / 2, jab = (t.ja + t.jb) / 2, ibc = (t.ib + t.ic) / 2, jbc = (t.jb + t.jc) / 2;
        const int ica = (t.ic + t.ia) / 2, jca = (t.jc + t.ja) / 2;
        out.push_back({t.a, ab, ca, t.r, t.ia, t.ja, iab, jab, ica, jca});
        out.push_back({ab, bc, ca, t.r, iab, jab, ibc, jbc, ica, jca});
        out.push_back({ab, t.b, bc, t.r, iab, jab, t.ib, t.jb, ibc, jbc});
        out.push_back({ca, bc, t.c, t.r, ica, jca, ibc, jbc, t.ic, t.jc});
    }
    tris.swap(out);
}

// Neighbours of every vertex in counter-clockwise order (seen from outside), starting from the
// smallest neighbour index; pentagons are padded with -1.
bool neighbour_table(int N, const std::vector<Tri>& tris, std::vector<int>& nbr, std::vector<int>& deg) {
    std::vector<int> from(size_t(N) * 6, -1), to(size_t(N) * 6, -1), cnt(N, 0);
    auto add = [&](int v, int a, int b) {
        if (cnt[v] >= 6) return false;
        from[size_t(v) * 6 + cnt[v]] = a;
        to[size_t(v) * 6 + cnt[v]] = b;
        ++cnt[v];
        return true;
    };
    for (const Tri& t : tris)
        if (!add(t.a, t.b, t.c) || !add(t.b, t.c, t.a) || !add(t.c, t.a, t.b)) return false;
    nbr.assign(size_t(N) * 6, -1);
    deg.assign(N, 0);
    for (int v = 0; v < N; ++v) {
        int m = cnt[v];
        if (m != 5 && m != 6) return false;
        const int* f = &from[size_t(v) * 6];
        const int* t = &to[size_t(v) * 6];
        int cur = *std::min_element(f, f + m);
        for (int k = 0; k < m; ++k) {
            nbr[size_t(v) * 6 + k] = cur;
            int nxt = -1;
            for (int q = 0; q < m; ++q)
                if (f[q] == cur) nxt = t[q];
            if (nxt < 0) return false;
            cur = nxt;
        }
        deg[v] = m;
    }
    return true;
}

// Eq. 10-12 on the host.  Returns the number of steps taken.
int spring_dynamics_host(int N, double* xyz, const int* nbr, const int* deg, const SpringParams& sp) {
    std::vector<V3> x(N), v(N, V3{0, 0, 0}), xn(N);
    for (int i = 0; i < N; ++i) x[i] = V3{xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2]};
    int it = 0;
    for (; it < sp.max_iter; ++it) {
        double worst = 0.0;
#pragma omp parallel for schedule(static) reduction(max : worst)
        for (int i = 0; i < N; ++i) {
            if (deg[i] == 5) {   // the twelve pentagon centres stay fixed (L109)
                xn[i] = x[i];
                continue;
            }
            const V3 p0 = x[i];
            V3 f{0, 0, 0};
            for (int k = 0; k < 6; ++k) {
                const V3 pj = x[nbr[size_t(i) * 6 + k]];
                double d = arc(p0, pj);
                V3 e = unit(pj - dot(pj, p0) * p0);               // unit tangent at P_0 towards P_j
                f = f + (sp.k * (d - sp.dspr)) * e;
            }
            f = f - sp.alpha * v[i];                              // Eq. 10
            V3 vi = v[i] + sp.dt * f;
            V3 pn = unit(p0 + sp.dt * vi);                        // Eq. 11, back onto the sphere
            v[i] = vi - dot(vi, pn) * pn;
            xn[i] = pn;
            worst = std::max(worst, norm(pn - p0));
        }
        x.swap(xn);
        if (it >= sp.min_iter && worst < sp.tol) {
            ++it;
            break;
        }
    }
    for (int i = 0; i < N; ++i) { xyz[3 * i] = x[i].x; xyz[3 * i + 1] = x[i].y; xyz[3 * i + 2] = x[i].z; }
    return it;
}

// the constants of one level's relaxation
SpringParams spring_params(int level) {
    SpringParams sp;
    sp.dspr = kBeta * 2 * kPi / (10.0 * std::pow(2.0, level - 1));   // Eq. 12, A = 1
    sp.k = kSpringK; sp.alpha = kAlpha; sp.dt = kSpringDt;
    // the tolerance follows the grid spacing above level 4 (a fixed displacement is a smaller and
    // smaller fraction of an edge there, and the long waves were already relaxed on the coarser levels)
    sp.tol = kSpringTol * std::pow(kSpringTolGrowth, std::max(0, level - 4));
    sp.min_iter = kSpringMinIter; sp.max_iter = kSpringMaxIter;
    return sp;
}

// Eq. 13 (G4): sum_i (r_i x r_i+1)/|r_i x r_i+1| * arc(r_i, r_i+1), normalised.
V3 centroid(const V3* r, int n) {
    V3 s{0, 0, 0};
    for (int i = 0; i < n; ++i) {
        V3 c = cross(r[i], r[(i + 1) % n]);
        double l = norm(c);
        s = s + (std::atan2(l, dot(r[i], r[(i + 1) % n])) / l) * c;
    }
    return unit(s);
}

double tri_area(V3 a, V3 b, V3 c) {   // spherical excess
    return 2.0 * std::atan2(std::fabs(dot(a, cross(b, c))), 1.0 + dot(a, b) + dot(b, c) + dot(c, a));
}

}  // namespace

int build_host_grid(int level, int nv, const thor_planet& P, HostGrid& g, const double* z_interfaces, int kord,
                    SpringFn spring, bool shallow) {
    if (level < 0 || level > 9 || nv < 2 || nv > 128) return THOR_EINVAL;
    if (kord != 1 && kord != 3) return THOR_EINVAL;
    if (z_interfaces) {
        if (z_interfaces[0] != 0.0) return THOR_EINVAL;
        for (int k = 0; k < nv; ++k)
            if (!(z_interfaces[k + 1] > z_interfaces[k])) return THOR_EINVAL;
    }
    if (!(P.radius > 0) || !(P.z_top > 0) || !(P.Rd > 0) || !(P.Cp > P.Rd) || !(P.p_ref > 0)) return THOR_EINVAL;
    g.level = level;
    g.nv = nv;
    g.P = P;
    if (z_interfaces) g.P.z_top = z_interfaces[nv];      // the lid is the last interface

    std::vector<V3> pts;
    std::vector<Tri> tris;
    std::vector<int> nbr, deg;
    icosahedron(pts, tris, 1 << level);
    g.spring_iterations = 0;
    for (int l = 1; l <= level; ++l) {
        bisect(pts, tris);
        if (!neighbour_table(int(pts.size()), tris, nbr, deg)) return THOR_EINVAL;
        static_assert(sizeof(V3) == 3 * sizeof(double), "V3 is three packed doubles");
        const int its = (spring ? spring : spring_dynamics_host)(int(pts.size()), &pts[0].x, nbr.data(), deg.data(), spring_params(l));
        if (its < 0) return THOR_ECUDA;
        g.spring_iterations += its;
    }
    if (level == 0 && !neighbour_table(int(pts.size()), tris, nbr, deg)) return THOR_EINVAL;
    const int N = int(pts.size());
    g.N = N;
    g.nbr = nbr;
    g.deg = deg;

    // --- centroid move (L120).  One C per triangle, shared bit-identically by its three columns.
    const int T = int(tris.size());
    std::vector<V3> Ctri(T);
    for (int t = 0; t < T; ++t) {
        V3 r[3] = {pts[tris[t].a], pts[tris[t].b], pts[tris[t].c]};
        Ctri[t] = centroid(r, 3);
    }
    // corner k of column i = the triangle (i, nbr[k], nbr[k+1]); find it through an edge map
    std::unordered_map<uint64_t, int> tri_of_edge;   // directed edge (a -> b) -> triangle on its left
    tri_of_edge.reserve(size_t(T) * 3);
    auto ekey = [](int a, int b) { return (uint64_t(uint32_t(a)) << 32) | uint32_t(b); };
    for (int t = 0; t < T; ++t) {
        tri_of_edge[ekey(tris[t].a, tris[t].b)] = t;
        tri_of_edge[ekey(tris[t].b, tris[t].c)] = t;
        tri_of_edge[ekey(tris[t].c, tris[t].a)] = t;
    }
    std::vector<int> corner_tri(size_t(N) * 6, -1);
    g.cv.assign(size_t(N) * 18, 0.0);
    for (int i = 0; i < N; ++i)
        for (int k = 0; k < deg[i]; ++k) {
            auto it = tri_of_edge.find(ekey(i, nbr[size_t(i) * 6 + k]));
            if (it == tri_of_edge.end()) return THOR_EINVAL;
            corner_tri[size_t(i) * 6 + k] = it->second;
            const V3 c = Ctri[it->second];
            double* o = &g.cv[size_t(i) * 18 + 3 * k];
            o[0] = c.x; o[1] = c.y; o[2] = c.z;
        }
    if (level > 0) {
        std::vector<V3> moved(N);
        for (int i = 0; i < N; ++i) {
            V3 poly[6];
            for (int k = 0; k < deg[i]; ++k) poly[k] = Ctri[corner_tri[size_t(i) * 6 + k]];
            moved[i] = centroid(poly, deg[i]);
        }
        pts.swap(moved);
    }
    g.xyz.resize(size_t(N) * 3);
    for (int i = 0; i < N; ++i) { g.xyz[3 * i] = pts[i].x; g.xyz[3 * i + 1] = pts[i].y; g.xyz[3 * i + 2] = pts[i].z; }

    // --- Eq. 5 weights per triangle (vertex order of the triangle list), from the FINAL P and the fixed C
    std::vector<double> bary(size_t(T) * 3);
    for (int t = 0; t < T; ++t) {
        V3 a = pts[tris[t].a], b = pts[tris[t].b], c = pts[tris[t].c], C = Ctri[t];
        double wa = tri_area(b, c, C), wb = tri_area(c, a, C), wc = tri_area(a, b, C);
        double s = wa + wb + wc;
        bary[size_t(t) * 3 + 0] = wa / s;   // each vertex is weighted by the sub-triangle opposite to it
        bary[size_t(t) * 3 + 1] = wb / s;
        bary[size_t(t) * 3 + 2] = wc / s;
    }
    // --- Eq. 7 on the primary grid (L369): gradient of a scalar on triangle t at its centre C_t as a
    // combination of the three vertex values, G_t = sum_v gw[t][v] s_v with
    //   G = sum_e E_e (s_e1 + s_e2 - 2 s_m),  E_e = l_e n_e / (2 A_T),  s_m = Eq. 5 value at C_t
    std::vector<V3> gw(size_t(T) * 3);
    for (int t = 0; t < T; ++t) {
        const V3 v[3] = {pts[tris[t].a], pts[tris[t].b], pts[tris[t].c]};
        const double AT = tri_area(v[0], v[1], v[2]);
        V3 Ee[3], ES{0, 0, 0};
        for (int e = 0; e < 3; ++e) {
            const V3 x = v[e], y = v[(e + 1) % 3];
            const V3 n = cross(x, y);
            Ee[e] = (-arc(x, y) / (2.0 * AT * norm(n))) * n;          // outward for counter-clockwise order
            ES = ES + Ee[e];
        }
        for (int q = 0; q < 3; ++q)                                     // vertex q sits on edges q-1 and q
            gw[size_t(t) * 3 + q] = Ee[(q + 2) % 3] + Ee[q] - (2.0 * bary[size_t(t) * 3 + q]) * ES;
    }
    auto gw_of = [&](int t, int v) {
        if (tris[t].a == v) return gw[size_t(t) * 3 + 0];
        if (tris[t].b == v) return gw[size_t(t) * 3 + 1];
        return gw[size_t(t) * 3 + 2];
    };
    auto weight_of = [&](int t, int v) {
        if (tris[t].a == v) return bary[size_t(t) * 3 + 0];
        if (tris[t].b == v) return bary[size_t(t) * 3 + 1];
        return bary[size_t(t) * 3 + 2];
    };

    // --- device column order.  Every rhombus owns the lattice points 0 <= I < n, 0 < J <= n (the ten
    // half-open rhombi tile the sphere; the two poles are left over), and its columns are laid out
    // along the Morton (Z-order) curve of (I, J-1): every aligned run of 4 / 8 / 16 columns is a
    // 2x2 / 2x4 / 4x4 lattice patch, so the tiles the kernels stage in shared memory have the
    // smallest possible halo (10 / 14 / 18 columns) and neighbours sit close in memory.
    g.order.assign(N, -1);
    g.rank.assign(N, -1);
    {
        const long long n = 1LL << level;
        auto morton = [](unsigned x, unsigned y) {
            unsigned long long m = 0;
            for (int b = 0; b < 16; ++b) m |= ((unsigned long long)((x >> b) & 1u) << (2 * b + 1)) | ((unsigned long long)((y >> b) & 1u) << (2 * b));
            return m;
        };
        std::vector<long long> key(N, -1);
        auto claim = [&](int v, int r, int I, int J) {
            if (I >= 0 && I < n && J > 0 && J <= n) key[v] = (long long)r * n * n + (long long)morton(unsigned(I), unsigned(J - 1));
        };
        for (const Tri& t : tris) { claim(t.a, t.r, t.ia, t.ja); claim(t.b, t.r, t.ib, t.jb); claim(t.c, t.r, t.ic, t.jc); }
        int poles = 0;
        for (int v = 0; v < N; ++v)
            if (key[v] < 0) key[v] = 10 * n * n + poles++;
        if (poles != 2) return THOR_EINVAL;
        std::vector<int> idx(N);
        for (int v = 0; v < N; ++v) idx[v] = v;
        std::sort(idx.begin(), idx.end(), [&](int x, int y) { return key[x] < key[y]; });
        for (int d = 0; d < N; ++d) {
            if (d > 0 && key[idx[d]] == key[idx[d - 1]]) return THOR_EINVAL;    // every column has one owner
            g.order[d] = idx[d];
            g.rank[idx[d]] = d;
        }
    }

    // --- l_k, n_k, A_c (Eq. 4, 6) and the expanded stencil weights
    g.area.assign(N, 0.0);
    g.len.assign(size_t(N) * 6, 0.0);
    g.nrm.assign(size_t(N) * 18, 0.0);
    g.d_nbr.assign(size_t(N) * 6, 0);
    g.d_wdiv.assign(size_t(N) * 21, 0.0);
    g.d_wgrad.assign(size_t(N) * 18, 0.0);
    g.d_rhat.assign(size_t(N) * 3, 0.0);
    g.d_wlap.assign(size_t(N) * 6, 0.0);
    g.d_area.assign(N, 0.0);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        const int m = deg[i];
        const V3 p0 = pts[i];
        V3 C[6], E[6], ln[6];
        for (int k = 0; k < m; ++k) C[k] = Ctri[corner_tri[size_t(i) * 6 + k]];
        double area = 0.0;
        for (int k = 0; k < m; ++k) {
            V3 c0 = C[k], c1 = C[(k + 1) % m];
            V3 n = cross(c0, c1);
            double l = arc(c0, c1);
            V3 nh = (-1.0 / norm(n)) * n;                      // outward for counter-clockwise order
            g.len[size_t(i) * 6 + k] = l;
            g.nrm[size_t(i) * 18 + 3 * k + 0] = nh.x;
            g.nrm[size_t(i) * 18 + 3 * k + 1] = nh.y;
            g.nrm[size_t(i) * 18 + 3 * k + 2] = nh.z;
            ln[k] = l * nh;
            area += tri_area(p0, c0, c1);
        }
        g.area[i] = area;
        // corner k sits on edges k-1 and k: Phi*_k is multiplied by E_k = (l_k-1 n_k-1 + l_k n_k)/2
        for (int k = 0; k < m; ++k) E[k] = 0.5 * (ln[(k + m - 1) % m] + ln[k]);
        V3 w[7];
        for (int j = 0; j < 7; ++j) w[j] = V3{0, 0, 0};
        for (int k = 0; k < m; ++k) {
            int t = corner_tri[size_t(i) * 6 + k];
            int na = nbr[size_t(i) * 6 + k], nb = nbr[size_t(i) * 6 + (k + 1) % m];
            w[0] = w[0] + weight_of(t, i) * E[k];
            w[1 + k] = w[1 + k] + weight_of(t, na) * E[k];
            w[1 + (k + 1) % m] = w[1 + (k + 1) % m] + weight_of(t, nb) * E[k];
        }
        const int d = g.rank[i];
        {   // Laplacian: Eq. 6 applied to the corner gradients, lap_i = sum_k (E_k / A_c) . G_k, kept in
            // difference form (the coefficient of s_i is minus the sum of the others)
            double wl[7] = {0, 0, 0, 0, 0, 0, 0};
            for (int k = 0; k < m; ++k) {
                const int t = corner_tri[size_t(i) * 6 + k];
                const int na = nbr[size_t(i) * 6 + k], nb = nbr[size_t(i) * 6 + (k + 1) % m];
                const V3 Ek = (1.0 / area) * E[k];
                wl[0] += dot(Ek, gw_of(t, i));
                wl[1 + k] += dot(Ek, gw_of(t, na));
                wl[1 + (k + 1) % m] += dot(Ek, gw_of(t, nb));
            }
            for (int j = 0; j < 6; ++j) g.d_wlap[size_t(d) * 6 + j] = wl[1 + j];
        }
        for (int j = 0; j < 7; ++j) {
            V3 wj = (1.0 / area) * w[j];
            g.d_wdiv[size_t(d) * 21 + 3 * j + 0] = wj.x;
            g.d_wdiv[size_t(d) * 21 + 3 * j + 1] = wj.y;
            g.d_wdiv[size_t(d) * 21 + 3 * j + 2] = wj.z;
            if (j >= 1) {
                V3 gj = wj - dot(wj, p0) * p0;                  // Eq. 28 (G5): tangential part
                g.d_wgrad[size_t(d) * 18 + 3 * (j - 1) + 0] = gj.x;
                g.d_wgrad[size_t(d) * 18 + 3 * (j - 1) + 1] = gj.y;
                g.d_wgrad[size_t(d) * 18 + 3 * (j - 1) + 2] = gj.z;
            }
        }
        for (int k = 0; k < 6; ++k) g.d_nbr[size_t(d) * 6 + k] = k < m ? g.rank[nbr[size_t(i) * 6 + k]] : d;
        g.d_rhat[size_t(d) * 3 + 0] = p0.x;
        g.d_rhat[size_t(d) * 3 + 1] = p0.y;
        g.d_rhat[size_t(d) * 3 + 2] = p0.z;
        g.d_area[d] = area;
    }

    // --- lattice neighbours: rotate the slots of every interior lattice point to the fixed direction order and
    // check the arithmetic the kernels use (Morton increments inside the rhombus) against the table
    {
        const unsigned nn = 1u << (2 * level), XM = 0xAAAAAAAAu & (nn - 1), YM = 0x55555555u & (nn - 1);
        bool ok = level >= 2;
        for (int d = 0; ok && d < N; ++d) {
            if (unsigned(d) >= 10u * nn) continue;
            const unsigned r = unsigned(d) >> (2 * level), m = unsigned(d) & (nn - 1), x = m & XM, y = m & YM;
            if (x == 0 || x == XM || y == 0 || y == YM) continue;
            const unsigned xp = ((m | YM) + 1) & XM, xn = ((m & XM) - 1) & XM, yp = ((m | XM) + 1) & YM, yn = ((m & YM) - 1) & YM;
            const unsigned base = r * nn;
            const int want[6] = {int(base + (xp | y)), int(base + (x | yp)), int(base + (xn | yp)),
                                 int(base + (xn | y)), int(base + (x | yn)), int(base + (xp | yn))};
            int* nb = &g.d_nbr[size_t(d) * 6];
            int k0 = -1;
            for (int k = 0; k < 6; ++k)
                if (nb[k] == want[0]) k0 = k;
            if (k0 < 0) { ok = false; break; }
            if (k0 > 0) {
                std::rotate(nb, nb + k0, nb + 6);
                double* wl = &g.d_wlap[size_t(d) * 6];
                std::rotate(wl, wl + k0, wl + 6);
                double* wd = &g.d_wdiv[size_t(d) * 21 + 3];
                std::rotate(wd, wd + 3 * k0, wd + 18);
                double* wg = &g.d_wgrad[size_t(d) * 18];
                std::rotate(wg, wg + 3 * k0, wg + 18);
            }
            for (int k = 0; k < 6; ++k)
                if (nb[k] != want[k]) ok = false;
        }
        g.lattice_nbr = ok;
    }

    // --- tangent basis per column and the stencils contracted with it.  e1 = z x r (x x r next to the
    // poles), e2 = r x e1: no smoothness is needed, the weights absorb the basis of every neighbour.
    g.d_basis.assign(size_t(N) * 6, 0.0);
    g.d_wdiv2.assign(size_t(N) * 14, 0.0);
    g.d_wgrad2.assign(size_t(N) * 12, 0.0);
    for (int d = 0; d < N; ++d) {
        const V3 r{g.d_rhat[size_t(d) * 3], g.d_rhat[size_t(d) * 3 + 1], g.d_rhat[size_t(d) * 3 + 2]};
        const V3 axis = std::fabs(r.z) < 0.9 ? V3{0, 0, 1} : V3{1, 0, 0};
        const V3 e1 = unit(cross(axis, r)), e2 = cross(r, e1);
        double* b = &g.d_basis[size_t(d) * 6];
        b[0] = e1.x; b[1] = e1.y; b[2] = e1.z; b[3] = e2.x; b[4] = e2.y; b[5] = e2.z;
    }
    for (int d = 0; d < N; ++d) {
        auto vec = [](const double* p) { return V3{p[0], p[1], p[2]}; };
        for (int j = 0; j < 7; ++j) {
            const int c = j == 0 ? d : g.d_nbr[size_t(d) * 6 + j - 1];
            const V3 w = vec(&g.d_wdiv[size_t(d) * 21 + 3 * j]);
            g.d_wdiv2[size_t(d) * 14 + 2 * j] = dot(w, vec(&g.d_basis[size_t(c) * 6]));
            g.d_wdiv2[size_t(d) * 14 + 2 * j + 1] = dot(w, vec(&g.d_basis[size_t(c) * 6 + 3]));
        }
        for (int j = 0; j < 6; ++j) {
            const V3 w = vec(&g.d_wgrad[size_t(d) * 18 + 3 * j]);
            g.d_wgrad2[size_t(d) * 12 + 2 * j] = dot(w, vec(&g.d_basis[size_t(d) * 6]));
            g.d_wgrad2[size_t(d) * 12 + 2 * j + 1] = dot(w, vec(&g.d_basis[size_t(d) * 6 + 3]));
        }
    }

    // --- vertical tables (R6: uniform dz unless interface altitudes are given; Eq. 27's radial operator;
    // Eq. 8-9 with k = 1 for the centre -> interface interpolation)
    g.dz = g.P.z_top / nv;
    g.zh.resize(nv + 1);
    for (int k = 0; k <= nv; ++k) g.zh[k] = z_interfaces ? z_interfaces[k] : k * g.dz;
    g.rinv.resize(nv); g.dlo.resize(nv); g.dhi.resize(nv); g.vol.resize(nv); g.zc.resize(nv);
    g.rhinv.resize(nv); g.wl.assign(nv, 0.0); g.wh.assign(nv, 0.0); g.idz.assign(nv, 0.0);
    for (int k = 0; k < nv; ++k) {
        const double zl = g.zh[k], zu = g.zh[k + 1], dzk = z_interfaces ? zu - zl : g.dz;
        const double zc = z_interfaces ? 0.5 * (zl + zu) : (k + 0.5) * g.dz;
        // RS1 (i): in the shallow atmosphere every radius is the planetary radius; altitudes are unchanged
        const double rc = P.radius + (shallow ? 0.0 : zc);
        const double rl = P.radius + (shallow ? 0.0 : zl), ru = P.radius + (shallow ? 0.0 : zu);
        g.zc[k] = zc;
        g.rinv[k] = 1.0 / rc;
        g.dlo[k] = rl * rl / (rc * rc * dzk);
        g.dhi[k] = ru * ru / (rc * rc * dzk);
        g.vol[k] = rc * rc * dzk;
        g.rhinv[k] = 1.0 / rl;
    }
    for (int k = 1; k < nv; ++k) {
        const double dc = g.zc[k] - g.zc[k - 1];
        g.wl[k] = z_interfaces ? (g.zc[k] - g.zh[k]) / dc : 0.5;
        g.wh[k] = z_interfaces ? (g.zh[k] - g.zc[k - 1]) / dc : 0.5;
        g.idz[k] = 1.0 / dc;
    }
    // Eq. 8-9 (L90-L94) at order 3: L_j(zt) = prod_(i != j) (zt - z_i)/(z_j - z_i) over the window of RV1 -- the two
    // nearest nodes on each side of the target, cut at the ends of the column
    g.kord = kord;
    g.shallow = shallow;
    g.ihw.assign(size_t(4) * nv, 0.0);
    g.icw.assign(size_t(4) * nv, 0.0);
    auto lagrange = [](const double* z, int n, double zt, int j) {
        double L = 1.0;
        for (int i = 0; i < n; ++i)
            if (i != j) L = L * (zt - z[i]) / (z[j] - z[i]);
        return L;
    };
    for (int k = 1; k < nv; ++k) {                         // centres lo..hi -> interface k
        const int lo = std::max(k - 2, 0), hi = std::min(k + 1, nv - 1);
        for (int j = lo; j <= hi; ++j) g.ihw[size_t(j - (k - 2)) * nv + k] = lagrange(&g.zc[lo], hi - lo + 1, g.zh[k], j - lo);
    }
    for (int k = 0; k < nv; ++k) {                         // interfaces lo..hi -> centre k
        const int lo = std::max(k - 1, 0), hi = std::min(k + 2, nv);
        for (int j = lo; j <= hi; ++j) g.icw[size_t(j - (k - 1)) * nv + k] = lagrange(&g.zh[lo], hi - lo + 1, g.zc[k], j - lo);
    }
    return THOR_OK;
}

}  // namespace thor
