/*
 * oracle/thor_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU statement of what one THOR HE-VI large time step computes
 * (arXiv 1607.05535; citations are PAPER.md:L<line> + equation; readings R-n and G-n are the ones
 * listed in SURVEY.md 8(c) and restated in DESIGN.md).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or constant with paper_1607_05535_b200/ (the CUDA path),
 * and recomputes every geometric coefficient from the point positions it is given.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/__init__.py).
 * Array-at-a-time, in the paper's order (Fig. 6); no blocking, fusion or reordering.
 * OpenMP only splits independent columns; there are no reductions inside a step, so results do
 * not depend on the thread count.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   geometry/div/grad ........ P2 P4 P5 P6 P7 P8 P9 (closed forms, convergence order, identities)
 *   tridiagonal (orc_substep)  P10 (dense solve of the three discrete fast equations)
 *   step ..................... P11 (mass), P12 (rest state), P13 (Coriolis), P14 (RK order), P15
 *   NEXT-1 (orc_hlap, hyper_diffusion, divergence_damping): Laplacian of a constant, flux form,
 *                              spherical-harmonic eigenvalues, Table 1 timescales (K_d, tau_d), closed forms of
 *                              the fluxes on simple states, mass conservation, rest state, damping acts on
 *                              divergence only; config 2 stays smooth for its 500 steps with the paper's D
 *   NEXT-3 (orc_geom_set_vertical; tests/test_oracle_vertical.py): Eq. 8-9 reproduces polynomials of its degree,
 *                              error order, closed forms of G_h and D_c on unequal layers, rest state and mass on
 *                              stretched layers (k = 1, 3), uniform interfaces = the uniform path, dense solve of the
 *                              fast equations on stretched layers, order k changes the slow terms only (RV2)
 *   NEXT-4 (orc_set_energy_fixer): E restored to round-off where the plain run drifts, rho untouched, one uniform dT
 *   NEXT-4 (orc_geom_set_shallow; tests/test_oracle_shallow.py): layer-independent operators, f r x V closed form,
 *                              solid-body rotation (horizontal curvature term kept, radial one gone), scalar advection
 *                              of w closed form, rest state, mass
 *   total energy (orc_diagnostics): P15, four closed forms (Cv, the 1/2, z_c, r_c, I_c)
 *   PARITY UNPINNED (readings the paper prints nothing for; constrained by the invariants above only): the window
 *   RV1 and the split RV2 of the order-k interpolation, the place and form RE1 of the energy fixer, which terms the
 *   shallow-atmosphere approximation drops (RS1), and, as before,
 *   the discrete advection form R7, the stage convention R1 (pinned in its ORDER by P14, not in value), the forcing
 *   convention R9, and the NEXT-1 readings RD2-RD4 (which state the fluxes use, where F_p enters, the
 *   form of the divergence-damping term; Eq. 43-46 are lost or damaged in PAPER.md) -- the paper fixes
 *   no value for them; only the invariants above constrain them.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    double radius, omega, gravity, Rd, Cp, p_ref, z_top; /* Table 1 (L409-L418), L213, L454 */
} orc_planet;

typedef struct {
    int N, nv;
    orc_planet P;
    double dz;
    double *r_c;  /* [nv]   centre radii     r_k   = A + (k+1/2) dz   (R6: uniform dz, L339, L432) */
    double *r_h;  /* [nv+1] interface radii  r_h,k = A + k dz */
    double *z_c;  /* [nv]   centre altitudes */
    /* NEXT-3 (orc_geom_set_vertical; readings RV1-RV3 of DESIGN.md): layers of unequal thickness and Eq. 8-9 of
     * order kord > 1.  uniform != 0 (the default) is the path above, arithmetic untouched. */
    int uniform, kord;
    /* NEXT-4 (orc_geom_set_shallow; reading RS1 of DESIGN.md): the shallow-atmosphere approximation of L178 */
    int shallow;
    double *z_h;  /* [nv+1] interface altitudes, z_h[0] = 0, z_h[nv] = z_top; the centre is the midpoint of its layer */
    double *xyz;  /* [N][3] unit-sphere positions P_i */
    int *nbr;     /* [N][6] neighbours, counter-clockwise seen from outside; -1 pads pentagons */
    int *deg;     /* [N] 5 or 6 */
    double *C;    /* [N][6][3] control-volume vertices C_k (L61-L63, Fig. 2) */
    double *len;  /* [N][6]    l_k geodesic arc C_k..C_k+1 (L67) */
    double *nrm;  /* [N][6][3] outward unit normal of that arc (L67) */
    double *bary; /* [N][6][3] Eq. 5 weights of (Phi_0, Phi_k, Phi_k+1) at corner k: A2,A3,A1 / sum */
    double *Ac;   /* [N] control-volume area (Eq. 6) */
    /* Eq. 7 on the primary (triangle) grid, for the Laplacian of L369-L371: per corner k the triangle's
     * vertices in canonical order and its three edge vectors l_e n_e/(2 A_T), the centre weights */
    int *tv;      /* [N][6][3]    triangle vertices a, b, c (smallest index first, counter-clockwise) */
    double *tE;   /* [N][6][3][3] E_ab, E_bc, E_ca */
    double *tbw;  /* [N][6][2]    Eq. 5 weights of b and c at the centre C_k */
} orc_geom;

static void cross3(const double *a, const double *b, double *c) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}
static double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static double norm3(const double *a) { return sqrt(dot3(a, a)); }

/* geodesic arc between unit vectors (L67 "geodesic arc length"; G4: atan2(|axb|, a.b)) */
static double arc3(const double *a, const double *b) {
    double c[3];
    cross3(a, b, c);
    return atan2(norm3(c), dot3(a, b));
}

/* area of the spherical triangle a,b,c on the unit sphere (spherical excess) */
static double tri_area(const double *a, const double *b, const double *c) {
    double bc[3];
    cross3(b, c, bc);
    double t = fabs(dot3(a, bc));
    return 2.0 * atan2(t, 1.0 + dot3(a, b) + dot3(b, c) + dot3(c, a));
}

/* Eq. 13 (L122) with reading G4: r_c ~ sum_i (r_i x r_i+1)/|r_i x r_i+1| * arc(r_i, r_i+1),
 * normalised to the unit sphere (the printed 1/2pi prefactor is irrelevant after normalising). */
static void centroid_eq13(const double *r, int n, double *out) {
    double s[3] = {0, 0, 0};
    for (int i = 0; i < n; i++) {
        const double *a = r + 3 * i, *b = r + 3 * ((i + 1) % n);
        double c[3];
        cross3(a, b, c);
        double l = norm3(c);
        double ang = atan2(l, dot3(a, b));
        for (int d = 0; d < 3; d++) s[d] += c[d] / l * ang;
    }
    double l = norm3(s);
    for (int d = 0; d < 3; d++) out[d] = s[d] / l;
}

void orc_geom_free(orc_geom *G) {
    if (!G) return;
    free(G->r_c); free(G->r_h); free(G->z_c); free(G->z_h); free(G->xyz); free(G->nbr); free(G->deg);
    free(G->C); free(G->len); free(G->nrm); free(G->bary); free(G->Ac);
    free(G->tv); free(G->tE); free(G->tbw);
    free(G);
}

/* O2 of SURVEY 8(c): every geometric coefficient from the grid description alone: positions P,
 * neighbour lists and the control-volume vertices C [N][6][3] that L120 leaves fixed while the
 * P_i move to the centroids (reading R4 as revised in DESIGN.md).  Cin == NULL: C_k = Eq. 13
 * centroid of the triangle (P_0, P_k, P_k+1) of the given positions (unmodified grid). */
orc_geom *orc_geom_build(int N, int nv, const orc_planet *P, const double *xyz, const int *nbr,
                         const double *Cin) {
    orc_geom *G = (orc_geom *)calloc(1, sizeof(orc_geom));
    G->N = N; G->nv = nv; G->P = *P;
    G->dz = P->z_top / nv;
    G->r_c = (double *)malloc(sizeof(double) * nv);
    G->z_c = (double *)malloc(sizeof(double) * nv);
    G->r_h = (double *)malloc(sizeof(double) * (nv + 1));
    for (int k = 0; k < nv; k++) { G->z_c[k] = (k + 0.5) * G->dz; G->r_c[k] = P->radius + G->z_c[k]; }
    for (int k = 0; k <= nv; k++) G->r_h[k] = P->radius + k * G->dz;
    G->uniform = 1; G->kord = 1;
    G->z_h = (double *)malloc(sizeof(double) * (nv + 1));
    for (int k = 0; k <= nv; k++) G->z_h[k] = k * G->dz;
    G->xyz = (double *)malloc(sizeof(double) * 3 * N);
    memcpy(G->xyz, xyz, sizeof(double) * 3 * N);
    G->nbr = (int *)malloc(sizeof(int) * 6 * N);
    memcpy(G->nbr, nbr, sizeof(int) * 6 * N);
    G->deg = (int *)malloc(sizeof(int) * N);
    G->C = (double *)calloc((size_t)N * 18, sizeof(double));
    G->len = (double *)calloc((size_t)N * 6, sizeof(double));
    G->nrm = (double *)calloc((size_t)N * 18, sizeof(double));
    G->bary = (double *)calloc((size_t)N * 18, sizeof(double));
    G->Ac = (double *)calloc((size_t)N, sizeof(double));
    G->tv = (int *)calloc((size_t)N * 18, sizeof(int));
    G->tE = (double *)calloc((size_t)N * 54, sizeof(double));
    G->tbw = (double *)calloc((size_t)N * 12, sizeof(double));
    for (int i = 0; i < N; i++) {
        int m = 6;
        if (nbr[6 * i + 5] < 0) m = 5;
        G->deg[i] = m;
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        int m = G->deg[i];
        double *Ci = G->C + 18 * (size_t)i;
        for (int k = 0; k < m; k++) {
            int a = nbr[6 * i + k], b = nbr[6 * i + (k + 1) % m];
            /* canonical rotation (smallest index first, orientation kept) so that the three
             * columns sharing this triangle obtain bit-identical C_k and Eq. 5 weights */
            int v[3] = {i, a, b}, rot = 0;
            if (a < i && a < b) rot = 1;
            if (b < i && b < a) rot = 2;
            int c0 = v[rot], c1 = v[(rot + 1) % 3], c2 = v[(rot + 2) % 3];
            double tri[9];
            memcpy(tri + 0, xyz + 3 * c0, 24);
            memcpy(tri + 3, xyz + 3 * c1, 24);
            memcpy(tri + 6, xyz + 3 * c2, 24);
            double Ck[3];
            if (Cin) memcpy(Ck, Cin + 18 * (size_t)i + 3 * k, 24);
            else centroid_eq13(tri, 3, Ck);
            memcpy(Ci + 3 * k, Ck, 24);
            /* Eq. 5 (L73-L75): each vertex is weighted by the sub-triangle opposite to it */
            double wa[3];
            wa[0] = tri_area(tri + 3, tri + 6, Ck);
            wa[1] = tri_area(tri + 6, tri + 0, Ck);
            wa[2] = tri_area(tri + 0, tri + 3, Ck);
            double ws = wa[0] + wa[1] + wa[2];
            /* (Phi_0, Phi_k, Phi_k+1) = canonical vertices (rot*2)%3 ... undo the rotation */
            double *B = G->bary + 18 * (size_t)i + 3 * k;
            B[0] = wa[(3 - rot) % 3] / ws;       /* A2/sum: weight of P_0   */
            B[1] = wa[(4 - rot) % 3] / ws;       /* A3/sum: weight of P_k   */
            B[2] = wa[(5 - rot) % 3] / ws;       /* A1/sum: weight of P_k+1 */
            /* triangle-grid gradient (Eq. 7 applied to the triangle a, b, c; L369): edge e between two
             * vertices: geodesic arc l_e, outward normal n_e; E_e = l_e n_e / (2 A_T) */
            {
                int *tv = G->tv + 18 * (size_t)i + 3 * k;
                double *tE = G->tE + 54 * (size_t)i + 9 * k, *tbw = G->tbw + 12 * (size_t)i + 2 * k;
                tv[0] = c0; tv[1] = c1; tv[2] = c2;
                double AT = tri_area(tri + 0, tri + 3, tri + 6);
                for (int e = 0; e < 3; e++) {
                    const double *x = tri + 3 * e, *y = tri + 3 * ((e + 1) % 3);
                    double n[3];
                    cross3(x, y, n);
                    double ln = norm3(n), l = arc3(x, y);
                    for (int d = 0; d < 3; d++) tE[3 * e + d] = l * (-n[d] / ln) / (2.0 * AT);
                }
                tbw[0] = wa[1] / ws;
                tbw[1] = wa[2] / ws;
            }
        }
        double area = 0.0;
        for (int k = 0; k < m; k++) {
            const double *c0 = Ci + 3 * k, *c1 = Ci + 3 * ((k + 1) % m);
            G->len[6 * i + k] = arc3(c0, c1);
            double n[3];
            cross3(c0, c1, n);
            double l = norm3(n);
            /* outward for counter-clockwise ordering: -(C_k x C_k+1)/|.| */
            for (int d = 0; d < 3; d++) G->nrm[18 * (size_t)i + 3 * k + d] = -n[d] / l;
            /* control-volume area as a fan of spherical triangles around P_0 */
            area += tri_area(xyz + 3 * i, c0, c1);
        }
        G->Ac[i] = area;
    }
    return G;
}

/* read-only accessors for the tests */
const double *orc_geom_Ac(const orc_geom *G) { return G->Ac; }
const double *orc_geom_len(const orc_geom *G) { return G->len; }
const double *orc_geom_nrm(const orc_geom *G) { return G->nrm; }
const double *orc_geom_C(const orc_geom *G) { return G->C; }
const double *orc_geom_bary(const orc_geom *G) { return G->bary; }
const int *orc_geom_deg(const orc_geom *G) { return G->deg; }

/* Eq. 13 exposed for pin P4 */
void orc_centroid_eq13(const double *r, int n, double *out) { centroid_eq13(r, n, out); }

/* ---------------------------------------------------------------------------------------------
 * Horizontal operators (O2).  vec: [N][nv][3], scalars: [N][nv].  Both return the operator at
 * radius r_k, i.e. the unit-sphere result times 1/r_k (L229, deep atmosphere).
 * ------------------------------------------------------------------------------------------- */

/* Eq. 4-6 (L65-L79): div_0 = (1/A_c) sum_k l_k (Phi*_k + Phi*_k+1)/2 . n_k, Phi* from Eq. 5 */
void orc_hdiv(const orc_geom *G, const double *vec, double *out) {
    const int N = G->N, nv = G->nv;
#pragma omp parallel
    {
        double *phis = (double *)malloc(sizeof(double) * 6 * nv * 3);
#pragma omp for schedule(static)
        for (int i = 0; i < N; i++) {
            int m = G->deg[i];
            const int *nb = G->nbr + 6 * i;
            const double *v0 = vec + (size_t)i * nv * 3;
            for (int k = 0; k < m; k++) {
                const double *B = G->bary + 18 * (size_t)i + 3 * k;
                const double *va = vec + (size_t)nb[k] * nv * 3;
                const double *vb = vec + (size_t)nb[(k + 1) % m] * nv * 3;
                double *ph = phis + (size_t)k * nv * 3;
                for (int q = 0; q < nv * 3; q++) ph[q] = B[0] * v0[q] + B[1] * va[q] + B[2] * vb[q];
            }
            for (int lay = 0; lay < nv; lay++) {
                double sum = 0.0;
                for (int k = 0; k < m; k++) {
                    const double *p0 = phis + ((size_t)k * nv + lay) * 3;
                    const double *p1 = phis + ((size_t)((k + 1) % m) * nv + lay) * 3;
                    const double *n = G->nrm + 18 * (size_t)i + 3 * k;
                    double f = 0.5 * (p0[0] + p1[0]) * n[0] + 0.5 * (p0[1] + p1[1]) * n[1] +
                               0.5 * (p0[2] + p1[2]) * n[2];
                    sum += G->len[6 * i + k] * f;                               /* F_k, Eq. 4 */
                }
                out[(size_t)i * nv + lay] = sum / G->Ac[i] / G->r_c[lay];      /* Eq. 6 */
            }
        }
        free(phis);
    }
}

/* Eq. 7 (L83-L86) in difference form: subtracting s_0 inside the sum IS the correction term,
 * because Eq. 5's weights sum to one.  R5: the radial part is projected out with
 * Eq. 28 as corrected by G5, Phi_h = Phi - (Phi.r)r. */
void orc_hgrad(const orc_geom *G, const double *s, double *out) {
    const int N = G->N, nv = G->nv;
#pragma omp parallel
    {
        double *ds = (double *)malloc(sizeof(double) * 6 * nv);
#pragma omp for schedule(static)
        for (int i = 0; i < N; i++) {
            int m = G->deg[i];
            const int *nb = G->nbr + 6 * i;
            const double *s0 = s + (size_t)i * nv;
            const double *rh = G->xyz + 3 * i;
            for (int k = 0; k < m; k++) {
                const double *B = G->bary + 18 * (size_t)i + 3 * k;
                const double *sa = s + (size_t)nb[k] * nv;
                const double *sb = s + (size_t)nb[(k + 1) % m] * nv;
                for (int lay = 0; lay < nv; lay++)
                    ds[k * nv + lay] = B[1] * (sa[lay] - s0[lay]) + B[2] * (sb[lay] - s0[lay]);
            }
            for (int lay = 0; lay < nv; lay++) {
                double g[3] = {0, 0, 0};
                for (int k = 0; k < m; k++) {
                    double f = G->len[6 * i + k] * 0.5 * (ds[k * nv + lay] + ds[((k + 1) % m) * nv + lay]);
                    const double *n = G->nrm + 18 * (size_t)i + 3 * k;
                    for (int d = 0; d < 3; d++) g[d] += f * n[d];
                }
                double gr = 0.0;
                for (int d = 0; d < 3; d++) { g[d] /= G->Ac[i]; }
                gr = g[0] * rh[0] + g[1] * rh[1] + g[2] * rh[2];
                for (int d = 0; d < 3; d++)
                    out[((size_t)i * nv + lay) * 3 + d] = (g[d] - gr * rh[d]) / G->r_c[lay];
            }
        }
        free(ds);
    }
}

/* Horizontal Laplacian of L369-L371 (NEXT-1 of SURVEY 8(f)): "we first compute the gradient using
 * Eq. (7) in the primary grid (triangles), which place the calculated vectors at the corners of the
 * control volume ... Then using these vectors we apply Eq. 6 to the control volume."
 *   corner k:  G_k = sum_e E_e ((s_e1 - s_m) + (s_e2 - s_m)),  s_m = Eq. 5 value at the centre C_k
 *              (difference form relative to vertex a, so that a constant gives exactly zero and
 *               the three columns sharing the triangle obtain the bit-identical vector)
 *   column:    lap_0 = (1/A_c) sum_k l_k (G_k + G_k+1)/2 . n_k,  times 1/r_k^2 at radius r_k.
 * s, out: [N][nv]. */
static void hlap_unit(const orc_geom *G, const double *s, int nv, double *out) {
    const int N = G->N;
#pragma omp parallel
    {
        double *gk = (double *)malloc(sizeof(double) * 6 * 3);
#pragma omp for schedule(static)
        for (int i = 0; i < N; i++) {
            int m = G->deg[i];
            for (int lay = 0; lay < nv; lay++) {
                for (int k = 0; k < m; k++) {
                    const int *tv = G->tv + 18 * (size_t)i + 3 * k;
                    const double *tE = G->tE + 54 * (size_t)i + 9 * k, *tbw = G->tbw + 12 * (size_t)i + 2 * k;
                    double sa = s[(size_t)tv[0] * nv + lay];
                    double db = s[(size_t)tv[1] * nv + lay] - sa, dc = s[(size_t)tv[2] * nv + lay] - sa;
                    double ma = -(tbw[0] * db + tbw[1] * dc);       /* s_a - s_m */
                    double mb = db + ma, mc = dc + ma;               /* s_b - s_m, s_c - s_m */
                    for (int d = 0; d < 3; d++)
                        gk[3 * k + d] = tE[0 + d] * (ma + mb) + tE[3 + d] * (mb + mc) + tE[6 + d] * (mc + ma);
                }
                double sum = 0.0;
                for (int k = 0; k < m; k++) {
                    const double *g0 = gk + 3 * k, *g1 = gk + 3 * ((k + 1) % m);
                    const double *n = G->nrm + 18 * (size_t)i + 3 * k;
                    double f = 0.5 * (g0[0] + g1[0]) * n[0] + 0.5 * (g0[1] + g1[1]) * n[1] + 0.5 * (g0[2] + g1[2]) * n[2];
                    sum += G->len[6 * i + k] * f;
                }
                out[(size_t)i * nv + lay] = sum / G->Ac[i];
            }
        }
        free(gk);
    }
}
void orc_hlap(const orc_geom *G, const double *s, double *out) {
    const int N = G->N, nv = G->nv;
    hlap_unit(G, s, nv, out);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++)
        for (int k = 0; k < nv; k++) out[(size_t)i * nv + k] = out[(size_t)i * nv + k] / (G->r_c[k] * G->r_c[k]);
}
/* the same operator on interface rows [N][nv+1] at the interface radii r_h,k */
static void hlap_interfaces(const orc_geom *G, const double *s, double *out) {
    const int N = G->N, nv = G->nv;
    hlap_unit(G, s, nv + 1, out);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++)
        for (int k = 0; k <= nv; k++) out[(size_t)i * (nv + 1) + k] = out[(size_t)i * (nv + 1) + k] / (G->r_h[k] * G->r_h[k]);
}

/* Eq. 49-50 (L373-L381): K_d = D dbar^4 / dt, tau_d = dbar^4 / (2^5 K_d); dbar from Eq. 2 (G13). */
double orc_dbar(double radius, int level) { return sqrt(2.0 * 3.14159265358979323846 / 5.0) * radius / pow(2.0, level); }
double orc_kd(double D, double dbar, double dt) { return D * dbar * dbar * dbar * dbar / dt; }
double orc_tau_d(double dbar, double kd) { return dbar * dbar * dbar * dbar / (32.0 * kd); }

/* ---------------------------------------------------------------------------------------------
 * Vertical operators (O3; Eq. 8-9 with k = 1, L88-L94; Eq. 27's radial part, L227).
 * Centre arrays are [nv]; interface arrays are [nv+1] with index 0 = bottom, nv = top.
 * ------------------------------------------------------------------------------------------- */
static double I_h_uniform(const double *Y, int k) { return 0.5 * (Y[k - 1] + Y[k]); }    /* k=1..nv-1 */
static double I_c(const double *X, int k) { return 0.5 * (X[k] + X[k + 1]); }            /* k=0..nv-1 */

/* Eq. 8-9 (L90-L94) written out: sum_j Phi_j L_j(zt), L_j(zt) = prod_(i != j) (zt - z_i)/(z_j - z_i), over the
 * n nodes z[0..n-1] with values Y[0..n-1]. */
static double lagrange(const double *z, const double *Y, int n, double zt) {
    double s = 0.0;
    for (int j = 0; j < n; j++) {
        double L = 1.0;
        for (int i = 0; i < n; i++)
            if (i != j) L = L * (zt - z[i]) / (z[j] - z[i]);
        s = s + Y[j] * L;
    }
    return s;
}
/* RV1: the nodes of Eq. 8-9 at a target between nodes m-1 and m of an array of n_nodes: the (kord+1)/2 nearest
 * nodes on each side; where the column ends first, the missing ones are dropped (the order falls by one per
 * missing node: kord = 3 is quadratic at the first and last interior interface).  kord = 1: the two neighbours. */
static void window(int kord, int m, int n_nodes, int *first, int *count) {
    int half = (kord + 1) / 2;
    int lo = m - half, hi = m + half - 1;
    if (lo < 0) lo = 0;
    if (hi > n_nodes - 1) hi = n_nodes - 1;
    *first = lo; *count = hi - lo + 1;
}
/* centre -> interface k (k = 1..nv-1), linear (Eq. 8-9 with k = 1): what the acoustic system uses (RV2) */
static double I_h(const orc_geom *G, const double *Y, int k) {
    if (G->uniform) return I_h_uniform(Y, k);
    return lagrange(G->z_c + k - 1, Y + k - 1, 2, G->z_h[k]);
}
/* centre -> interface k at the order of the run (RV2: the explicit slow terms) */
static double I_hk(const orc_geom *G, const double *Y, int k) {
    if (G->kord <= 1) return I_h(G, Y, k);
    int f, n;
    window(G->kord, k, G->nv, &f, &n);
    return lagrange(G->z_c + f, Y + f, n, G->z_h[k]);
}
/* interface -> centre k (k = 0..nv-1) at the order of the run: nodes are the interfaces 0..nv (RV2: the
 * vertical momentum at the layer centre, L88); order 1 = the mean of the layer's two interfaces */
static double I_ck(const orc_geom *G, const double *X, int k) {
    if (G->kord <= 1) return I_c(X, k);
    int f, n;
    window(G->kord, k + 1, G->nv + 1, &f, &n);
    return lagrange(G->z_h + f, X + f, n, G->z_c[k]);
}
static double G_h(const orc_geom *G, const double *Y, int k) {                            /* k=1..nv-1 */
    if (G->uniform) return (Y[k] - Y[k - 1]) / G->dz;
    return (Y[k] - Y[k - 1]) / (G->z_c[k] - G->z_c[k - 1]);
}
static double D_c(const orc_geom *G, const double *X, int k) {                            /* k=0..nv-1 */
    const double *rh = G->r_h;
    const double dzk = G->uniform ? G->dz : G->z_h[k + 1] - G->z_h[k];
    return (rh[k + 1] * rh[k + 1] * X[k + 1] - rh[k] * rh[k] * X[k]) / (G->r_c[k] * G->r_c[k] * dzk);
}

/* NEXT-3: layers of unequal thickness (z_h: nv+1 increasing interface altitudes from 0 to z_top, NULL = keep)
 * and the order of Eq. 8-9 (odd, >= 1).  Returns 0, or -1 for a bad argument (nothing changed). */
int orc_geom_set_vertical(orc_geom *G, const double *z_h, int kord) {
    const int nv = G->nv;
    if (kord < 1 || kord % 2 == 0) return -1;
    if (z_h) {
        if (z_h[0] != 0.0) return -1;
        for (int k = 0; k < nv; k++) if (!(z_h[k + 1] > z_h[k])) return -1;
        G->uniform = 0;
        for (int k = 0; k <= nv; k++) { G->z_h[k] = z_h[k]; G->r_h[k] = G->P.radius + z_h[k]; }
        for (int k = 0; k < nv; k++) { G->z_c[k] = 0.5 * (z_h[k] + z_h[k + 1]); G->r_c[k] = G->P.radius + G->z_c[k]; }
        G->P.z_top = z_h[nv];
        G->dz = z_h[nv] / nv;
    }
    G->kord = kord;
    return 0;
}

/* NEXT-4, shallow-atmosphere approximation (L178: "The spherical components of the fluid equations that depend on 1/r
 * are changed to the constant 1/A ... In order to conserve axial angular momentum some metric terms have to be neglected
 * and also the Coriolis terms involved in the horizontal components of planet's angular velocity", the "traditional
 * approximations").  The paper prints no equations for it; reading RS1:
 *   (i)   every radius in the discrete operators is the planetary radius A: r_k = r_h,k = A (horizontal operators / A,
 *         D_c without its r^2 factors, cell volume A_c A^2 dz); altitudes z are unchanged;
 *   (ii)  Coriolis keeps the radial component of Omega only: C = 2 Omega sin(lat) r x V, on the horizontal momentum
 *         alone; W neither feels nor causes a Coriolis force;
 *   (iii) the metric terms that couple horizontal and vertical motion are dropped: the horizontal momentum equation
 *         advects the horizontal velocity u_h = V/rho only (no rho v_h v_r / r term), and the vertical momentum equation
 *         advects w = I_c[W]/rho as a scalar (no -rho |v_h|^2 / r term).  The curvature terms of the horizontal flow on
 *         the sphere of radius A (u v tan(lat)/A ...) stay: they are what the Cartesian form of Eq. 28 produces.
 * on = 0 restores the deep atmosphere. */
void orc_geom_set_shallow(orc_geom *G, int on) {
    G->shallow = on ? 1 : 0;
    for (int k = 0; k < G->nv; k++) G->r_c[k] = G->P.radius + (on ? 0.0 : G->z_c[k]);
    for (int k = 0; k <= G->nv; k++) G->r_h[k] = G->P.radius + (on ? 0.0 : G->z_h[k]);
}

/* Eq. 24 (L210) and its inverse */
static double eos_p(const orc_planet *P, double rt) {
    double gam = P->Cp / (P->Cp - P->Rd);
    return P->p_ref * pow(P->Rd * rt / P->p_ref, gam);
}
static double eos_rt(const orc_planet *P, double p) {
    double gam = P->Cp / (P->Cp - P->Rd);
    return P->p_ref / P->Rd * pow(p / P->p_ref, 1.0 / gam);
}

/* Thomas algorithm (L339) for a_k x_k-1 + b_k x_k + c_k x_k+1 = d_k, k = 1..n; arrays are
 * indexed 1..n (index 0 unused); a_1 and c_n multiply the zero boundary values (rigid lid). */
void orc_thomas(int n, const double *a, const double *b, const double *c, const double *d, double *x) {
    double *cp = (double *)malloc(sizeof(double) * (n + 2));
    double *dp = (double *)malloc(sizeof(double) * (n + 2));
    cp[1] = c[1] / b[1];
    dp[1] = d[1] / b[1];
    for (int k = 2; k <= n; k++) {
        double den = b[k] - a[k] * cp[k - 1];
        cp[k] = c[k] / den;
        dp[k] = (d[k] - a[k] * dp[k - 1]) / den;
    }
    x[n] = dp[n];
    for (int k = n - 1; k >= 1; k--) x[k] = dp[k] - cp[k] * x[k + 1];
    free(cp); free(dp);
}

/* ---------------------------------------------------------------------------------------------
 * Work space of one large step
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    size_t nc, ni;                      /* N*nv, N*(nv+1) */
    /* Phi^n */
    double *rho_n, *V_n, *W_n, *p_n, *rt_n;
    /* reference state of the stage, Phi^[t] */
    double *rho_t, *V_t, *W_t, *p_t;
    /* a1: stage coefficients */
    double *h, *th, *gt;                /* gt: [N][nv+1], interior interfaces only */
    /* a2: slow terms */
    double *slowV, *slowrho, *Svr, *slowp, *slowrt;
    /* deviations */
    double *rho_s, *V_s, *W_s, *p_s, *rt;
    /* scratch */
    double *vec, *sc1, *sc2, *sc3, *gradp, *u, *Avec, *Wc;
    /* NEXT-1 (Eq. 43-50): diffusion coefficients K_d (0 = term off), scratch, divergence-damping flux */
    double Kd_hyp, Kd_div;
    double *di1, *di2, *di3, *Fdd;     /* di*: [N][nv+1]; Fdd: [N][nv][3] */
} orc_work;

static double *dalloc(size_t n) { return (double *)calloc(n, sizeof(double)); }

static orc_work *work_new(const orc_geom *G) {
    orc_work *w = (orc_work *)calloc(1, sizeof(orc_work));
    size_t nc = (size_t)G->N * G->nv, ni = (size_t)G->N * (G->nv + 1);
    w->nc = nc; w->ni = ni;
    w->rho_n = dalloc(nc); w->V_n = dalloc(3 * nc); w->W_n = dalloc(ni); w->p_n = dalloc(nc); w->rt_n = dalloc(nc);
    w->rho_t = dalloc(nc); w->V_t = dalloc(3 * nc); w->W_t = dalloc(ni); w->p_t = dalloc(nc);
    w->h = dalloc(nc); w->th = dalloc(nc); w->gt = dalloc(ni);
    w->slowV = dalloc(3 * nc); w->slowrho = dalloc(nc); w->Svr = dalloc(ni); w->slowp = dalloc(nc); w->slowrt = dalloc(nc);
    w->rho_s = dalloc(nc); w->V_s = dalloc(3 * nc); w->W_s = dalloc(ni); w->p_s = dalloc(nc); w->rt = dalloc(nc);
    w->vec = dalloc(3 * nc); w->sc1 = dalloc(nc); w->sc2 = dalloc(nc); w->sc3 = dalloc(nc);
    w->gradp = dalloc(3 * nc); w->u = dalloc(3 * nc); w->Avec = dalloc(3 * nc); w->Wc = dalloc(nc);
    w->di1 = dalloc(ni); w->di2 = dalloc(ni); w->di3 = dalloc(ni); w->Fdd = dalloc(3 * nc);
    return w;
}
static void work_free(orc_work *w) {
    double **p[] = {&w->rho_n, &w->V_n, &w->W_n, &w->p_n, &w->rt_n, &w->rho_t, &w->V_t, &w->W_t, &w->p_t,
                    &w->h, &w->th, &w->gt, &w->slowV, &w->slowrho, &w->Svr, &w->slowp, &w->slowrt,
                    &w->rho_s, &w->V_s, &w->W_s, &w->p_s, &w->rt, &w->vec, &w->sc1, &w->sc2, &w->sc3,
                    &w->gradp, &w->u, &w->Avec, &w->Wc, &w->di1, &w->di2, &w->di3, &w->Fdd};
    for (size_t i = 0; i < sizeof(p) / sizeof(p[0]); i++) free(*p[i]);
    free(w);
}

/* a1 (Eq. 38-39; Fig. 6 large-step 1): h = Cp T = Cp p/(Rd rho) (G9),
 * theta = (rho theta)/rho with rho theta from Eq. 24 inverted, g~ = G_h[p]/I_h[rho] at interfaces */
static void stage_coefficients(const orc_geom *G, orc_work *w) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double *rho = w->rho_t + (size_t)i * nv, *p = w->p_t + (size_t)i * nv;
        double *h = w->h + (size_t)i * nv, *th = w->th + (size_t)i * nv, *gt = w->gt + (size_t)i * (nv + 1);
        for (int k = 0; k < nv; k++) {
            h[k] = P->Cp * p[k] / (P->Rd * rho[k]);
            th[k] = eos_rt(P, p[k]) / rho[k];
        }
        gt[0] = 0.0; gt[nv] = 0.0;
        for (int k = 1; k < nv; k++) gt[k] = G_h(G, p, k) / I_h(G, rho, k);
    }
}

/* a2 (RHS of Eq. 32-35, Eq. 40-42; L258-L299, L268; O4 with reading R7) */
static void slow_terms(const orc_geom *G, orc_work *w) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
    const double kv = P->Rd / (P->Cp - P->Rd);
    const size_t nc = w->nc;

    /* full Cartesian momentum M = V + I_c[W] r, velocity u = M/rho (L268 "non-projected") */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double *rh = G->xyz + 3 * i;
        const double *W = w->W_t + (size_t)i * (nv + 1);
        for (int k = 0; k < nv; k++) {
            size_t c = (size_t)i * nv + k;
            double wc = I_ck(G, W, k);
            w->Wc[c] = wc;
            if (G->shallow)                                   /* RS1 (iii): the horizontal velocity alone is advected */
                for (int d = 0; d < 3; d++) w->u[3 * c + d] = w->V_t[3 * c + d] / w->rho_t[c];
            else
                for (int d = 0; d < 3; d++) w->u[3 * c + d] = (w->V_t[3 * c + d] + wc * rh[d]) / w->rho_t[c];
        }
    }

    /* advection A_j = div_h(V u_j) + D_c[W I_h[u_j]] for each Cartesian component j (Eq. 21, 27) */
    for (int j = 0; j < 3; j++) {
#pragma omp parallel for schedule(static)
        for (size_t c = 0; c < nc; c++)
            for (int d = 0; d < 3; d++) w->vec[3 * c + d] = w->V_t[3 * c + d] * w->u[3 * c + j];
        orc_hdiv(G, w->vec, w->sc1);
#pragma omp parallel
        {
            double *X = (double *)calloc(nv + 1, sizeof(double));
            double *uj = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
            for (int i = 0; i < N; i++) {
                const double *W = w->W_t + (size_t)i * (nv + 1);
                for (int k = 0; k < nv; k++) uj[k] = w->u[3 * ((size_t)i * nv + k) + j];
                X[0] = 0.0; X[nv] = 0.0;
                for (int k = 1; k < nv; k++) X[k] = W[k] * I_hk(G, uj, k);
                for (int k = 0; k < nv; k++) {
                    size_t c = (size_t)i * nv + k;
                    w->Avec[3 * c + j] = w->sc1[c] + D_c(G, X, k);
                }
            }
            free(X); free(uj);
        }
    }

    /* RS1 (iii): w = I_c[W]/rho advected as a scalar, A_w = div_h(V w) + D_c[W I_h[w]]  (scratch: di3, free here) */
    double *Aw = w->di3;
    if (G->shallow) {
#pragma omp parallel for schedule(static)
        for (size_t c = 0; c < nc; c++) {
            double wv = w->Wc[c] / w->rho_t[c];
            for (int d = 0; d < 3; d++) w->vec[3 * c + d] = w->V_t[3 * c + d] * wv;
        }
        orc_hdiv(G, w->vec, w->sc1);
#pragma omp parallel
        {
            double *X = (double *)calloc(nv + 1, sizeof(double));
            double *wv = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
            for (int i = 0; i < N; i++) {
                const double *W = w->W_t + (size_t)i * (nv + 1);
                for (int k = 0; k < nv; k++) wv[k] = w->Wc[(size_t)i * nv + k] / w->rho_t[(size_t)i * nv + k];
                X[0] = 0.0; X[nv] = 0.0;
                for (int k = 1; k < nv; k++) X[k] = W[k] * I_hk(G, wv, k);
                for (int k = 0; k < nv; k++) Aw[(size_t)i * nv + k] = w->sc1[(size_t)i * nv + k] + D_c(G, X, k);
            }
            free(X); free(wv);
        }
    }

    /* grad_h p^[t] */
    orc_hgrad(G, w->p_t, w->gradp);
    /* div_h V, div_h (h V), div_h (theta V) */
    orc_hdiv(G, w->V_t, w->sc1);
#pragma omp parallel for schedule(static)
    for (size_t c = 0; c < nc; c++)
        for (int d = 0; d < 3; d++) w->vec[3 * c + d] = w->h[c] * w->V_t[3 * c + d];
    orc_hdiv(G, w->vec, w->sc2);
#pragma omp parallel for schedule(static)
    for (size_t c = 0; c < nc; c++)
        for (int d = 0; d < 3; d++) w->vec[3 * c + d] = w->th[c] * w->V_t[3 * c + d];
    orc_hdiv(G, w->vec, w->sc3);

#pragma omp parallel
    {
        double *X = (double *)calloc(nv + 1, sizeof(double));
        double *Fr = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
        for (int i = 0; i < N; i++) {
            const double *rh = G->xyz + 3 * i;
            const double *W = w->W_t + (size_t)i * (nv + 1);
            const double *rho = w->rho_t + (size_t)i * nv, *p = w->p_t + (size_t)i * nv;
            const double *h = w->h + (size_t)i * nv, *th = w->th + (size_t)i * nv;
            const double *gt = w->gt + (size_t)i * (nv + 1);
            double *Svr = w->Svr + (size_t)i * (nv + 1);
            for (int k = 0; k < nv; k++) {
                size_t c = (size_t)i * nv + k;
                const double *A = w->Avec + 3 * c;
                /* Coriolis C = 2 Omega z x M (Eq. 21), rotation axis through the polar vertices */
                double M[3], Cor[3];
                for (int d = 0; d < 3; d++) M[d] = w->V_t[3 * c + d] + w->Wc[c] * rh[d];
                if (G->shallow) {                     /* RS1 (ii): f r x V, f = 2 Omega sin(lat), sin(lat) = z of r */
                    const double f = 2.0 * P->omega * rh[2];
                    const double *V = w->V_t + 3 * c;
                    Cor[0] = f * (rh[1] * V[2] - rh[2] * V[1]);
                    Cor[1] = f * (rh[2] * V[0] - rh[0] * V[2]);
                    Cor[2] = f * (rh[0] * V[1] - rh[1] * V[0]);
                } else {
                    Cor[0] = -2.0 * P->omega * M[1];
                    Cor[1] = 2.0 * P->omega * M[0];
                    Cor[2] = 0.0;
                }
                double Ar = dot3(A, rh), Cr = dot3(Cor, rh);                   /* Eq. 29 */
                Fr[k] = G->shallow ? Aw[c] : Ar + Cr;                          /* RS1 (iii) */
                for (int d = 0; d < 3; d++) {                                   /* Eq. 28 (G5) */
                    double Ah = A[d] - Ar * rh[d], Ch = Cor[d] - Cr * rh[d];
                    w->slowV[3 * c + d] = -w->gradp[3 * c + d] - Ah - Ch;       /* RHS of Eq. 33 */
                }
            }
            /* RHS of Eq. 32 */
            for (int k = 0; k < nv; k++) w->slowrho[(size_t)i * nv + k] = -w->sc1[(size_t)i * nv + k] - D_c(G, W, k);
            /* Eq. 42 at interior interfaces */
            Svr[0] = 0.0; Svr[nv] = 0.0;
            for (int k = 1; k < nv; k++) Svr[k] = -G_h(G, p, k) - P->gravity * I_hk(G, rho, k) - I_hk(G, Fr, k);
            /* slow part of the pressure equation (Eq. 40 with the signs of G10) */
            X[0] = 0.0; X[nv] = 0.0;
            for (int k = 1; k < nv; k++) X[k] = I_hk(G, h, k) * W[k];
            for (int k = 0; k < nv; k++) {
                size_t c = (size_t)i * nv + k;
                double vgp = 0.0;
                for (int d = 0; d < 3; d++) vgp += w->V_t[3 * c + d] / rho[k] * w->gradp[3 * c + d];
                double gW = 0.5 * (gt[k] * W[k] + gt[k + 1] * W[k + 1]);        /* I_c[g~ W] */
                w->slowp[c] = -kv * (w->sc2[c] + D_c(G, X, k) - vgp - gW);
            }
            /* slow part of Eq. 35 (G7: with the r^2 factors of Eq. 27) */
            for (int k = 1; k < nv; k++) X[k] = I_hk(G, th, k) * W[k];
            for (int k = 0; k < nv; k++) {
                size_t c = (size_t)i * nv + k;
                w->slowrt[c] = -w->sc3[c] - D_c(G, X, k);
            }
        }
        free(X); free(Fr);
    }
}

/* ---------------------------------------------------------------------------------------------
 * NEXT-1: explicit fourth-order hyper-diffusion and 3-D divergence damping (section 4;
 * Eq. 43-48, of which 43-44 are lost and 45-46 damaged in PAPER.md -- readings RD1-RD5 of DESIGN.md).
 * Every nabla_h^2 is orc_hlap's operator (L369-L371).  K_d = D dbar^4 / dt (Eq. 49).
 * ------------------------------------------------------------------------------------------- */

/* RD2 (Fig. 6 large-step 2, L307: "Compute diffuse fluxes" inside the three-stage loop): fluxes of the
 * stage reference state, added to the slow terms of the stage:
 *   F_rho = -K_d lap(lap(rho))                                   (Eq. 43 by the pattern of Eq. 47)
 *   F_vhj = -K_d lap(rho lap(v_j)), v = V/rho, j = x, y, z, then Eq. 28   (Eq. 44-46, first term)
 *   F_vr  = -K_d lap(rho_h lap(w)) on interfaces, w = W/I_h[rho]          (Eq. 47)
 *   F_p   = -Rd K_d lap(rho lap(T)), T = p/(Rd rho)                        (Eq. 48)
 * RD3: F_p enters the slow pressure term and, because the substeps carry rho*theta (Eq. 35) and
 * diagnose p from it (Eq. 36), the slow rho*theta term through Eq. 24: d(rho theta) = (rho theta)/(gamma p) dp. */
static void hyper_diffusion(const orc_geom *G, orc_work *w) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
    const size_t nc = w->nc, ni = w->ni;
    const double Kd = w->Kd_hyp, gam = P->Cp / (P->Cp - P->Rd);
    double *a = w->di1, *b = w->di2, *c = w->di3;
    /* density */
    orc_hlap(G, w->rho_t, a);
    orc_hlap(G, a, b);
#pragma omp parallel for schedule(static)
    for (size_t q = 0; q < nc; q++) w->slowrho[q] = w->slowrho[q] + (-Kd * b[q]);
    /* horizontal momentum, one Cartesian component at a time */
    for (int j = 0; j < 3; j++) {
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < nc; q++) a[q] = w->V_t[3 * q + j] / w->rho_t[q];
        orc_hlap(G, a, b);
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < nc; q++) b[q] = w->rho_t[q] * b[q];
        orc_hlap(G, b, c);
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < nc; q++) w->Avec[3 * q + j] = -Kd * c[q];
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double *rh = G->xyz + 3 * i;
        for (int k = 0; k < nv; k++) {
            size_t q = (size_t)i * nv + k;
            double Fr = dot3(w->Avec + 3 * q, rh);
            for (int d = 0; d < 3; d++) w->slowV[3 * q + d] = w->slowV[3 * q + d] + (w->Avec[3 * q + d] - Fr * rh[d]);
        }
    }
    /* vertical momentum on interior interfaces */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double *rho = w->rho_t + (size_t)i * nv, *W = w->W_t + (size_t)i * (nv + 1);
        double *wv = a + (size_t)i * (nv + 1);
        wv[0] = 0.0; wv[nv] = 0.0;
        for (int k = 1; k < nv; k++) wv[k] = W[k] / I_hk(G, rho, k);
    }
    hlap_interfaces(G, a, b);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double *rho = w->rho_t + (size_t)i * nv;
        double *x = b + (size_t)i * (nv + 1);
        x[0] = 0.0; x[nv] = 0.0;
        for (int k = 1; k < nv; k++) x[k] = I_hk(G, rho, k) * x[k];
    }
    hlap_interfaces(G, b, c);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++)
        for (int k = 1; k < nv; k++) {
            size_t q = (size_t)i * (nv + 1) + k;
            w->Svr[q] = w->Svr[q] + (-Kd * c[q]);
        }
    (void)ni;
    /* pressure through temperature */
#pragma omp parallel for schedule(static)
    for (size_t q = 0; q < nc; q++) a[q] = w->p_t[q] / (P->Rd * w->rho_t[q]);
    orc_hlap(G, a, b);
#pragma omp parallel for schedule(static)
    for (size_t q = 0; q < nc; q++) b[q] = w->rho_t[q] * b[q];
    orc_hlap(G, b, c);
#pragma omp parallel for schedule(static)
    for (size_t q = 0; q < nc; q++) {
        double Fp = -P->Rd * Kd * c[q];
        w->slowp[q] = w->slowp[q] + Fp;
        w->slowrt[q] = w->slowrt[q] + Fp * eos_rt(P, w->p_t[q]) / (gam * w->p_t[q]);
    }
}

/* RD4 (Eq. 44-46 second term; Fig. 6 small-step 1, L318; "updated every short time step", L367):
 *   D3 = div_h(V) + D_c[W] of the CURRENT momentum V = V^[t] + V*, W = W^[t] + W*;
 *   F_dd = -K_d lap(grad_h D3), the Laplacian applied to each Cartesian component, then Eq. 28;
 * it enters the explicit horizontal momentum step (Eq. 33) only (Eq. 47 carries no such term). */
static void divergence_damping(const orc_geom *G, orc_work *w) {
    const int N = G->N, nv = G->nv;
    const size_t nc = w->nc;
    double *a = w->di1, *b = w->di2;
#pragma omp parallel for schedule(static)
    for (size_t q = 0; q < 3 * nc; q++) w->vec[q] = w->V_t[q] + w->V_s[q];
    orc_hdiv(G, w->vec, w->sc1);
#pragma omp parallel
    {
        double *X = (double *)calloc(nv + 1, sizeof(double));
#pragma omp for schedule(static)
        for (int i = 0; i < N; i++) {
            const double *Wt = w->W_t + (size_t)i * (nv + 1), *Ws = w->W_s + (size_t)i * (nv + 1);
            for (int k = 0; k <= nv; k++) X[k] = Wt[k] + Ws[k];
            for (int k = 0; k < nv; k++) w->sc1[(size_t)i * nv + k] = w->sc1[(size_t)i * nv + k] + D_c(G, X, k);
        }
        free(X);
    }
    orc_hgrad(G, w->sc1, w->gradp);                 /* gradp is free here: Eq. 33 recomputes it afterwards */
    for (int j = 0; j < 3; j++) {
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < nc; q++) a[q] = w->gradp[3 * q + j];
        orc_hlap(G, a, b);
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < nc; q++) w->Fdd[3 * q + j] = -w->Kd_div * b[q];
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double *rh = G->xyz + 3 * i;
        for (int k = 0; k < nv; k++) {
            size_t q = (size_t)i * nv + k;
            double Fr = dot3(w->Fdd + 3 * q, rh);
            for (int d = 0; d < 3; d++) w->Fdd[3 * q + d] = w->Fdd[3 * q + d] - Fr * rh[d];
        }
    }
}

/* Tridiagonal coefficients of O6 item 3 for one column at interior interfaces k = 1..nv-1
 * (exact elimination of Eq. 32, the linearised pressure equation and Eq. 34; reading R8). */
static void tridiag_coefficients(const orc_geom *G, double delta, const double *h, const double *gt,
                                 double *a, double *b, double *c) {
    const int nv = G->nv;
    const orc_planet *P = &G->P;
    const double kv = P->Rd / (P->Cp - P->Rd), dz = G->dz, g = P->gravity;
    const double *rc = G->r_c, *rh = G->r_h;
    const double d2 = delta * delta;
    if (!G->uniform) {
        /* the same elimination with layers of unequal thickness: t_k = z_h,k+1 - z_h,k (layer), s_k = z_k - z_k-1
         * (centre spacing of G_h), I_h[Y]_k = wl Y_k-1 + wu Y_k (Eq. 8-9, k = 1) */
        const double *zh = G->z_h, *zc = G->z_c;
        for (int k = 1; k < nv; k++) {
            double hk = I_h(G, h, k);
            double hkp = (k + 1 < nv) ? I_h(G, h, k + 1) : 0.0;
            double hkm = (k - 1 > 0) ? I_h(G, h, k - 1) : 0.0;
            double rk2 = rc[k] * rc[k], rkm2 = rc[k - 1] * rc[k - 1];
            double tk = zh[k + 1] - zh[k], tkm = zh[k] - zh[k - 1], sk = zc[k] - zc[k - 1];
            double wl = (zc[k] - zh[k]) / sk, wu = (zh[k] - zc[k - 1]) / sk;
            c[k] = -(d2 * kv / sk) * (rh[k + 1] * rh[k + 1] * hkp / (rk2 * tk) - gt[k + 1] / 2.0)
                   - d2 * g * wu * rh[k + 1] * rh[k + 1] / (rk2 * tk);
            a[k] = -(d2 * kv / sk) * (rh[k - 1] * rh[k - 1] * hkm / (rkm2 * tkm) + gt[k - 1] / 2.0)
                   + d2 * g * wl * rh[k - 1] * rh[k - 1] / (rkm2 * tkm);
            b[k] = 1.0 + (d2 * kv / sk) * rh[k] * rh[k] * hk * (1.0 / (rk2 * tk) + 1.0 / (rkm2 * tkm))
                   - d2 * g * rh[k] * rh[k] * (wl / (rkm2 * tkm) - wu / (rk2 * tk));
        }
        return;
    }
    for (int k = 1; k < nv; k++) {
        double hk = I_h(G, h, k);
        double hkp = (k + 1 < nv) ? I_h(G, h, k + 1) : 0.0;   /* multiplies W_nv = 0 */
        double hkm = (k - 1 > 0) ? I_h(G, h, k - 1) : 0.0;    /* multiplies W_0  = 0 */
        double rk2 = rc[k] * rc[k], rkm2 = rc[k - 1] * rc[k - 1];
        c[k] = -(d2 * kv / dz) * (rh[k + 1] * rh[k + 1] * hkp / (rk2 * dz) - gt[k + 1] / 2.0)
               - (d2 * g / (2.0 * dz)) * rh[k + 1] * rh[k + 1] / rk2;
        a[k] = -(d2 * kv / dz) * (rh[k - 1] * rh[k - 1] * hkm / (rkm2 * dz) + gt[k - 1] / 2.0)
               + (d2 * g / (2.0 * dz)) * rh[k - 1] * rh[k - 1] / rkm2;
        b[k] = 1.0 + (d2 * kv / (dz * dz)) * rh[k] * rh[k] * hk * (1.0 / rk2 + 1.0 / rkm2)
               - (d2 * g / (2.0 * dz)) * rh[k] * rh[k] * (1.0 / rkm2 - 1.0 / rk2);
    }
}

/* a4-a9: one acoustic substep (O6; Eq. 33, 37, 32, 35, 36; Fig. 6 small-step 2-6, L318-L329) */
static void substep(const orc_geom *G, orc_work *w, double delta) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
    const double kv = P->Rd / (P->Cp - P->Rd), g = P->gravity;
    const size_t nc = w->nc;

    /* Fig. 6 small-step 1 (NEXT-1, only when K_d > 0) */
    if (w->Kd_div > 0.0) divergence_damping(G, w);
    /* a4: Eq. 33 */
    orc_hgrad(G, w->p_s, w->gradp);
    if (w->Kd_div > 0.0) {
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < 3 * nc; q++) w->V_s[q] = w->V_s[q] + delta * (-w->gradp[q] + w->slowV[q] + w->Fdd[q]);
    } else {
#pragma omp parallel for schedule(static)
        for (size_t q = 0; q < 3 * nc; q++) w->V_s[q] = w->V_s[q] + delta * (-w->gradp[q] + w->slowV[q]);
    }

    /* a5: divergences of the new momentum */
    orc_hdiv(G, w->V_s, w->sc1);
#pragma omp parallel for schedule(static)
    for (size_t c = 0; c < nc; c++)
        for (int d = 0; d < 3; d++) w->vec[3 * c + d] = w->h[c] * w->V_s[3 * c + d];
    orc_hdiv(G, w->vec, w->sc2);
#pragma omp parallel for schedule(static)
    for (size_t c = 0; c < nc; c++)
        for (int d = 0; d < 3; d++) w->vec[3 * c + d] = w->th[c] * w->V_s[3 * c + d];
    orc_hdiv(G, w->vec, w->sc3);

#pragma omp parallel
    {
        double *a = (double *)calloc(nv + 1, sizeof(double)), *b = (double *)calloc(nv + 1, sizeof(double));
        double *c = (double *)calloc(nv + 1, sizeof(double)), *d = (double *)calloc(nv + 1, sizeof(double));
        double *Wn = (double *)calloc(nv + 1, sizeof(double)), *X = (double *)calloc(nv + 1, sizeof(double));
        double *Srho = (double *)malloc(sizeof(double) * nv), *Sp = (double *)malloc(sizeof(double) * nv);
        double *pq = (double *)malloc(sizeof(double) * nv), *rq = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
        for (int i = 0; i < N; i++) {
            size_t c0 = (size_t)i * nv;
            const double *h = w->h + c0, *th = w->th + c0, *gt = w->gt + (size_t)i * (nv + 1);
            double *Ws = w->W_s + (size_t)i * (nv + 1);
            const double *Svr = w->Svr + (size_t)i * (nv + 1);
            for (int k = 0; k < nv; k++) {
                Srho[k] = w->slowrho[c0 + k] - w->sc1[c0 + k];                 /* Eq. 41 */
                Sp[k] = w->slowp[c0 + k] - kv * w->sc2[c0 + k];                /* Eq. 40 (G10) */
                pq[k] = w->p_s[c0 + k] + delta * Sp[k];
                rq[k] = w->rho_s[c0 + k] + delta * Srho[k];
            }
            /* a6: assemble and solve (Eq. 37 as defined by elimination, R8; L339) */
            tridiag_coefficients(G, delta, h, gt, a, b, c);
            for (int k = 1; k < nv; k++)
                d[k] = Ws[k] + delta * Svr[k] - delta * G_h(G, pq, k) - delta * g * I_h(G, rq, k);
            Wn[0] = 0.0; Wn[nv] = 0.0;
            if (nv > 1) orc_thomas(nv - 1, a, b, c, d, Wn);
            /* a7: Eq. 32 with the new momenta (L341) */
            for (int k = 0; k < nv; k++) w->rho_s[c0 + k] = w->rho_s[c0 + k] + delta * (Srho[k] - D_c(G, Wn, k));
            /* a8: Eq. 35 (G7) */
            X[0] = 0.0; X[nv] = 0.0;
            for (int k = 1; k < nv; k++) X[k] = I_h(G, th, k) * Wn[k];
            for (int k = 0; k < nv; k++)
                w->rt[c0 + k] = w->rt[c0 + k] + delta * (w->slowrt[c0 + k] - w->sc3[c0 + k] - D_c(G, X, k));
            /* a9: Eq. 36 */
            for (int k = 0; k < nv; k++) w->p_s[c0 + k] = eos_p(P, w->rt[c0 + k]) - w->p_t[c0 + k];
            for (int k = 0; k <= nv; k++) Ws[k] = Wn[k];
        }
        free(a); free(b); free(c); free(d); free(Wn); free(X); free(Srho); free(Sp); free(pq); free(rq);
    }
}

/* a11: Eq. 51-52 backward Euler with the large step (L385-L399; R9).  Tables are [N][nv]; NULL = off */
static void forcing(const orc_geom *G, double dt, double *rho, double *V, double *p,
                    const double *T_eq, const double *k_T, const double *k_v) {
    const size_t nc = (size_t)G->N * G->nv;
    const double Rd = G->P.Rd;
#pragma omp parallel for schedule(static)
    for (size_t c = 0; c < nc; c++) {
        if (k_v)
            for (int d = 0; d < 3; d++) V[3 * c + d] = V[3 * c + d] / (1.0 + k_v[c] * dt);      /* Eq. 51 */
        if (k_T && T_eq) {
            double T = p[c] / (rho[c] * Rd);                                                    /* Eq. 25 */
            T = (T + k_T[c] * dt * T_eq[c]) / (1.0 + k_T[c] * dt);                              /* Eq. 52 */
            p[c] = rho[c] * Rd * T;
        }
    }
}

/* NEXT-2: the Held-Suarez forcing of section 7.1 with K_v, K_T, T_eq from the EVOLVING
 * state (Eq. 51-55): sigma = p / p_s, the surface pressure "estimated extrapolating the
 * pressures to the surface using the hydrostatic equation and keeping the temperature constant in that
 * region" (L390): p_s = p_0 exp(g z_0 / (Rd T_0)) from the lowest layer centre.
 *   K_v  = k_f max(0, (sigma - sigma_b)/(1 - sigma_b))                                    (Eq. 53)
 *   T_eq = max{T_min, [T_surf - dT_y sin^2(phi) - dth_z ln(p/p*) cos^2(phi)] (p/p*)^(Rd/Cp)}  (Eq. 54, G14)
 *   K_T  = k_a + (k_s - k_a) max(0, (sigma - sigma_b)/(1 - sigma_b)) cos^4(phi)              (Eq. 55, G14)
 * then Eq. 51-52 as in forcing() (R9: rho unchanged, p = rho Rd T).  phi: latitude, sin(phi) = z of the
 * column's unit vector (rotation axis through the polar vertices, L45). */
typedef struct { double T_surf, dT_y, dth_z, T_min, k_a, k_s, k_f, sigma_b, p_star; } orc_held_suarez;

static void forcing_held_suarez(const orc_geom *G, double dt, double *rho, double *V, double *p, const orc_held_suarez *H) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
    const double kappa = P->Rd / P->Cp;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double sphi = G->xyz[3 * i + 2], cphi2 = 1.0 - sphi * sphi;
        size_t c0 = (size_t)i * nv;
        const double T0 = p[c0] / (rho[c0] * P->Rd);
        const double ps = p[c0] * exp(P->gravity * G->z_c[0] / (P->Rd * T0));                   /* L390 */
        for (int k = 0; k < nv; k++) {
            size_t c = c0 + k;
            const double sigma = p[c] / ps;
            double ramp = (sigma - H->sigma_b) / (1.0 - H->sigma_b);
            if (ramp < 0.0) ramp = 0.0;
            const double Kv = H->k_f * ramp;                                                     /* Eq. 53 */
            const double pr = p[c] / H->p_star;
            double Teq = (H->T_surf - H->dT_y * sphi * sphi - H->dth_z * log(pr) * cphi2) * pow(pr, kappa);
            if (Teq < H->T_min) Teq = H->T_min;                                                  /* Eq. 54 */
            const double KT = H->k_a + (H->k_s - H->k_a) * ramp * cphi2 * cphi2;                 /* Eq. 55 */
            for (int d = 0; d < 3; d++) V[3 * c + d] = V[3 * c + d] / (1.0 + Kv * dt);           /* Eq. 51 */
            double T = p[c] / (rho[c] * P->Rd);
            T = (T + KT * dt * Teq) / (1.0 + KT * dt);                                           /* Eq. 52 */
            p[c] = rho[c] * P->Rd * T;
        }
    }
}
/* NEXT-2, second half: the tidally locked hot-Jupiter forcing of section 7.2 (Eq. 59-61):
 *   K_v = 0 (L512); K_T = 1/tau_rad, constant (L529: 1.5e5 s);
 *   T_eq = T_vert(z) + beta_trop(sigma, z) dT_EP cos(lon) cos(lat)                           (Eq. 59)
 *   beta_trop = sin(pi (sigma - sigma_stra) / (2 (1 - sigma_stra))) for z <= z_stra, else 0    (Eq. 60)
 *   T_vert = T_surf - Gamma (z_stra + (z - z_stra)/2) + sqrt((Gamma (z - z_stra)/2)^2 + dT_stra^2)  for z <= z_stra,
 *            T_surf - Gamma z_stra + dT_stra                                                   for z >  z_stra  (Eq. 61, G15)
 * cos(lon) cos(lat) is the x component of the column's unit vector: the substellar point is on the x axis.
 * sigma as in the Held-Suarez forcing (L390).  beta_trop is clamped at 0 where sigma < sigma_stra below
 * z_stra (the sine would turn negative; reading RJ1). */
typedef struct { double T_surf, Gamma, dT_stra, z_stra, sigma_stra, dT_EP, tau_rad; } orc_hot_jupiter;

static void forcing_hot_jupiter(const orc_geom *G, double dt, double *rho, double *p, const orc_hot_jupiter *J) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
    const double KT = 1.0 / J->tau_rad, pi = 3.14159265358979323846;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; i++) {
        const double mu = G->xyz[3 * i];
        size_t c0 = (size_t)i * nv;
        const double T0 = p[c0] / (rho[c0] * P->Rd);
        const double ps = p[c0] * exp(P->gravity * G->z_c[0] / (P->Rd * T0));
        for (int k = 0; k < nv; k++) {
            size_t c = c0 + k;
            const double z = G->z_c[k], sigma = p[c] / ps;
            double Tvert, beta = 0.0;
            if (z <= J->z_stra) {
                const double hz = 0.5 * J->Gamma * (z - J->z_stra);
                Tvert = J->T_surf - J->Gamma * (J->z_stra + 0.5 * (z - J->z_stra)) + sqrt(hz * hz + J->dT_stra * J->dT_stra);
                if (sigma > J->sigma_stra) beta = sin(pi * (sigma - J->sigma_stra) / (2.0 * (1.0 - J->sigma_stra)));
            } else {
                Tvert = J->T_surf - J->Gamma * J->z_stra + J->dT_stra;
            }
            const double Teq = Tvert + beta * J->dT_EP * mu;                                     /* Eq. 59 */
            double T = p[c] / (rho[c] * P->Rd);
            T = (T + KT * dt * Teq) / (1.0 + KT * dt);                                           /* Eq. 52 */
            p[c] = rho[c] * P->Rd * T;
        }
    }
}
void orc_forcing_hot_jupiter(const orc_geom *G, double dt, double *rho, double *p, const double *hj) {
    forcing_hot_jupiter(G, dt, rho, p, (const orc_hot_jupiter *)hj);
}

void orc_forcing_held_suarez(const orc_geom *G, double dt, double *rho, double *V, double *p, const double *hs) {
    forcing_held_suarez(G, dt, rho, V, p, (const orc_held_suarez *)hs);
}

/* One call = n_large large steps (Fig. 6; stage convention R1 of SURVEY O5).
 * State arrays are updated in place: rho,p [N][nv]; V [N][nv][3]; W [N][nv+1] (ends forced to 0). */
double orc_dbar(double radius, int level);
double orc_kd(double D, double dbar, double dt);

/* D_hyp, D_div: the non-dimensional diffusion parameter of Eq. 49 for the hyper-diffusion and for the
 * divergence damping (the paper uses the same value for both, L367); 0 switches a term off, and
 * (0, 0) is the base path of SURVEY 8(a), arithmetic untouched. */
/* NEXT-4, energy fixer (L215: "a scheme proposed by Williamson et al. (2009), which globally uniform adjusts the
 * internal energy at all grid points"; the paper's own runs leave it off).  Reading RE1: after the
 * dynamics of a large step and before its forcing, the total energy E' (orc_diagnostics, R10) is brought back to its
 * value E before the step by ONE temperature increment for all cells, dT = (E - E')/(Cv M) with M the total mass:
 * rho unchanged, p <- p + rho Rd dT, which adds Cv dT M = E - E' of internal energy.  Off by default. */
static int g_efix = 0;
void orc_set_energy_fixer(int on) { g_efix = on; }
void orc_diagnostics(const orc_geom *G, const double *rho, const double *V, const double *W, const double *p,
                     double *mass, double *energy);
static const orc_held_suarez *g_hs = NULL;   /* set by orc_step_held_suarez for the duration of its call */
static const orc_hot_jupiter *g_hj = NULL;   /* likewise, orc_step_hot_jupiter */

void orc_step_diffusion(const orc_geom *G, double *rho, double *V, double *W, double *p, int n_large, double dt,
                        int n_sub, const double *T_eq, const double *k_T, const double *k_v, double D_hyp, double D_div) {
    const int N = G->N, nv = G->nv;
    orc_work *w = work_new(G);
    const size_t nc = w->nc, ni = w->ni;
    {
        int level = 0;
        while (10 * (1 << (2 * level)) + 2 < N) level++;          /* Eq. 1 inverted */
        const double dbar = orc_dbar(G->P.radius, level);         /* Eq. 2 */
        w->Kd_hyp = D_hyp > 0.0 ? orc_kd(D_hyp, dbar, dt) : 0.0;  /* Eq. 49 */
        w->Kd_div = D_div > 0.0 ? orc_kd(D_div, dbar, dt) : 0.0;
    }
    for (int i = 0; i < N; i++) { W[(size_t)i * (nv + 1)] = 0.0; W[(size_t)i * (nv + 1) + nv] = 0.0; }
    for (int step = 0; step < n_large; step++) {
        double M0 = 0.0, E0 = 0.0;
        if (g_efix) orc_diagnostics(G, rho, V, W, p, &M0, &E0);
        memcpy(w->rho_n, rho, 8 * nc); memcpy(w->V_n, V, 24 * nc); memcpy(w->W_n, W, 8 * ni); memcpy(w->p_n, p, 8 * nc);
#pragma omp parallel for schedule(static)
        for (size_t c = 0; c < nc; c++) w->rt_n[c] = eos_rt(&G->P, w->p_n[c]);
        memcpy(w->rho_t, rho, 8 * nc); memcpy(w->V_t, V, 24 * nc); memcpy(w->W_t, W, 8 * ni); memcpy(w->p_t, p, 8 * nc);
        for (int stage = 1; stage <= 3; stage++) {                 /* Eq. 30 (L245-L250) */
            stage_coefficients(G, w);                              /* Fig. 6 large-step 1 */
            slow_terms(G, w);                                      /* Fig. 6 large-step 3 */
            if (w->Kd_hyp > 0.0) hyper_diffusion(G, w);            /* Fig. 6 large-step 2 (NEXT-1) */
            int ns; double delta;                                  /* L252, L312-L316 */
            if (stage == 1) { ns = 1; delta = dt / 3.0; }
            else if (stage == 2) { ns = n_sub / 2; delta = dt / n_sub; }
            else { ns = n_sub; delta = dt / n_sub; }
            /* Eq. 31: deviations from the stage reference, every stage starting from t_n */
#pragma omp parallel for schedule(static)
            for (size_t c = 0; c < nc; c++) {
                w->rho_s[c] = w->rho_n[c] - w->rho_t[c];
                w->p_s[c] = w->p_n[c] - w->p_t[c];
                w->rt[c] = w->rt_n[c];
                for (int d = 0; d < 3; d++) w->V_s[3 * c + d] = w->V_n[3 * c + d] - w->V_t[3 * c + d];
            }
#pragma omp parallel for schedule(static)
            for (size_t c = 0; c < ni; c++) w->W_s[c] = w->W_n[c] - w->W_t[c];
            for (int s = 0; s < ns; s++) substep(G, w, delta);
            /* Fig. 6 large-step 4: Phi^(s) = Phi^[t] + Phi* */
#pragma omp parallel for schedule(static)
            for (size_t c = 0; c < nc; c++) {
                w->rho_t[c] = w->rho_t[c] + w->rho_s[c];
                w->p_t[c] = w->p_t[c] + w->p_s[c];
                for (int d = 0; d < 3; d++) w->V_t[3 * c + d] = w->V_t[3 * c + d] + w->V_s[3 * c + d];
            }
#pragma omp parallel for schedule(static)
            for (size_t c = 0; c < ni; c++) w->W_t[c] = w->W_t[c] + w->W_s[c];
        }
        memcpy(rho, w->rho_t, 8 * nc); memcpy(V, w->V_t, 24 * nc); memcpy(W, w->W_t, 8 * ni); memcpy(p, w->p_t, 8 * nc);
        if (g_efix) {                                              /* RE1 */
            double M1, E1;
            orc_diagnostics(G, rho, V, W, p, &M1, &E1);
            const double dT = (E0 - E1) / ((G->P.Cp - G->P.Rd) * M1);
            for (size_t c = 0; c < nc; c++) p[c] = p[c] + rho[c] * G->P.Rd * dT;
        }
        if (g_hj) forcing_hot_jupiter(G, dt, rho, p, g_hj);
        else if (g_hs) forcing_held_suarez(G, dt, rho, V, p, g_hs);
        else forcing(G, dt, rho, V, p, T_eq, k_T, k_v);
    }
    work_free(w);
}
void orc_step_hot_jupiter(const orc_geom *G, double *rho, double *V, double *W, double *p, int n_large, double dt,
                          int n_sub, const double *hj, double D_hyp, double D_div) {
    g_hj = (const orc_hot_jupiter *)hj;
    orc_step_diffusion(G, rho, V, W, p, n_large, dt, n_sub, NULL, NULL, NULL, D_hyp, D_div);
    g_hj = NULL;
}
/* hs: the nine numbers of orc_held_suarez */
void orc_step_held_suarez(const orc_geom *G, double *rho, double *V, double *W, double *p, int n_large, double dt,
                          int n_sub, const double *hs, double D_hyp, double D_div) {
    g_hs = (const orc_held_suarez *)hs;
    orc_step_diffusion(G, rho, V, W, p, n_large, dt, n_sub, NULL, NULL, NULL, D_hyp, D_div);
    g_hs = NULL;
}
void orc_step(const orc_geom *G, double *rho, double *V, double *W, double *p, int n_large, double dt,
              int n_sub, const double *T_eq, const double *k_T, const double *k_v) {
    orc_step_diffusion(G, rho, V, W, p, n_large, dt, n_sub, T_eq, k_T, k_v, 0.0, 0.0);
}

/* a12 (O8, R10): total mass and total energy with the weight A_c r_k^2 dz under which D_c telescopes.
 * Neumaier-compensated sums, serial, so the result does not depend on threads. */
static void ksum(double *s, double *comp, double x) {
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *comp += (*s - t) + x; else *comp += (x - t) + *s;
    *s = t;
}
void orc_diagnostics(const orc_geom *G, const double *rho, const double *V, const double *W, const double *p,
                     double *mass, double *energy) {
    const int N = G->N, nv = G->nv;
    const orc_planet *P = &G->P;
    const double Cv = P->Cp - P->Rd;
    double sm = 0, cm = 0, se = 0, ce = 0;
    for (int i = 0; i < N; i++)
        for (int k = 0; k < nv; k++) {
            size_t c = (size_t)i * nv + k;
            double vol = G->Ac[i] * G->r_c[k] * G->r_c[k] * (G->uniform ? G->dz : G->z_h[k + 1] - G->z_h[k]);
            double wc = I_c(W + (size_t)i * (nv + 1), k);
            double ke = 0.5 * (V[3 * c] * V[3 * c] + V[3 * c + 1] * V[3 * c + 1] + V[3 * c + 2] * V[3 * c + 2] + wc * wc) / rho[c];
            double e = Cv * p[c] / P->Rd + ke + rho[c] * P->gravity * G->z_c[k];
            ksum(&sm, &cm, rho[c] * vol);
            ksum(&se, &ce, e * vol);
        }
    *mass = sm + cm;
    *energy = se + ce;
}

/* ---------------------------------------------------------------------------------------------
 * Pieces exposed one at a time for the pins (same code the step runs)
 * ------------------------------------------------------------------------------------------- */

/* NEXT-3 pins: the vertical operators alone on one column.  order_k != 0: the interpolations at the order of
 * the run (I_hk, I_ck), else the linear ones of the acoustic system.  Yc [nv] -> Ih [nv+1] (ends 0), Gh [nv+1]
 * (ends 0); Xh [nv+1] -> Ic [nv], Dc [nv]. */
void orc_vertical_ops(const orc_geom *G, int order_k, const double *Yc, const double *Xh,
                      double *Ih, double *Gh, double *Ic, double *Dc) {
    const int nv = G->nv;
    Ih[0] = Ih[nv] = Gh[0] = Gh[nv] = 0.0;
    for (int k = 1; k < nv; k++) {
        Ih[k] = order_k ? I_hk(G, Yc, k) : I_h(G, Yc, k);
        Gh[k] = G_h(G, Yc, k);
    }
    for (int k = 0; k < nv; k++) {
        Ic[k] = order_k ? I_ck(G, Xh, k) : I_c(Xh, k);
        Dc[k] = D_c(G, Xh, k);
    }
}

/* P10: tridiagonal coefficients of one column, arrays [nv+1] indexed by interface */
void orc_tridiag_coefficients(const orc_geom *G, double delta, const double *h, const double *gt,
                              double *a, double *b, double *c) {
    tridiag_coefficients(G, delta, h, gt, a, b, c);
}

/* P13 / P12: slow terms of a given state; outputs sized as in orc_work */
void orc_slow_terms(const orc_geom *G, const double *rho, const double *V, const double *W, const double *p,
                    double *slowV, double *slowrho, double *Svr, double *slowp, double *slowrt,
                    double *h, double *th, double *gt) {
    orc_work *w = work_new(G);
    memcpy(w->rho_t, rho, 8 * w->nc); memcpy(w->V_t, V, 24 * w->nc); memcpy(w->W_t, W, 8 * w->ni); memcpy(w->p_t, p, 8 * w->nc);
    stage_coefficients(G, w);
    slow_terms(G, w);
    memcpy(slowV, w->slowV, 24 * w->nc); memcpy(slowrho, w->slowrho, 8 * w->nc); memcpy(Svr, w->Svr, 8 * w->ni);
    memcpy(slowp, w->slowp, 8 * w->nc); memcpy(slowrt, w->slowrt, 8 * w->nc);
    memcpy(h, w->h, 8 * w->nc); memcpy(th, w->th, 8 * w->nc); memcpy(gt, w->gt, 8 * w->ni);
    work_free(w);
}

/* P10: one substep on caller-provided stage data (all arrays in/out as named in O6) */
void orc_substep(const orc_geom *G, double delta, const double *h, const double *th, const double *gt,
                 const double *p_t, const double *slowV, const double *slowrho, const double *Svr,
                 const double *slowp, const double *slowrt,
                 double *rho_s, double *V_s, double *W_s, double *p_s, double *rt) {
    orc_work *w = work_new(G);
    size_t nc = w->nc, ni = w->ni;
    memcpy(w->h, h, 8 * nc); memcpy(w->th, th, 8 * nc); memcpy(w->gt, gt, 8 * ni); memcpy(w->p_t, p_t, 8 * nc);
    memcpy(w->slowV, slowV, 24 * nc); memcpy(w->slowrho, slowrho, 8 * nc); memcpy(w->Svr, Svr, 8 * ni);
    memcpy(w->slowp, slowp, 8 * nc); memcpy(w->slowrt, slowrt, 8 * nc);
    memcpy(w->rho_s, rho_s, 8 * nc); memcpy(w->V_s, V_s, 24 * nc); memcpy(w->W_s, W_s, 8 * ni);
    memcpy(w->p_s, p_s, 8 * nc); memcpy(w->rt, rt, 8 * nc);
    substep(G, w, delta);
    memcpy(rho_s, w->rho_s, 8 * nc); memcpy(V_s, w->V_s, 24 * nc); memcpy(W_s, w->W_s, 8 * ni);
    memcpy(p_s, w->p_s, 8 * nc); memcpy(rt, w->rt, 8 * nc);
    work_free(w);
}

/* NEXT-1 pins: the diffusive fluxes of a given state alone (slow terms start at zero), and the
 * divergence-damping flux of a given momentum field */
void orc_diffusion_fluxes(const orc_geom *G, const double *rho, const double *V, const double *W, const double *p,
                          double Kd, double *Frho, double *FV, double *FW, double *Fp, double *Frt) {
    orc_work *w = work_new(G);
    memcpy(w->rho_t, rho, 8 * w->nc); memcpy(w->V_t, V, 24 * w->nc); memcpy(w->W_t, W, 8 * w->ni); memcpy(w->p_t, p, 8 * w->nc);
    w->Kd_hyp = Kd;
    hyper_diffusion(G, w);
    memcpy(Frho, w->slowrho, 8 * w->nc); memcpy(FV, w->slowV, 24 * w->nc); memcpy(FW, w->Svr, 8 * w->ni);
    memcpy(Fp, w->slowp, 8 * w->nc); memcpy(Frt, w->slowrt, 8 * w->nc);
    work_free(w);
}
void orc_divergence_damping(const orc_geom *G, const double *V, const double *W, double Kd, double *Fdd) {
    orc_work *w = work_new(G);
    memcpy(w->V_t, V, 24 * w->nc); memcpy(w->W_t, W, 8 * w->ni);
    w->Kd_div = Kd;
    divergence_damping(G, w);
    memcpy(Fdd, w->Fdd, 24 * w->nc);
    work_free(w);
}

int orc_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    extern void omp_set_num_threads(int);
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
