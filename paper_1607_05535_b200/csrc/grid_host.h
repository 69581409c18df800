// Host-side icosahedral grid generator and finite-volume stencil weights (PAPER.md:L43-L125,
// Eq. 1-13).  Internal to the library; the C-ABI in include/thor.h exposes it as thor_grid_*.
#pragma once
#include <vector>

#include "thor.h"

namespace thor {

struct HostGrid {
    int level = 0, N = 0, nv = 0;
    thor_planet P{};
    int spring_iterations = 0;
    // canonical order (the generator's numbering)
    std::vector<double> xyz;       // [N][3]
    std::vector<int> nbr;          // [N][6], -1 pads pentagons
    std::vector<int> deg;          // [N]
    std::vector<double> cv;        // [N][6][3] control-volume vertices C_k
    std::vector<double> area;      // [N]
    std::vector<double> len;       // [N][6]
    std::vector<double> nrm;       // [N][6][3]
    std::vector<int> order;        // [N] device slot -> canonical index
    std::vector<int> rank;         // [N] canonical index -> device slot
    // device order, ready to upload
    std::vector<int> d_nbr;        // [N][6] device slots of the neighbours; pentagons: slot 5 = self
    std::vector<double> d_wdiv;    // [N][7][3] div_i = sum_j wdiv[j] . Phi_j   (j = 0 self, 1..6 neighbours)
    std::vector<double> d_wgrad;   // [N][6][3] grad_i = sum_j wgrad[j] (s_j - s_i), already tangent (Eq. 28)
    std::vector<double> d_rhat;    // [N][3]
    std::vector<double> d_wlap;    // [N][6] lap_i = sum_j wlap[j] (s_j - s_i): gradient on the triangles, then Eq. 6 (L369-L371)
    // tangent-plane storage of the acoustic horizontal momentum: per-column orthonormal basis (e1, e2)
    // and the same two stencils contracted with it, so that V* = a e1 + b e2 moves as 2 rows, not 3
    std::vector<double> d_basis;   // [N][6]  e1(3), e2(3)
    std::vector<double> d_wdiv2;   // [N][7][2] (wdiv[j] . e1_j, wdiv[j] . e2_j)  with e of column j (0 = self)
    std::vector<double> d_wgrad2;  // [N][6][2] (wgrad[j] . e1_i, wgrad[j] . e2_i) with e of the column itself
    std::vector<double> d_area;    // [N]
    // per-layer tables
    std::vector<double> rinv;      // [nv] 1/r_k
    std::vector<double> dlo;       // [nv] r_h,k^2   / (r_k^2 dz)
    std::vector<double> dhi;       // [nv] r_h,k+1^2 / (r_k^2 dz)
    std::vector<double> vol;       // [nv] r_k^2 dz
    std::vector<double> zc;        // [nv] centre altitude (midpoint of the layer's interfaces)
    std::vector<double> zh;        // [nv+1] interface altitudes, zh[0] = 0, zh[nv] = z_top (uniform unless given)
    std::vector<double> rhinv;     // [nv] 1/r_h,k (lower interface of layer k)
    // Eq. 8-9 with k = 1 at the lower interface of layer k >= 1 (0 for k = 0)
    std::vector<double> wl, wh;    // [nv] weights of the centres below / above the interface
    std::vector<double> idz;       // [nv] 1/(z_k - z_k-1)
    double dz = 0;                 // z_top / nv (mean thickness)
    // NEXT-3: Eq. 8-9 of order kord (1 or 3) in the explicit slow terms (RV1, RV2).  kord = 3: Lagrange weights of
    // the four nearest nodes, 0 for the nodes the column's end cuts off (the order falls by one per missing node)
    // Interior lattice points of a rhombus (1 <= I <= n-2, 1 <= J-1 <= n-2) have their six neighbours at the fixed
    // lattice offsets (1,0), (0,1), (-1,1), (-1,0), (0,-1), (1,-1), counter-clockwise, in the same rhombus: their
    // device slots are rotated to start at (1,0), so that the kernels can COMPUTE the neighbour columns from the
    // column's own Morton index instead of loading them (true when the generator has verified it for every such column)
    bool lattice_nbr = false;
    // NEXT-4 (reading RS1): shallow-atmosphere approximation -- every radius in the vertical tables is the planetary
    // radius (1/r_k = 1/A, no r^2 factors in D_c, volume A^2 dz); the slow-term kernels switch their Coriolis and
    // advection terms on the same flag
    bool shallow = false;
    int kord = 1;
    std::vector<double> ihw;       // [4][nv] centre k-2, k-1, k, k+1 -> lower interface of layer k (0 for k = 0)
    std::vector<double> icw;       // [4][nv] interface k-1, k, k+1, k+2 -> centre of layer k
};

// One spring-dynamics relaxation (Eq. 10-12) of the N points xyz [N][3] (in place) on the refinement level whose
// neighbour table is nbr [N][6] / deg [N]; returns the number of steps taken, < 0 on failure.  The constants of the
// iteration are passed in so that the host loop (grid_host.cpp) and the device loop (thor_api.cu, NEXT-3) share them.
struct SpringParams {
    double dspr, k, alpha, dt, tol;   // Eq. 12 natural length (unit sphere), spring constant, drag, time step, stop test
    int min_iter, max_iter;
};
using SpringFn = int (*)(int N, double* xyz, const int* nbr, const int* deg, const SpringParams& sp);

// Builds everything above.  Returns THOR_OK or THOR_EINVAL / THOR_ENOMEM (THOR_ECUDA from a device `spring`).
// kord: order of Eq. 8-9 in the explicit slow terms, 1 (the paper's choice, L94) or 3.  spring: nullptr = the host loop.
// z_interfaces: nullptr (uniform layers, R6) or nv+1 strictly increasing altitudes from 0 to P.z_top.
int build_host_grid(int level, int nv, const thor_planet& P, HostGrid& g, const double* z_interfaces = nullptr, int kord = 1,
                    SpringFn spring = nullptr, bool shallow = false);

}  // namespace thor
