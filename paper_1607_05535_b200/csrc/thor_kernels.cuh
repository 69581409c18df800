// sm_100a kernels of the THOR HE-VI large step (Fig. 6).
//
// Data layout in HBM: ONE slab of column records, columns in the
// locality-preserving device order, padded to a whole number of thread blocks:
//
//     S[column][field][layer]     field = one of the NF rows below, layer fastest, NVP doubles per row
//
// NVP = G*E is the layer count rounded up to 8/16/32/64/128.  A column is owned by a group of G
// lanes; each lane holds E (even) CONSECUTIVE layers, so every row access is a 128-bit load/store,
// a neighbour column's row is one contiguous 8*NVP-byte segment, every field of a column sits at a
// compile-time offset from one base address, and vertical neighbours are in the same lane or one
// shuffle away.  The rows a kernel reads together are adjacent in the record (the acoustic
// column-solve kernel reads rows 0..15 of its own column: one contiguous 16*NVP*8-byte block).
//
// W (= rho v_r) is stored on the LOWER interface of each layer (slot 0 = ground = 0; the lid above
// the top layer is an implicit 0).  Pad layers (k >= n_layers) and pad columns hold exact zeros in
// every deviation / slow-term / LU-factor row and harmless finite values elsewhere, so they never
// need a branch and never leak into real layers (see "pad invariant" in DESIGN.md).
//
// The path is an HBM-bound 7-point gather plus a per-column recurrence: no tensor cores.
#pragma once
#include <cuda_runtime.h>

#include <cstddef>

namespace thor {

constexpr unsigned kFull = 0xffffffffu;
// measurement knobs (compile time; the defaults are the measured best, profiles/r02*_variants.md)
#ifndef THOR_WPB
#define THOR_WPB 4
#endif
#ifndef THOR_K2_MINB
#define THOR_K2_MINB 4
#endif
#ifndef THOR_KS_MINB
#define THOR_KS_MINB 4
#endif
#ifndef THOR_KP_MINB
#define THOR_KP_MINB 5
#endif
#ifndef THOR_GEOMPF
#define THOR_GEOMPF 1     // 1: the look-ahead also prefetches the stencil data (neighbour slots, weights) of the block ahead
#endif
constexpr int kWarpsPerBlock = THOR_WPB;
constexpr int kColPad = 64;      // columns are padded to a multiple of this (>= columns per block of any shape)
constexpr int kEosTerms = 11;    // degree of the binomial series of Eq. 36 in deviation form
constexpr double kEosSmall = 0.03125;   // |x| <= 2^-5: series; beyond: expm1/log1p

// rows of a column record
enum Field : int {
    // --- acoustic substep, gathered from the 6 neighbours by the column-solve kernel
    F_VAS = 0, F_VBS,            // V* = (rho v_h)* = a e1 + b e2 in the column's tangent basis  (Eq. 31, 33)
    F_H, F_TH,                   // h = Cp T, theta of the stage reference state                (Eq. 38)
    // --- acoustic substep, column-local
    F_PS,                        // p*        (gathered by the momentum kernel)
    F_RHOS, F_WS, F_RTS,         // rho*, W* = (rho v_r)*, (rho theta)*
    F_SRHO, F_SP, F_SW, F_SRT,   // slow terms of Eq. 32, 40, 42, 35
    F_FA, F_FI, F_FC,            // LU factors of the tridiagonal matrix of Eq. 37
    F_PT,                        // p^[t]     (gathered by the slow-term kernel)
    F_SVA, F_SVB,                // slow term of Eq. 33, tangent basis
    // --- stage reference state Phi^[t] (R1): horizontal momentum in the tangent basis, 1/rho, W, rho.
    //     The slow-term kernel gathers VAT, VBT, IRT, WT (+ TH, PT) from the neighbours and rebuilds the
    //     un-projected velocity u = (V + I_c[W] r)/rho of L268 and h = Cp p/(Rd rho) from them.
    F_VAT, F_VBT, F_IRT, F_WT, F_RHOT,
    // --- Phi^n (the prognostic state between large steps, Cartesian momentum: what thor_state_get returns
    //     bit-exactly) and (rho theta)^n
    F_RHON, F_VXN, F_VYN, F_VZN, F_WN, F_PN, F_RTN,
    NF
};

// rows of the NEXT-1 work slab X (hyper-diffusion and divergence damping)
enum XField : int {
    X_W = 0,                                     // k_stage_prepare: w = W/I_h[rho] of Phi^[t] on interior interfaces
    X_Q0, X_Q1, X_Q2, X_Q3, X_Q4, X_Q5,          // k_slow_terms<HYP>: lap(rho), rho lap(v_x..z), rho_h lap(w), rho lap(T)
    X_D3,                                        // 3-D divergence of the current momentum (column-solve kernel, per substep)
    X_D3T,                                       // ... of the stage reference state (k_slow_terms, per stage)
    X_D3N,                                       // ... of Phi^n (k_slow_terms of stage 1): the first substep's D3 of every stage
    XF
};

// NOTE: the struct is a kernel parameter, so its layout decides the constant-bank offsets the kernels read their scalars
// from.  Shifting the fields after lvl2 by 8 bytes made k_slow_terms (at its 128-register cap) 5 us slower per launch
// (profiles/r02c_variants.md): flags that only choose a kernel variant belong on the host (HostGrid), not in here.
struct Geom {                 // device pointers, device column order, padded to Npad columns
    int N, Npad, nv;
    const int* nbr;           // [Npad][8]   6 neighbours (pentagons, pad columns: self), 2 x self
    const double* wdiv;       // [Npad][24]  7 x 3 divergence weights (Eq. 4-6 expanded), 3 pad        (config-1 operators)
    const double* wgrad;      // [Npad][18]  6 x 3 gradient weights (Eq. 7, projected by Eq. 28)       (config-1 operators)
    const double* wlap;       // [Npad][8]   6 Laplacian weights (Eq. 7 on the triangles, then Eq. 6; L369-L371), 2 pad
    const int* dd_idx;        // [Npad][20]  NEXT-1 divergence damping composed over two rings: columns m ...
    const double* dd_coef;    // [Npad][20][2] ... and tangent coefficients of (D3_m - D3_i); F_dd = -K_d/r^3 sum_m coef_m (D3_m - D3_i)
    const double* frame;      // [Npad][12]  tangent basis e1(3), e2(3), unit vector r(3) of the column, 3 pad
    const double* wdiv2;      // [Npad][16]  7 x 2 divergence weights contracted with the basis of column j, 2 pad
    const double* wgrad2;     // [Npad][12]  6 x 2 gradient weights contracted with the column's own basis
    const double* area;       // [Npad]
    // per-layer tables [128]; layers need not be uniform (NEXT-3): layer k spans the interfaces z_h,k .. z_h,k+1,
    // its centre is their midpoint
    const double* rinv;       // 1/r_k              (pad layers: 0)
    const double* dlo;        // r_h,k^2/(r_k^2 dz_k)
    const double* dhi;        // r_h,k+1^2/(r_k^2 dz_k)
    const double* vol;        // r_k^2 dz_k
    const double* zc;         // centre altitude
    const double* rhinv;      // 1/r_h,k: radius of the LOWER interface of layer k (pad layers: 0)
    // Eq. 8-9 with k = 1 at the LOWER interface of layer k (0 for k = 0 and on pads):
    const double* wl;         // weight of the centre below:  (z_k - z_h,k)/(z_k - z_k-1)
    const double* wh;         // weight of the centre above:  (z_h,k - z_k-1)/(z_k - z_k-1)
    const double* idz;        // 1/(z_k - z_k-1), the spacing of G_h
    // NEXT-3 (RV1, RV2): Eq. 8-9 of order 3 in the explicit slow terms, [8][128]: rows 0-3 the weights of the centres
    // k-2, k-1, k, k+1 at the lower interface of layer k; rows 4-7 those of the interfaces k-1, k, k+1, k+2 at the
    // centre of layer k (0 for the nodes the column's end cuts off, and on pads); used when kord == 3
    const double* vk;
    int kord;
    // >= 0: twice the grid level; interior lattice points of a rhombus then have their neighbour columns COMPUTED
    // from their own Morton index (HostGrid::lattice_nbr); -1: always the nbr table
    int lvl2;
    double omega, gravity, Rd, Cp, p_ref;
    double eosq[kEosTerms + 1];   // q_k = C(gamma, k+1)/gamma, k = 0..kEosTerms
};
// measured (profiles/r02c_variants.md): with the scalar block 8 bytes further on (or at the head of the struct) the
// large step of config 3 is 1053 us instead of 1037 us; 16 or 32 bytes further on it is 1037 us again
static_assert(offsetof(Geom, omega) % 16 == 8, "keep the scalar block of Geom where the kernels were tuned (see above)");

struct Forcing {              // [Npad][NVP] each, may be null (Eq. 51-52)
    const double *T_eq, *k_T, *k_v;
};
// NEXT-2: Held-Suarez forcing from the evolving sigma = p/p_s (Eq. 53-55); on != 0 replaces the tables
struct HeldSuarez {
    int on;
    double T_surf, dT_y, dth_z, T_min, k_a, k_s, k_f, sigma_b, p_star;
};
// NEXT-2: tidally locked hot-Jupiter forcing of section 7.2 (Eq. 59-61); K_v = 0, K_T = 1/tau_rad
struct HotJupiter {
    int on;
    double T_surf, Gamma, dT_stra, z_stra, sigma_stra, dT_EP, tau_rad;
};

// L2 schedule of one launch (defaults in thor_api.cu).  Successive kernels of a
// large step walk the columns in ALTERNATING directions, so each starts on the rows the previous one has
// just left in the 126 MB L2.
struct Tune {
    int rev;    // 1: this launch walks the blocks in descending column order
    int ahead;  // blocks of look-ahead of the in-kernel bulk L2 prefetch (0 = off)
    int tail;   // the last `tail` blocks (in walking order) prefetch rows the NEXT kernel reads first (0 = off)
};
struct Walk {
    int bid;         // block of columns this thread block works on
    int ahead_bid;   // block to prefetch for (walking order), -1 = none
    bool in_tail;
    __device__ explicit Walk(const Tune& tn) {
        const int nblk = gridDim.x, b = blockIdx.x;
        bid = tn.rev ? nblk - 1 - b : b;
        ahead_bid = (tn.ahead > 0 && b + tn.ahead < nblk) ? (tn.rev ? nblk - 1 - (b + tn.ahead) : b + tn.ahead) : -1;
        in_tail = tn.tail > 0 && b >= nblk - tn.tail;
    }
};

// TMA bulk prefetch of a contiguous global range into L2 (no shared memory, no registers held)
__device__ __forceinline__ void bulk_prefetch_l2(const void* p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
// rows [f0, f0 + nf) of every column of block `bid`, issued by the first warp of the calling block
template <int G, int E>
__device__ __forceinline__ void prefetch_block_rows(const double* S, int bid, int f0, int nf) {
    constexpr int NVP = G * E, CPB = kWarpsPerBlock * (32 / G);
    if (threadIdx.x < 32)
        for (int c = threadIdx.x; c < CPB; c += 32)
            bulk_prefetch_l2(S + (size_t(bid) * CPB + c) * (size_t(NF) * NVP) + size_t(f0) * NVP, unsigned(nf) * NVP * 8u);
}

// rows [f0, f0 + nf) of the NEXT-1 work slab X of every column of block `bid`; one [Npad][NVP] table row per column
template <int G, int E>
__device__ __forceinline__ void prefetch_block_xrows(const double* X, int bid, int f0, int nf) {
    constexpr int NVP = G * E, CPB = kWarpsPerBlock * (32 / G);
    if (threadIdx.x < 32)
        for (int c = threadIdx.x; c < CPB; c += 32)
            bulk_prefetch_l2(X + (size_t(bid) * CPB + c) * (size_t(XF) * NVP) + size_t(f0) * NVP, unsigned(nf) * NVP * 8u);
}
template <int G, int E>
__device__ __forceinline__ void prefetch_block_table(const double* T, int bid) {
    constexpr int NVP = G * E, CPB = kWarpsPerBlock * (32 / G);
    if (T && threadIdx.x == 0) bulk_prefetch_l2(T + size_t(bid) * CPB * NVP, unsigned(CPB) * NVP * 8u);
}
// the per-column stencil data of block `bid` (contiguous per array): `per_col` doubles or ints of `bytes_per` bytes each
template <int G>
__device__ __forceinline__ void prefetch_block_geom(const void* base, int bid, int bytes_per_col) {
    constexpr int CPB = kWarpsPerBlock * (32 / G);
    if (threadIdx.x == 0)
        bulk_prefetch_l2(static_cast<const char*>(base) + size_t(bid) * CPB * bytes_per_col, unsigned(CPB * bytes_per_col));
}

// ---------------------------------------------------------------------------------------------
// lane <-> (column, layers) mapping of the record kernels
// ---------------------------------------------------------------------------------------------
template <int G, int E>
struct Map {
    static_assert(E % 2 == 0, "two layers per 128-bit access");
    static constexpr int NVP = G * E;
    static constexpr int CPW = 32 / G;                 // columns per warp
    static constexpr size_t REC = size_t(NF) * NVP;    // doubles per column record
    int col, gl, k0;
    __device__ explicit Map(int bid = blockIdx.x) {
        const int lane = threadIdx.x & 31;
        const int warp = bid * (blockDim.x >> 5) + (threadIdx.x >> 5);
        col = warp * CPW + lane / G;                   // < Npad by construction of the grid
        gl = lane & (G - 1);
        k0 = gl * E;
    }
};

// The six neighbour columns of `col`.  Device order: rhombus r owns columns r n^2 .. (r+1) n^2 - 1 along the Morton
// curve of its lattice (I in the odd bits, J-1 in the even bits).  A lattice point that is not on the rim of its
// rhombus has its neighbours at the offsets (1,0), (0,1), (-1,1), (-1,0), (0,-1), (1,-1) -- the slot order the host
// generator gives such columns -- so their indices follow from the column's own by Morton increments: no load, and
// the gathers that depend on them can be issued at once.  Rim columns, the poles and pad columns read the table.
__device__ __forceinline__ void neighbours(const Geom& g, int col, int (&nb)[6]) {
    if (g.lvl2 >= 0) {
        const unsigned nn = 1u << g.lvl2, XM = 0xAAAAAAAAu & (nn - 1), YM = 0x55555555u & (nn - 1);
        const unsigned m = unsigned(col) & (nn - 1), x = m & XM, y = m & YM;
        if (unsigned(col) < 10u * nn && x != 0 && x != XM && y != 0 && y != YM) {
            const unsigned base = unsigned(col) - m;
            const unsigned xp = ((m | YM) + 1) & XM, xn = (x - 1) & XM, yp = ((m | XM) + 1) & YM, yn = (y - 1) & YM;
            nb[0] = int(base + (xp | y));  nb[1] = int(base + (x | yp));  nb[2] = int(base + (xn | yp));
            nb[3] = int(base + (xn | y));  nb[4] = int(base + (x | yn));  nb[5] = int(base + (xp | yn));
            return;
        }
    }
    const int4 n03 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8));
    const int4 n47 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8) + 1);
    nb[0] = n03.x; nb[1] = n03.y; nb[2] = n03.z; nb[3] = n03.w; nb[4] = n47.x; nb[5] = n47.y;
}

template <int E>
__device__ __forceinline__ void ld_nc(const double* p, double (&v)[E]) {     // rows nobody writes in this kernel
#pragma unroll
    for (int i = 0; i < E / 2; ++i) {
        const double2 t = __ldg(reinterpret_cast<const double2*>(p) + i);
        v[2 * i] = t.x; v[2 * i + 1] = t.y;
    }
}
template <int E>
__device__ __forceinline__ void ld_rw(const double* p, double (&v)[E]) {
#pragma unroll
    for (int i = 0; i < E / 2; ++i) {
        const double2 t = reinterpret_cast<const double2*>(p)[i];
        v[2 * i] = t.x; v[2 * i + 1] = t.y;
    }
}
// A second read of a row this thread has already loaded (an L1 hit), kept out of the compiler's
// common-subexpression elimination so that the first copy does not have to stay in registers.
template <int E>
__device__ __forceinline__ void ld_again(const double* p, double (&v)[E]) {
#pragma unroll
    for (int i = 0; i < E / 2; ++i)
        asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(v[2 * i]), "=d"(v[2 * i + 1]) : "l"(p + 2 * i));
}
template <int E>
__device__ __forceinline__ void st_row(double* p, const double (&v)[E]) {
#pragma unroll
    for (int i = 0; i < E / 2; ++i) reinterpret_cast<double2*>(p)[i] = make_double2(v[2 * i], v[2 * i + 1]);
}

struct Frame { double3 e1, e2, r; };
__device__ __forceinline__ Frame ld_frame(const double* frame, int col) {   // [Npad][12]
    const double2* p = reinterpret_cast<const double2*>(frame) + 6 * size_t(col);
    const double2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2), d = __ldg(p + 3), e = __ldg(p + 4);
    return Frame{make_double3(a.x, a.y, b.x), make_double3(b.y, c.x, c.y), make_double3(d.x, d.y, e.x)};
}

// Per-column stencil weights staged once per warp in shared memory (every lane of a column group
// would otherwise hold the same 21-39 doubles in registers): the G lanes of a group copy `n2`
// double2's from `src` to `dst`; the caller reads them back as broadcast LDS.
template <int G>
__device__ __forceinline__ void stage_weights(const double* src, double* dst, int n2, int gl) {
    for (int i = gl; i < n2; i += G)
        reinterpret_cast<double2*>(dst)[i] = __ldg(reinterpret_cast<const double2*>(src) + i);
}

// value at layer k-1 (fill below the ground)
template <int G, int E>
__device__ __forceinline__ void below(const double (&v)[E], double (&out)[E], int gl, double fill) {
    double prev = __shfl_up_sync(kFull, v[E - 1], 1, G);
    if (gl == 0) prev = fill;
    out[0] = prev;
#pragma unroll
    for (int e = 1; e < E; ++e) out[e] = v[e - 1];
}
// value at layer k+1 (fill above the last lane)
template <int G, int E>
__device__ __forceinline__ void above(const double (&v)[E], double (&out)[E], int gl, double fill) {
    double next = __shfl_down_sync(kFull, v[0], 1, G);
    if (gl == G - 1) next = fill;
#pragma unroll
    for (int e = 0; e < E - 1; ++e) out[e] = v[e + 1];
    out[E - 1] = next;
}

// value at layer k-2 / k+2
template <int G, int E>
__device__ __forceinline__ void below2(const double (&v)[E], double (&out)[E], int gl, double fill) {
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const double prev = __shfl_up_sync(kFull, v[E - 2 + e], 1, G);
        out[e] = gl == 0 ? fill : prev;
    }
#pragma unroll
    for (int e = 2; e < E; ++e) out[e] = v[e - 2];
}
template <int G, int E>
__device__ __forceinline__ void above2(const double (&v)[E], double (&out)[E], int gl, double fill) {
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const double next = __shfl_down_sync(kFull, v[e], 1, G);
        out[E - 2 + e] = gl == G - 1 ? fill : next;
    }
#pragma unroll
    for (int e = 0; e < E - 2; ++e) out[e] = v[e + 2];
}
// NEXT-3, Eq. 8-9 of order 3 (RV1): centres -> lower interface of each layer, and interfaces -> centres;
// w points at the lane's first layer of Geom::vk rows 0-3 (resp. 4-7), row stride 128
template <int G, int E>
__device__ __forceinline__ void interp_h3(const double* w, const double (&q)[E], double (&out)[E], int gl) {
    double b2[E], b1[E], a1[E], w0[E], w1[E], w2[E], w3[E];
    below2<G, E>(q, b2, gl, 0.0); below<G, E>(q, b1, gl, 0.0); above<G, E>(q, a1, gl, 0.0);
    ld_nc<E>(w, w0); ld_nc<E>(w + 128, w1); ld_nc<E>(w + 256, w2); ld_nc<E>(w + 384, w3);
#pragma unroll
    for (int e = 0; e < E; ++e) out[e] = fma(a1[e], w3[e], fma(q[e], w2[e], fma(b1[e], w1[e], b2[e] * w0[e])));
}
template <int G, int E>
__device__ __forceinline__ void interp_c3(const double* w, const double (&X)[E], double (&out)[E], int gl) {
    double b1[E], a1[E], a2[E], w0[E], w1[E], w2[E], w3[E];
    below<G, E>(X, b1, gl, 0.0); above<G, E>(X, a1, gl, 0.0); above2<G, E>(X, a2, gl, 0.0);
    ld_nc<E>(w, w0); ld_nc<E>(w + 128, w1); ld_nc<E>(w + 256, w2); ld_nc<E>(w + 384, w3);
#pragma unroll
    for (int e = 0; e < E; ++e) out[e] = fma(a2[e], w3[e], fma(a1[e], w2[e], fma(X[e], w1[e], b1[e] * w0[e])));
}

// Eq. 24 (L210) and its inverse
__device__ __forceinline__ double eos_rt(double p, double Rd, double p_ref, double inv_gam) {
    return p_ref / Rd * pow(p / p_ref, inv_gam);
}

// Eq. 36 (L270) in deviation form: with x = (rho theta)* / (rho theta)^[t],
//   p* = p_ref (Rd (rho theta)/p_ref)^gamma - p^[t] = p^[t] ((1 + x)^gamma - 1)
//      = p^[t] gamma x (1 + q_1 x + q_2 x^2 + ...),   q_k = C(gamma, k+1)/gamma.
// Free of the cancellation of the printed form.  |x| <= 2^-5: the series is
// below 2^-57 relative after kEosTerms terms; beyond, expm1(gamma log1p x).
__device__ __forceinline__ double eos_dev(double x, double pt, double gam, const Geom& g) {
    if (fabs(x) <= kEosSmall) {
        double q = g.eosq[kEosTerms];
#pragma unroll
        for (int k = kEosTerms - 1; k >= 0; --k) q = fma(q, x, g.eosq[k]);
        return (pt * gam) * x * q;
    }
    return pt * expm1(gam * log1p(x));
}

// ---------------------------------------------------------------------------------------------
// Inclusive scan of the affine recurrence y_k = A_k y_(k-1) + B_k over the layers of a column
// (y_(-1) = 0), upward (DOWN = false) or x_k = A_k x_(k+1) + B_k downward (DOWN = true).
// Work-efficient inside a lane (E serial steps), Kogge-Stone across the G lanes.
// ---------------------------------------------------------------------------------------------
template <int G, int E, bool DOWN>
__device__ __forceinline__ void affine_scan(const double (&A)[E], const double (&B)[E], double (&y)[E], int gl) {
    double a = 1.0, b = 0.0;
    if (!DOWN) {
#pragma unroll
        for (int e = 0; e < E; ++e) { b = fma(A[e], b, B[e]); a = A[e] * a; }
    } else {
#pragma unroll
        for (int e = E - 1; e >= 0; --e) { b = fma(A[e], b, B[e]); a = A[e] * a; }
    }
#pragma unroll
    for (int s = 1; s < G; s <<= 1) {
        double ap = DOWN ? __shfl_down_sync(kFull, a, s, G) : __shfl_up_sync(kFull, a, s, G);
        double bp = DOWN ? __shfl_down_sync(kFull, b, s, G) : __shfl_up_sync(kFull, b, s, G);
        const bool has = DOWN ? (gl + s < G) : (gl >= s);
        if (has) { b = fma(a, bp, b); a = a * ap; }
    }
    double carry = DOWN ? __shfl_down_sync(kFull, b, 1, G) : __shfl_up_sync(kFull, b, 1, G);
    if (DOWN ? (gl == G - 1) : (gl == 0)) carry = 0.0;
    if (!DOWN) {
#pragma unroll
        for (int e = 0; e < E; ++e) { carry = fma(A[e], carry, B[e]); y[e] = carry; }
    } else {
#pragma unroll
        for (int e = E - 1; e >= 0; --e) { carry = fma(A[e], carry, B[e]); y[e] = carry; }
    }
}

// ---------------------------------------------------------------------------------------------
// Config-1 operators (Eq. 6 and Eq. 7) on caller-owned [column][layer] arrays (row length nv, no
// padding): G lanes per column, E layers per lane with stride G (coalesced scalar accesses).
// ---------------------------------------------------------------------------------------------
template <int G, int E>
struct Lanes {
    int col; bool live; int gl;
    __device__ Lanes(int N) {
        const int lane = threadIdx.x & 31;
        const int warp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
        const int c = warp * (32 / G) + lane / G;
        live = c < N;
        col = live ? c : N - 1;
        gl = lane & (G - 1);
    }
};

template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_div(Geom g, const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
      double* __restrict__ out) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const double* w = g.wdiv + size_t(L.col) * 24;
    double acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const int c = j == 0 ? L.col : __ldg(g.nbr + size_t(L.col) * 8 + j - 1);
        const double wx = __ldg(w + 3 * j), wy = __ldg(w + 3 * j + 1), wz = __ldg(w + 3 * j + 2);
        const size_t o = size_t(c) * nv;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = L.gl + e * G;
            if (k < nv) acc[e] = fma(wx, __ldg(vx + o + k), fma(wy, __ldg(vy + o + k), fma(wz, __ldg(vz + o + k), acc[e])));
        }
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.gl + e * G;
        if (L.live && k < nv) out[size_t(L.col) * nv + k] = acc[e] * __ldg(g.rinv + k);
    }
}

template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_grad(Geom g, const double* __restrict__ s, double* __restrict__ gx, double* __restrict__ gy,
       double* __restrict__ gz) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const double* w = g.wgrad + size_t(L.col) * 18;
    double s0[E], ax[E], ay[E], az[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.gl + e * G;
        s0[e] = k < nv ? __ldg(s + size_t(L.col) * nv + k) : 0.0;
        ax[e] = ay[e] = az[e] = 0.0;
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int c = __ldg(g.nbr + size_t(L.col) * 8 + j);
        const double wx = __ldg(w + 3 * j), wy = __ldg(w + 3 * j + 1), wz = __ldg(w + 3 * j + 2);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = L.gl + e * G;
            const double d = (k < nv ? __ldg(s + size_t(c) * nv + k) : 0.0) - s0[e];
            ax[e] = fma(wx, d, ax[e]); ay[e] = fma(wy, d, ay[e]); az[e] = fma(wz, d, az[e]);
        }
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.gl + e * G;
        if (L.live && k < nv) {
            const double ri = __ldg(g.rinv + k);
            const size_t o = size_t(L.col) * nv + k;
            gx[o] = ax[e] * ri; gy[o] = ay[e] * ri; gz[o] = az[e] * ri;
        }
    }
}

// Horizontal Laplacian of L369-L371 at radius r_k (NEXT-1 building block): lap_i = sum_j wlap[j] (s_j - s_i) / r_k^2
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_lap(Geom g, const double* __restrict__ s, double* __restrict__ out) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const double* w = g.wlap + size_t(L.col) * 8;
    double s0[E], acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.gl + e * G;
        s0[e] = k < nv ? __ldg(s + size_t(L.col) * nv + k) : 0.0;
        acc[e] = 0.0;
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int c = __ldg(g.nbr + size_t(L.col) * 8 + j);
        const double wj = __ldg(w + j);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = L.gl + e * G;
            acc[e] = fma(wj, (k < nv ? __ldg(s + size_t(c) * nv + k) : 0.0) - s0[e], acc[e]);
        }
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.gl + e * G;
        if (L.live && k < nv) {
            const double ri = __ldg(g.rinv + k);
            out[size_t(L.col) * nv + k] = acc[e] * ri * ri;
        }
    }
}

// The same two operators for even layer counts <= 64: two consecutive layers per lane (128-bit
// accesses), G = 4..32 lanes per column, weights staged in shared memory -- the fast path of config 1.
template <int G>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_div2(Geom g, const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
       double* __restrict__ out) {
    const int lane = threadIdx.x & 31, warp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int c0 = warp * (32 / G) + lane / G, gl = lane & (G - 1), k0 = 2 * gl, nv = g.nv;
    const bool live = c0 < g.N;
    const int col = live ? c0 : g.N - 1;
    __shared__ double wsm[kWarpsPerBlock * 32 / G][24];
    double* w = wsm[threadIdx.x / G];
    stage_weights<G>(g.wdiv + size_t(col) * 24, w, 12, gl);
    const int4 n03 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8));
    const int4 n47 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8) + 1);
    const int nb[7] = {col, n03.x, n03.y, n03.z, n03.w, n47.x, n47.y};
    __syncwarp();
    if (k0 >= nv) return;
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const size_t o = size_t(nb[j]) * nv + k0;
        const double2 x = __ldg(reinterpret_cast<const double2*>(vx + o)), y = __ldg(reinterpret_cast<const double2*>(vy + o)),
                      z = __ldg(reinterpret_cast<const double2*>(vz + o));
        const double wx = w[3 * j], wy = w[3 * j + 1], wz = w[3 * j + 2];
        acc.x = fma(wx, x.x, fma(wy, y.x, fma(wz, z.x, acc.x)));
        acc.y = fma(wx, x.y, fma(wy, y.y, fma(wz, z.y, acc.y)));
    }
    const double2 ri = __ldg(reinterpret_cast<const double2*>(g.rinv + k0));
    if (live) *reinterpret_cast<double2*>(out + size_t(col) * nv + k0) = make_double2(acc.x * ri.x, acc.y * ri.y);
}

template <int G>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_grad2(Geom g, const double* __restrict__ s, double* __restrict__ gx, double* __restrict__ gy, double* __restrict__ gz) {
    const int lane = threadIdx.x & 31, warp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int c0 = warp * (32 / G) + lane / G, gl = lane & (G - 1), k0 = 2 * gl, nv = g.nv;
    const bool live = c0 < g.N;
    const int col = live ? c0 : g.N - 1;
    __shared__ double wsm[kWarpsPerBlock * 32 / G][18];
    double* w = wsm[threadIdx.x / G];
    stage_weights<G>(g.wgrad + size_t(col) * 18, w, 9, gl);
    const int4 n03 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8));
    const int4 n47 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8) + 1);
    const int nb[6] = {n03.x, n03.y, n03.z, n03.w, n47.x, n47.y};
    __syncwarp();
    if (k0 >= nv) return;
    const double2 s0 = __ldg(reinterpret_cast<const double2*>(s + size_t(col) * nv + k0));
    double2 ax = make_double2(0.0, 0.0), ay = ax, az = ax;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const double2 sj = __ldg(reinterpret_cast<const double2*>(s + size_t(nb[j]) * nv + k0));
        const double d0 = sj.x - s0.x, d1 = sj.y - s0.y;
        ax.x = fma(w[3 * j], d0, ax.x); ay.x = fma(w[3 * j + 1], d0, ay.x); az.x = fma(w[3 * j + 2], d0, az.x);
        ax.y = fma(w[3 * j], d1, ax.y); ay.y = fma(w[3 * j + 1], d1, ay.y); az.y = fma(w[3 * j + 2], d1, az.y);
    }
    const double2 ri = __ldg(reinterpret_cast<const double2*>(g.rinv + k0));
    if (live) {
        const size_t o = size_t(col) * nv + k0;
        *reinterpret_cast<double2*>(gx + o) = make_double2(ax.x * ri.x, ax.y * ri.y);
        *reinterpret_cast<double2*>(gy + o) = make_double2(ay.x * ri.x, ay.y * ri.y);
        *reinterpret_cast<double2*>(gz + o) = make_double2(az.x * ri.x, az.y * ri.y);
    }
}

template <int G>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_lap2(Geom g, const double* __restrict__ s, double* __restrict__ out) {
    const int lane = threadIdx.x & 31, warp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int c0 = warp * (32 / G) + lane / G, gl = lane & (G - 1), k0 = 2 * gl, nv = g.nv;
    const bool live = c0 < g.N;
    const int col = live ? c0 : g.N - 1;
    if (k0 >= nv) return;
    const int4 n03 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8));
    const int4 n47 = __ldg(reinterpret_cast<const int4*>(g.nbr + size_t(col) * 8) + 1);
    const int nb[6] = {n03.x, n03.y, n03.z, n03.w, n47.x, n47.y};
    const double2* wp = reinterpret_cast<const double2*>(g.wlap + size_t(col) * 8);
    const double2 w01 = __ldg(wp), w23 = __ldg(wp + 1), w45 = __ldg(wp + 2);
    const double w[6] = {w01.x, w01.y, w23.x, w23.y, w45.x, w45.y};
    const double2 s0 = __ldg(reinterpret_cast<const double2*>(s + size_t(col) * nv + k0));
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const double2 sj = __ldg(reinterpret_cast<const double2*>(s + size_t(nb[j]) * nv + k0));
        acc.x = fma(w[j], sj.x - s0.x, acc.x);
        acc.y = fma(w[j], sj.y - s0.y, acc.y);
    }
    const double2 ri = __ldg(reinterpret_cast<const double2*>(g.rinv + k0));
    if (live) *reinterpret_cast<double2*>(out + size_t(col) * nv + k0) = make_double2(acc.x * ri.x * ri.x, acc.y * ri.y * ri.y);
}

// ---------------------------------------------------------------------------------------------
// S1: stage preparation (column-local).  Fig. 6 large-step 4 of the previous stage and
// large-step 1 of this one:  Phi^[t] <- Phi^n (stage 1) or Phi^[t] + Phi* (stages 2, 3), the
// horizontal momentum kept as its two components in the column's tangent basis;
// h = Cp p/(Rd rho) (Eq. 38, G9), theta, 1/rho, the LU factors of the tridiagonal matrix of Eq. 37
// (g~ of Eq. 39 inside; coefficients: DESIGN.md "tridiagonal", R8) for this stage's substep length
// delta, and the initial deviations of Eq. 31 (R1: every stage starts from t_n).  The matrix does not
// change between the substeps of a stage, so it is factorised once here and the substeps only run
// the two sweeps.  Vertical operators: Eq. 8-9 with k = 1 on possibly non-uniform layers
// (Geom::wl, wh, idz).  Xw != null (NEXT-1 hyper-diffusion on): also w = W/I_h[rho] for its Laplacian.
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, THOR_KP_MINB)
k_stage_prepare(Geom g, double* __restrict__ S, int stage, double delta, Tune tn, double* __restrict__ Xw) {
    const Walk wk(tn);
    Map<G, E> L(wk.bid);
    if (wk.ahead_bid >= 0) {
        prefetch_block_rows<G, E>(S, wk.ahead_bid, F_RHON, stage == 1 ? 6 : 7);
#if THOR_GEOMPF
        prefetch_block_geom<G>(g.frame, wk.ahead_bid, 96);
#endif
        if (stage > 1) {
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAS, 2);   prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PS, 4);
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PT, 1);    prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAT, 5);
        }
    }
    constexpr int NVP = Map<G, E>::NVP;
    double* me = S + size_t(L.col) * Map<G, E>::REC + L.k0;
    const int nv = g.nv;
    const double gam = g.Cp / (g.Cp - g.Rd), kv = g.Rd / (g.Cp - g.Rd);
    bool real[E];
#pragma unroll
    for (int e = 0; e < E; ++e) real[e] = (L.k0 + e < nv) && (L.col < g.N);

    const Frame fr = ld_frame(g.frame, L.col);
    double rho[E], va[E], vb[E], W[E], p[E], d[E];
    if (stage == 1) {
        double Vx[E], Vy[E], Vz[E];
        ld_rw<E>(me + F_RHON * NVP, rho); ld_rw<E>(me + F_VXN * NVP, Vx); ld_rw<E>(me + F_VYN * NVP, Vy);
        ld_rw<E>(me + F_VZN * NVP, Vz);   ld_rw<E>(me + F_WN * NVP, W);   ld_rw<E>(me + F_PN * NVP, p);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            va[e] = Vx[e] * fr.e1.x + Vy[e] * fr.e1.y + Vz[e] * fr.e1.z;
            vb[e] = Vx[e] * fr.e2.x + Vy[e] * fr.e2.y + Vz[e] * fr.e2.z;
        }
    } else {
        auto add = [&](int ft, int fs, double (&out)[E]) {
            ld_rw<E>(me + ft * NVP, out); ld_rw<E>(me + fs * NVP, d);
#pragma unroll
            for (int e = 0; e < E; ++e) out[e] += d[e];
        };
        add(F_RHOT, F_RHOS, rho); add(F_WT, F_WS, W); add(F_PT, F_PS, p);
        add(F_VAT, F_VAS, va);    add(F_VBT, F_VBS, vb);
    }
#pragma unroll
    for (int e = 0; e < E; ++e)
        if (!real[e]) { rho[e] = 1.0; p[e] = g.p_ref; va[e] = vb[e] = W[e] = 0.0; }

    double h[E], th[E], rtt[E], ir[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        h[e] = g.Cp * p[e] / (g.Rd * rho[e]);
        rtt[e] = eos_rt(p[e], g.Rd, g.p_ref, 1.0 / gam);
        th[e] = rtt[e] / rho[e];
        ir[e] = 1.0 / rho[e];
    }
    // interface quantities on the lower interface of each layer
    double pb[E], rb[E], hb[E], hh[E], gt[E], rhoh[E], wl[E], wh[E], idz[E];
    below<G, E>(p, pb, L.gl, 0.0); below<G, E>(rho, rb, L.gl, 1.0); below<G, E>(h, hb, L.gl, 0.0);
    ld_nc<E>(g.wl + L.k0, wl); ld_nc<E>(g.wh + L.k0, wh); ld_nc<E>(g.idz + L.k0, idz);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        const bool in = k >= 1 && k < nv;                 // interior interface
        rhoh[e] = in ? wl[e] * rb[e] + wh[e] * rho[e] : 1.0;                      // I_h[rho]
        hh[e] = in ? wl[e] * hb[e] + wh[e] * h[e] : 0.0;                          // I_h[h]
        gt[e] = in ? ((p[e] - pb[e]) * idz[e]) / rhoh[e] : 0.0;                   // Eq. 39
    }
    double hhb[E], hha[E], gtb[E], gta[E], dlo[E], dhi[E], dlob[E], dhib[E];
    below<G, E>(hh, hhb, L.gl, 0.0); above<G, E>(hh, hha, L.gl, 0.0);
    below<G, E>(gt, gtb, L.gl, 0.0); above<G, E>(gt, gta, L.gl, 0.0);
    ld_nc<E>(g.dlo + L.k0, dlo); ld_nc<E>(g.dhi + L.k0, dhi);
    below<G, E>(dlo, dlob, L.gl, 0.0); below<G, E>(dhi, dhib, L.gl, 0.0);
    double ta[E], tb[E], tc[E];
    const double d2 = delta * delta, d2g = d2 * g.gravity;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        // hh, g~ are 0 on the lid and on the ground: a_1 and c_(nv-1) multiply the zero boundary values
        const double ck = d2 * kv * idz[e];
        tc[e] = -ck * (dhi[e] * hha[e] - 0.5 * gta[e]) - d2g * wh[e] * dhi[e];
        ta[e] = -ck * (dlob[e] * hhb[e] + 0.5 * gtb[e]) + d2g * wl[e] * dlob[e];
        tb[e] = 1.0 + ck * hh[e] * (dlo[e] + dhib[e]) - d2g * (wl[e] * dhib[e] - wh[e] * dlo[e]);
    }
    // Thomas forward elimination of the matrix (L339): b'_k = b_k - a_k c_(k-1)/b'_(k-1).  The leading
    // minors theta_k = b'_1 ... b'_k obey the LINEAR recurrence theta_k = b_k theta_(k-1) - a_k c_(k-1) theta_(k-2),
    // so the pivots come out of a scan of 2x2 matrices instead of a serial chain of divisions.  Scaled
    // by s_k = 1/b_k (t_k = theta_k s_1...s_k stays in (0, 1] for these diagonally dominant matrices, no
    // overflow at 128 layers):  t_k = t_(k-1) - beta_k t_(k-2),  beta_k = a_k s_k c_(k-1) s_(k-1),
    // 1/b'_k = s_k t_(k-1)/t_k.  fi = 1/b'_k, fa = a_k/b'_k, fc = c_k/b'_k; 0 on the ground, on pads and
    // in pad columns (identity maps in the scan).
    double fa[E], fi[E], fc[E];
    {
        bool in[E];
        double sk[E], cs[E], csb[E], beta[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = L.k0 + e;
            in[e] = k >= 1 && k < nv && L.col < g.N;
            sk[e] = in[e] ? 1.0 / tb[e] : 0.0;
            cs[e] = in[e] ? tc[e] * sk[e] : 0.0;
        }
        below<G, E>(cs, csb, L.gl, 0.0);
        double p00 = 1.0, p01 = 0.0, p10 = 0.0, p11 = 1.0;      // product of this lane's maps [[1, -beta], [1, 0]]
#pragma unroll
        for (int e = 0; e < E; ++e) {
            beta[e] = in[e] ? ta[e] * sk[e] * csb[e] : 0.0;
            if (in[e]) {
                const double n00 = fma(-beta[e], p10, p00), n01 = fma(-beta[e], p11, p01);
                p10 = p00; p11 = p01; p00 = n00; p01 = n01;
            }
        }
#pragma unroll
        for (int sft = 1; sft < G; sft <<= 1) {                   // Kogge-Stone: P_lane <- P_lane x P_(lane - sft)
            const double o00 = __shfl_up_sync(kFull, p00, sft, G), o01 = __shfl_up_sync(kFull, p01, sft, G);
            const double o10 = __shfl_up_sync(kFull, p10, sft, G), o11 = __shfl_up_sync(kFull, p11, sft, G);
            if (L.gl >= sft) {
                const double r00 = fma(p00, o00, p01 * o10), r01 = fma(p00, o01, p01 * o11);
                const double r10 = fma(p10, o00, p11 * o10), r11 = fma(p10, o01, p11 * o11);
                p00 = r00; p01 = r01; p10 = r10; p11 = r11;
            }
        }
        double t1 = __shfl_up_sync(kFull, p00, 1, G), t2 = __shfl_up_sync(kFull, p10, 1, G);   // t_(k0-1), t_(k0-2)
        if (L.gl == 0) { t1 = 1.0; t2 = 0.0; }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            fi[e] = 0.0;
            if (in[e]) {
                const double t0 = fma(-beta[e], t2, t1);
                fi[e] = sk[e] * t1 / t0;
                t2 = t1; t1 = t0;
            }
            fa[e] = ta[e] * fi[e];
            fc[e] = tc[e] * fi[e];
        }
    }
    st_row<E>(me + F_RHOT * NVP, rho); st_row<E>(me + F_IRT * NVP, ir);  st_row<E>(me + F_WT * NVP, W);
    st_row<E>(me + F_PT * NVP, p);     st_row<E>(me + F_VAT * NVP, va);  st_row<E>(me + F_VBT * NVP, vb);
    st_row<E>(me + F_H * NVP, h);      st_row<E>(me + F_TH * NVP, th);
    st_row<E>(me + F_FA * NVP, fa);    st_row<E>(me + F_FI * NVP, fi);   st_row<E>(me + F_FC * NVP, fc);
    if (Xw) {                                                    // NEXT-1: w on interior interfaces (0 elsewhere)
        if (g.kord == 3) interp_h3<G, E>(g.vk + L.k0, rho, rhoh, L.gl);   // RV2: I_h of the order of the run
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = L.k0 + e;
            d[e] = (k >= 1 && k < nv) ? W[e] / rhoh[e] : 0.0;
        }
        st_row<E>(Xw + size_t(L.col) * (size_t(XF) * NVP) + L.k0 + X_W * NVP, d);
    }

    // Eq. 31: Phi*(0) = Phi^n - Phi^[t]; (rho theta)*(0) = (rho theta)^n - (rho theta)^[t]
    if (stage == 1) {
        // Phi*(0) = 0 exactly: the six deviation rows are neither written here nor read by the stage's single
        // substep (V*' = delta slowV written by k_slow_terms / k_diff2 / k_momentum_dd_stage1; k_vertical with first = 2),
        // which overwrites all of them
        st_row<E>(me + F_RTN * NVP, rtt);
    } else {
        auto dev = [&](int fn, int fs, const double (&t)[E]) {
            ld_rw<E>(me + fn * NVP, d);
#pragma unroll
            for (int e = 0; e < E; ++e) d[e] = real[e] ? d[e] - t[e] : 0.0;
            st_row<E>(me + fs * NVP, d);
        };
        dev(F_RHON, F_RHOS, rho); dev(F_WN, F_WS, W); dev(F_PN, F_PS, p); dev(F_RTN, F_RTS, rtt);
        double dx[E], dy[E], dz[E];                             // V^n in the tangent basis, minus V^[t]
        ld_rw<E>(me + F_VXN * NVP, dx); ld_rw<E>(me + F_VYN * NVP, dy); ld_rw<E>(me + F_VZN * NVP, dz);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double an = dx[e] * fr.e1.x + dy[e] * fr.e1.y + dz[e] * fr.e1.z;
            const double bn = dx[e] * fr.e2.x + dy[e] * fr.e2.y + dz[e] * fr.e2.z;
            va[e] = real[e] ? an - va[e] : 0.0;
            vb[e] = real[e] ? bn - vb[e] : 0.0;
        }
        st_row<E>(me + F_VAS * NVP, va); st_row<E>(me + F_VBS * NVP, vb);
    }
}

// ---------------------------------------------------------------------------------------------
// S2: slow terms of the stage (Fig. 6 large-step 3; RHS of Eq. 32-35 and Eq. 42; O4 with R7).
// Gathers six rows from the column and its 6 neighbours: V^[t] (2 tangent components), theta, p^[t],
// 1/rho^[t], W^[t]; the neighbour's un-projected velocity u = (V + I_c[W] r)/rho (L268) is rebuilt
// from them with the neighbour's frame (staged in shared memory per column), h = Cp p/(Rd rho) likewise.
// The pressure gradient is accumulated directly in the column's tangent basis (wgrad2).
// HYP (NEXT-1 hyper-diffusion on, X != null): the same loop also forms the first Laplacians of
// rho, v = V/rho (Cartesian components), w and T (RD2) and stores them weighted for the second one.
// dd: 1 = also store D3^[t] = div_h V^[t] + D_c[W^[t]] (RD4); 2 (stage 1, where Phi^[t] = Phi^n) = and D3^n.
// delta1 > 0 (stage 1 of the base path): also the stage's explicit horizontal step, which with V*(0) = 0 and
// p*(0) = 0 is V*' = delta1 slowV (Eq. 33) -- the slow term is in registers here, so no k_momentum launch.
// ---------------------------------------------------------------------------------------------
// SH (NEXT-4, reading RS1): the shallow-atmosphere form -- the radii are already A in the per-layer tables; here the
// horizontal equation advects the horizontal velocity only, w = I_c[W]/rho is advected as a scalar into the vertical
// one, and Coriolis is f r x V with f = 2 Omega sin(lat) on the horizontal momentum alone.
template <int G, int E, bool HYP, bool K3, bool SH = false>
__device__ __forceinline__ void slow_terms_block(const Geom& g, double* __restrict__ S, const Tune& tn,
                                                 double* __restrict__ X, int dd, double delta1) {
    const Walk wk(tn);
    Map<G, E> L(wk.bid);
    if (wk.ahead_bid >= 0) {
        prefetch_block_rows<G, E>(S, wk.ahead_bid, F_TH, 1);   prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PT, 1);
        prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAT, 5);
#if THOR_GEOMPF
        prefetch_block_geom<G>(g.nbr, wk.ahead_bid, 32); prefetch_block_geom<G>(g.wdiv2, wk.ahead_bid, 128);
        prefetch_block_geom<G>(g.wgrad2, wk.ahead_bid, 96); prefetch_block_geom<G>(g.frame, wk.ahead_bid, 96);
        if (HYP) { prefetch_block_geom<G>(g.wlap, wk.ahead_bid, 64); prefetch_block_xrows<G, E>(X, wk.ahead_bid, X_W, 1); }
#endif
    }
    constexpr int NVP = Map<G, E>::NVP;
    constexpr size_t REC = Map<G, E>::REC, XREC = size_t(XF) * NVP;
    constexpr int CPB = kWarpsPerBlock * 32 / G;
    double* me = S + size_t(L.col) * REC + L.k0;
    const int nv = g.nv;
    const double kv = g.Rd / (g.Cp - g.Rd), cph = g.Cp / g.Rd;
    // per column group: 14 divergence weights (+2 pad), 12 gradient weights, the frames of the column and its
    // 6 neighbours (7 x 12), 6 Laplacian weights (+2 pad), 8 neighbour slots
    // The base kernel stages them in shared memory (registers are what limits it); the hyper-diffusion variant, which
    // is short of shared-memory bandwidth rather than registers, reads them straight from global memory -- L1 hits
    // after the first touch (measured: profiles/r02c_variants.md).
    const double *wdv, *wgv, *wlp, *frm;
    int nb[7];
    constexpr bool DIRECT = HYP;
    if constexpr (DIRECT) {
        (void)CPB;
        wdv = g.wdiv2 + size_t(L.col) * 16; wgv = g.wgrad2 + size_t(L.col) * 12; wlp = g.wlap + size_t(L.col) * 8;
        int n6[6];
        neighbours(g, L.col, n6);
        nb[0] = L.col;
#pragma unroll
        for (int j = 0; j < 6; ++j) nb[j + 1] = n6[j];
        frm = nullptr;
    } else {
        __shared__ double wsm[CPB][16 + 12 + 84 + 8];
        __shared__ int nsm[CPB][8];
        double* ws = wsm[threadIdx.x / G];
        int* nbs = nsm[threadIdx.x / G];
        stage_weights<G>(g.wdiv2 + size_t(L.col) * 16, ws, 8, L.gl);
        stage_weights<G>(g.wgrad2 + size_t(L.col) * 12, ws + 16, 6, L.gl);
        for (int i = L.gl; i < 8; i += G) nbs[i] = i == 0 ? L.col : __ldg(g.nbr + size_t(L.col) * 8 + i - 1);
        __syncwarp();
        for (int i = L.gl; i < 42; i += G)
            reinterpret_cast<double2*>(ws + 28)[i] = __ldg(reinterpret_cast<const double2*>(g.frame) + 6 * size_t(nbs[i / 6]) + i % 6);
#pragma unroll
        for (int j = 0; j < 7; ++j) nb[j] = nbs[j];
        wdv = ws; wgv = ws + 16; frm = ws + 28; wlp = ws + 112;
        __syncwarp();
    }
    auto frame_of = [&](int j) { return DIRECT ? g.frame + size_t(nb[j]) * 12 : frm + 12 * j; };

    double p0[E];
    double divV[E], divhV[E], divtV[E], Ax[E], Ay[E], Az[E], ga[E], gb[E];
    double Aw[SH ? E : 1];                                 // RS1 (iii): scalar advection of w
#pragma unroll
    for (int e = 0; e < E; ++e) divV[e] = divhV[e] = divtV[e] = Ax[e] = Ay[e] = Az[e] = ga[e] = gb[e] = 0.0;
    if constexpr (SH) {
#pragma unroll
        for (int e = 0; e < E; ++e) Aw[e] = 0.0;
    }
    // NEXT-1: first Laplacians sum_j wlap_j (s_j - s_0) of rho, v_x, v_y, v_z, w, T
    double s0[HYP ? 6 : 1][E], lp[HYP ? 6 : 1][E];
    if (HYP) {
#pragma unroll
        for (int f = 0; f < 6; ++f)
#pragma unroll
            for (int e = 0; e < E; ++e) lp[f][e] = 0.0;
    }
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const double* q = S + size_t(nb[j]) * REC + L.k0;
        const double wa = wdv[2 * j], wb = wdv[2 * j + 1];
        const double* f = frame_of(j);
        double a[E], b[E], tj[E], pj[E], irj[E], Wj[E], Wup[E];
        ld_nc<E>(q + F_VAT * NVP, a);  ld_nc<E>(q + F_VBT * NVP, b);  ld_nc<E>(q + F_TH * NVP, tj);
        ld_nc<E>(q + F_PT * NVP, pj);  ld_nc<E>(q + F_IRT * NVP, irj); ld_nc<E>(q + F_WT * NVP, Wj);
        if (K3) interp_c3<G, E>(g.vk + 512 + L.k0, Wj, Wup, L.gl);           // RV2: Wup holds I_c[W]_j itself
        else above<G, E>(Wj, Wup, L.gl, 0.0);
        if (j == 0) {
#pragma unroll
            for (int e = 0; e < E; ++e) p0[e] = pj[e];
        } else {
            const double g1 = wgv[2 * (j - 1)], g2 = wgv[2 * (j - 1) + 1];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const double dp = pj[e] - p0[e];
                ga[e] = fma(g1, dp, ga[e]); gb[e] = fma(g2, dp, gb[e]);
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = fma(wa, a[e], wb * b[e]);                        // w_j . V_j
            const double wc = K3 ? Wup[e] : 0.5 * (Wj[e] + Wup[e]);           // I_c[W]_j; the lid's W is the pad's 0
            const double t = d * irj[e];
            divV[e] += d;
            divhV[e] = fma(cph * pj[e] * irj[e], d, divhV[e]);                // h_j = Cp p_j/(Rd rho_j)
            divtV[e] = fma(tj[e], d, divtV[e]);
            if constexpr (SH) {                                                   // u_h,j (w_j . V_j) and w_j (w_j . V_j)
                Ax[e] = fma(fma(a[e], f[0], b[e] * f[3]), t, Ax[e]);
                Ay[e] = fma(fma(a[e], f[1], b[e] * f[4]), t, Ay[e]);
                Az[e] = fma(fma(a[e], f[2], b[e] * f[5]), t, Az[e]);
                Aw[e] = fma(wc, t, Aw[e]);
            } else {
            Ax[e] = fma(fma(a[e], f[0], fma(b[e], f[3], wc * f[6])), t, Ax[e]);   // u_j (w_j . V_j), u = (V + I_c[W] r)/rho
            Ay[e] = fma(fma(a[e], f[1], fma(b[e], f[4], wc * f[7])), t, Ay[e]);
            Az[e] = fma(fma(a[e], f[2], fma(b[e], f[5], wc * f[8])), t, Az[e]);
            }
        }
        if (HYP) {
            double rj[E], wj[E], sj[6][E];
            ld_nc<E>(q + F_RHOT * NVP, rj);
            ld_nc<E>(X + size_t(nb[j]) * XREC + L.k0 + X_W * NVP, wj);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                sj[0][e] = rj[e];
                sj[1][e] = fma(a[e], f[0], b[e] * f[3]) * irj[e];
                sj[2][e] = fma(a[e], f[1], b[e] * f[4]) * irj[e];
                sj[3][e] = fma(a[e], f[2], b[e] * f[5]) * irj[e];
                sj[4][e] = wj[e];
                sj[5][e] = pj[e] * irj[e] / g.Rd;
            }
            const double lw = j == 0 ? 0.0 : wlp[j - 1];
#pragma unroll
            for (int fi = 0; fi < 6; ++fi)
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    if (j == 0) s0[fi][e] = sj[fi][e];
                    else lp[fi][e] = fma(lw, sj[fi][e] - s0[fi][e], lp[fi][e]);
                }
        }
    }
    double ri[E], dlo[E], dhi[E], wl[E], wh[E], idz[E];
    ld_nc<E>(g.rinv + L.k0, ri); ld_nc<E>(g.dlo + L.k0, dlo); ld_nc<E>(g.dhi + L.k0, dhi);
    ld_nc<E>(g.wl + L.k0, wl);   ld_nc<E>(g.wh + L.k0, wh);   ld_nc<E>(g.idz + L.k0, idz);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        divV[e] *= ri[e]; divhV[e] *= ri[e]; divtV[e] *= ri[e];
        Ax[e] *= ri[e]; Ay[e] *= ri[e]; Az[e] *= ri[e];
        ga[e] *= ri[e]; gb[e] *= ri[e];
        if constexpr (SH) Aw[e] *= ri[e];
    }
    // the column's own rows again (L1 hits), one at a time
    double rho[E], W[E], Wup[E], a0[E], b0[E], ir0[E];
    ld_nc<E>(me + F_RHOT * NVP, rho);
    ld_again<E>(me + F_WT * NVP, W);
    above<G, E>(W, Wup, L.gl, 0.0);
    double Wc3[K3 ? E : 1];
    if constexpr (K3) interp_c3<G, E>(g.vk + 512 + L.k0, W, Wc3, L.gl);
    ld_again<E>(me + F_VAT * NVP, a0); ld_again<E>(me + F_VBT * NVP, b0); ld_again<E>(me + F_IRT * NVP, ir0);
    const double* f0 = frame_of(0);
    const double e1x = f0[0], e1y = f0[1], e1z = f0[2], e2x = f0[3], e2y = f0[4], e2z = f0[5];
    const double rx = f0[6], ry = f0[7], rz = f0[8];
    double Mx[E], My[E], Mz[E];                                              // full momentum M = V + I_c[W] r
#pragma unroll
    for (int e = 0; e < E; ++e) {
        double wc = 0.5 * (W[e] + Wup[e]);
        if constexpr (K3) wc = Wc3[e];
        if constexpr (SH) {                                  // the horizontal momentum alone (RS1 ii, iii)
            Mx[e] = fma(a0[e], e1x, b0[e] * e2x);
            My[e] = fma(a0[e], e1y, b0[e] * e2y);
            Mz[e] = fma(a0[e], e1z, b0[e] * e2z);
        } else {
        Mx[e] = fma(a0[e], e1x, fma(b0[e], e2x, wc * rx));
        My[e] = fma(a0[e], e1y, fma(b0[e], e2y, wc * ry));
        Mz[e] = fma(a0[e], e1z, fma(b0[e], e2z, wc * rz));
        }
    }

    // vertical flux divergences D_c[W I_h[q]] for q = u_x, u_y, u_z, h, theta, and D_c[W]
    double qb[E], Xf[E], Xup[E];
    auto vflux = [&](const double (&q)[E], double (&out)[E]) {
        if constexpr (K3) {
            interp_h3<G, E>(g.vk + L.k0, q, qb, L.gl);
#pragma unroll
            for (int e = 0; e < E; ++e) Xf[e] = W[e] * qb[e];
        } else {
            below<G, E>(q, qb, L.gl, 0.0);
#pragma unroll
            for (int e = 0; e < E; ++e) Xf[e] = W[e] * (wl[e] * qb[e] + wh[e] * q[e]);    // W = 0 on the ground and on the lid
        }
        above<G, E>(Xf, Xup, L.gl, 0.0);
#pragma unroll
        for (int e = 0; e < E; ++e) out[e] = dhi[e] * Xup[e] - dlo[e] * Xf[e];
    };
    double t[E], q0[E];
#pragma unroll
    for (int e = 0; e < E; ++e) q0[e] = Mx[e] * ir0[e];
    vflux(q0, t);
#pragma unroll
    for (int e = 0; e < E; ++e) { Ax[e] += t[e]; q0[e] = My[e] * ir0[e]; }
    vflux(q0, t);
#pragma unroll
    for (int e = 0; e < E; ++e) { Ay[e] += t[e]; q0[e] = Mz[e] * ir0[e]; }
    vflux(q0, t);
#pragma unroll
    for (int e = 0; e < E; ++e) { Az[e] += t[e]; q0[e] = cph * p0[e] * ir0[e]; }
    if constexpr (SH) {                                      // + D_c[W I_h[w]], w = I_c[W]/rho
        double qw[E];
#pragma unroll
        for (int e = 0; e < E; ++e) qw[e] = (K3 ? Wc3[K3 ? e : 0] : 0.5 * (W[e] + Wup[e])) * ir0[e];
        vflux(qw, t);
#pragma unroll
        for (int e = 0; e < E; ++e) Aw[e] += t[e];
    }
    double DhW[E], DtW[E], DW[E];
    vflux(q0, DhW);
    ld_again<E>(me + F_TH * NVP, q0); vflux(q0, DtW);
#pragma unroll
    for (int e = 0; e < E; ++e) DW[e] = dhi[e] * Wup[e] - dlo[e] * W[e];

    double sa[E], sb[E], Fr[E], srho[E], sp[E], srt[E];
    // g~ W on interfaces, then I_c
    double pb[E], rb[E], rhoh[E], Z[E], Zup[E];
    below<G, E>(p0, pb, L.gl, 0.0); below<G, E>(rho, rb, L.gl, 1.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        const bool in = k >= 1 && k < nv;
        rhoh[e] = in ? wl[e] * rb[e] + wh[e] * rho[e] : 1.0;
        Z[e] = in ? ((p0[e] - pb[e]) * idz[e]) / rhoh[e] * W[e] : 0.0;
    }
    above<G, E>(Z, Zup, L.gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const bool real = (L.k0 + e < nv) && (L.col < g.N);
        double Cx = -2.0 * g.omega * My[e], Cy = 2.0 * g.omega * Mx[e], Cz = 0.0;   // 2 Omega z x M
        if constexpr (SH) {                                                         // f r x V, f = 2 Omega sin(lat)
            const double fc = 2.0 * g.omega * rz;
            Cx = fc * (ry * Mz[e] - rz * My[e]); Cy = fc * (rz * Mx[e] - rx * Mz[e]); Cz = fc * (rx * My[e] - ry * Mx[e]);
        }
        const double Ar = Ax[e] * rx + Ay[e] * ry + Az[e] * rz;
        const double Cr = SH ? Cx * rx + Cy * ry + Cz * rz : Cx * rx + Cy * ry;
        if constexpr (SH) Fr[e] = Aw[e]; else Fr[e] = Ar + Cr;
        const double sx = -(Ax[e] - Ar * rx) - (Cx - Cr * rx);                      // Eq. 28 (G5)
        const double sy = -(Ay[e] - Ar * ry) - (Cy - Cr * ry);
        const double sz = -(Az[e] - Ar * rz) - (Cz - Cr * rz);
        sa[e] = real ? (sx * e1x + sy * e1y + sz * e1z) - ga[e] : 0.0;
        sb[e] = real ? (sx * e2x + sy * e2y + sz * e2z) - gb[e] : 0.0;
        srho[e] = real ? -divV[e] - DW[e] : 0.0;
        const double vgp = (a0[e] * ga[e] + b0[e] * gb[e]) * ir0[e];               // v_h . grad_h p
        sp[e] = real ? -kv * (divhV[e] + DhW[e] - vgp - 0.5 * (Z[e] + Zup[e])) : 0.0;
        srt[e] = real ? -divtV[e] - DtW[e] : 0.0;
    }
    double Frb[E], sW[E];
    if constexpr (K3) {                                      // RV2: I_h[rho] and I_h[F_r] of Eq. 42 at the order of the run
        interp_h3<G, E>(g.vk + L.k0, rho, rhoh, L.gl);       // (g~ above keeps the acoustic system's linear one)
        interp_h3<G, E>(g.vk + L.k0, Fr, Frb, L.gl);
    } else {
        below<G, E>(Fr, Frb, L.gl, 0.0);
#pragma unroll
        for (int e = 0; e < E; ++e) Frb[e] = wl[e] * Frb[e] + wh[e] * Fr[e];
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        sW[e] = (k >= 1 && k < nv && L.col < g.N)
                    ? -(p0[e] - pb[e]) * idz[e] - g.gravity * rhoh[e] - Frb[e]
                    : 0.0;                                                    // Eq. 42
    }
    st_row<E>(me + F_SVA * NVP, sa);    st_row<E>(me + F_SVB * NVP, sb);
    if (delta1 > 0.0) {
#pragma unroll
        for (int e = 0; e < E; ++e) { sa[e] *= delta1; sb[e] *= delta1; }
        st_row<E>(me + F_VAS * NVP, sa); st_row<E>(me + F_VBS * NVP, sb);
    }
    st_row<E>(me + F_SRHO * NVP, srho); st_row<E>(me + F_SW * NVP, sW); st_row<E>(me + F_SP * NVP, sp);
    st_row<E>(me + F_SRT * NVP, srt);
    if (dd) {                                                                 // NEXT-1 divergence damping (RD4)
        double* xe = X + size_t(L.col) * XREC + L.k0;
#pragma unroll
        for (int e = 0; e < E; ++e) t[e] = divV[e] + DW[e];
        st_row<E>(xe + X_D3T * NVP, t);
        if (dd == 2) st_row<E>(xe + X_D3N * NVP, t);
    }
    if (HYP) {                                                                // q = lap(rho) | rho lap(v_j) | rho_h lap(w) | rho lap(T)
        double* xe = X + size_t(L.col) * XREC + L.k0;
        double rhi[E];
        ld_nc<E>(g.rhinv + L.k0, rhi);
#pragma unroll
        for (int fi = 0; fi < 6; ++fi) {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int k = L.k0 + e;
                const double sc = fi == 4 ? rhi[e] * rhi[e] : ri[e] * ri[e];
                const double wgt = fi == 0 ? 1.0 : (fi == 4 ? rhoh[e] : rho[e]);
                t[e] = wgt * (lp[fi][e] * sc);
                if (fi == 4 && !(k >= 1 && k < nv)) t[e] = 0.0;
            }
            st_row<E>(xe + (X_Q0 + fi) * NVP, t);
        }
    }
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, THOR_KS_MINB)
k_slow_terms(Geom g, double* __restrict__ S, Tune tn, double* __restrict__ X, int dd, double delta1) {
    slow_terms_block<G, E, false, false>(g, S, tn, X, dd, delta1);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 3)
k_slow_terms_hyp(Geom g, double* __restrict__ S, Tune tn, double* __restrict__ X, int dd, double delta1) {
    slow_terms_block<G, E, true, false>(g, S, tn, X, dd, delta1);
}
// NEXT-4: the same two kernels in the shallow-atmosphere form (RS1; linear vertical interpolation only)
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 3)
k_slow_terms_sh(Geom g, double* __restrict__ S, Tune tn, double* __restrict__ X, int dd, double delta1) {
    slow_terms_block<G, E, false, false, true>(g, S, tn, X, dd, delta1);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 3)
k_slow_terms_hyp_sh(Geom g, double* __restrict__ S, Tune tn, double* __restrict__ X, int dd, double delta1) {
    slow_terms_block<G, E, true, false, true>(g, S, tn, X, dd, delta1);
}
// NEXT-3: the same two kernels with Eq. 8-9 of order 3 in the vertical interpolations (RV2)
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 3)
k_slow_terms_k3(Geom g, double* __restrict__ S, Tune tn, double* __restrict__ X, int dd, double delta1) {
    slow_terms_block<G, E, false, true>(g, S, tn, X, dd, delta1);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 3)
k_slow_terms_hyp_k3(Geom g, double* __restrict__ S, Tune tn, double* __restrict__ X, int dd, double delta1) {
    slow_terms_block<G, E, true, true>(g, S, tn, X, dd, delta1);
}

// ---------------------------------------------------------------------------------------------
// K1 (a4): explicit horizontal momentum, Eq. 33 (Fig. 6 small-step 2):
//   V*' = V* + delta (-grad_h p* / r + slowV).  Gathers p* from the 6 neighbours.
// ---------------------------------------------------------------------------------------------
// ZERO: the substep of stage 1, where V*(0) = 0 and p*(0) = 0 exactly (Eq. 31 with Phi^[t] = Phi^n): nothing of the
// deviation rows is read and there is no gradient to gather; V*' = delta slowV.
template <int G, int E, bool DD, bool ZERO = false>
__device__ __forceinline__ void momentum_block(const Geom& g, double* __restrict__ S, double delta, const Tune& tn,
                                               const double* __restrict__ Xdd, double Kd_div, int d3row) {
    const Walk wk(tn);
    Map<G, E> L(wk.bid);
    if (wk.ahead_bid >= 0) {
        if (!ZERO) {
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAS, 2);
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PS, 1);
        }
        prefetch_block_rows<G, E>(S, wk.ahead_bid, F_SVA, 2);
#if THOR_GEOMPF
        prefetch_block_geom<G>(g.nbr, wk.ahead_bid, 32); prefetch_block_geom<G>(g.wgrad2, wk.ahead_bid, 96);
        if (DD) {
            prefetch_block_geom<G>(g.dd_idx, wk.ahead_bid, 80); prefetch_block_geom<G>(g.dd_coef, wk.ahead_bid, 320);
            prefetch_block_xrows<G, E>(Xdd, wk.ahead_bid, d3row, 1);
        }
#endif
    }
    if (wk.in_tail) prefetch_block_rows<G, E>(S, wk.bid, F_H, F_PT - F_H + 1);   // the column-solve kernel starts here
    constexpr int NVP = Map<G, E>::NVP;
    constexpr size_t REC = Map<G, E>::REC;
    double* me = S + size_t(L.col) * REC + L.k0;
    // the 12 gradient weights are read straight from global memory where they are used: one 96-byte line per column,
    // L1 hits after the first touch, and nothing waits for them before the gathers can be issued
    const double* wgv = g.wgrad2 + size_t(L.col) * 12;
    int nb[6];
    neighbours(g, L.col, nb);
    double ga[E], gb[E], ri[E], va[E], vb[E], sa[E], sb[E];
#pragma unroll
    for (int e = 0; e < E; ++e) ga[e] = gb[e] = va[e] = vb[e] = 0.0;
    if constexpr (!ZERO) {
        double p0[E], pj[6][E];
        ld_nc<E>(me + F_PS * NVP, p0);
#pragma unroll
        for (int j = 0; j < 6; ++j) ld_nc<E>(S + size_t(nb[j]) * REC + L.k0 + F_PS * NVP, pj[j]);
        ld_rw<E>(me + F_VAS * NVP, va); ld_rw<E>(me + F_VBS * NVP, vb);
#pragma unroll
        for (int j = 0; j < 6; ++j) {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const double d = pj[j][e] - p0[e];
                ga[e] = fma(wgv[2 * j], d, ga[e]); gb[e] = fma(wgv[2 * j + 1], d, gb[e]);
            }
        }
    }
    ld_nc<E>(g.rinv + L.k0, ri);
    ld_nc<E>(me + F_SVA * NVP, sa); ld_nc<E>(me + F_SVB * NVP, sb);
    if constexpr (DD) {
        // NEXT-1, Fig. 6 small-step 1: divergence damping F_dd = -K_d lap(grad_h D3) (RD4) as ONE two-ring
        // stencil on the D3 row (composed on the host: thor_api.cu), already projected and in the tangent basis
        constexpr size_t XREC = size_t(XF) * NVP;
        const int* di = g.dd_idx + size_t(L.col) * 20;
        const double2* dc = reinterpret_cast<const double2*>(g.dd_coef + size_t(L.col) * 40);
        double d0[E], fa[E], fb[E];
        ld_nc<E>(Xdd + size_t(L.col) * XREC + L.k0 + d3row * NVP, d0);
#pragma unroll
        for (int e = 0; e < E; ++e) fa[e] = fb[e] = 0.0;
        // the 18 column indices up front (five 128-bit loads), then the D3 rows in batches of kDdBatch gathers that are
        // all requested before the first is used (measured: profiles/r02c_variants.md)
#ifndef THOR_DD_BATCH
#define THOR_DD_BATCH 18
#endif
        constexpr int kDdBatch = THOR_DD_BATCH;
        int mi[20];
#pragma unroll
        for (int q4 = 0; q4 < 5; ++q4) {
            const int4 t = __ldg(reinterpret_cast<const int4*>(di) + q4);
            mi[4 * q4] = t.x; mi[4 * q4 + 1] = t.y; mi[4 * q4 + 2] = t.z; mi[4 * q4 + 3] = t.w;
        }
#pragma unroll
        for (int q0 = 0; q0 < 18; q0 += kDdBatch) {
            double dm[kDdBatch][E];
#pragma unroll
            for (int b = 0; b < kDdBatch; ++b)
                if (q0 + b < 18) ld_nc<E>(Xdd + size_t(mi[q0 + b]) * XREC + L.k0 + d3row * NVP, dm[b]);
#pragma unroll
            for (int b = 0; b < kDdBatch; ++b) {
                if (q0 + b < 18) {
                    const double2 c = __ldg(dc + q0 + b);
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        const double dd = dm[b][e] - d0[e];
                        fa[e] = fma(c.x, dd, fa[e]); fb[e] = fma(c.y, dd, fb[e]);
                    }
                }
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double sc = -Kd_div * (ri[e] * ri[e] * ri[e]);
            sa[e] += sc * fa[e]; sb[e] += sc * fb[e];
        }
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        va[e] = fma(delta, sa[e] - ga[e] * ri[e], va[e]);
        vb[e] = fma(delta, sb[e] - gb[e] * ri[e], vb[e]);
    }
    st_row<E>(me + F_VAS * NVP, va); st_row<E>(me + F_VBS * NVP, vb);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_momentum(Geom g, double* __restrict__ S, double delta, Tune tn) {
    momentum_block<G, E, false>(g, S, delta, tn, nullptr, 0.0, 0);
}
// the same kernel with NEXT-1's divergence damping added to Eq. 33; d3row: the X row that holds the 3-D
// divergence of the current momentum (X_D3N in the first substep of a stage, where V^[t] + V*(0) = V^n; X_D3 after)
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 8)      // 64 registers, 8 blocks per SM: measured, profiles/r02c_variants.md
k_momentum_dd(Geom g, double* __restrict__ S, double delta, Tune tn, const double* __restrict__ Xdd, double Kd_div, int d3row) {
    momentum_block<G, E, true>(g, S, delta, tn, Xdd, Kd_div, d3row);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_momentum_dd_stage1(Geom g, double* __restrict__ S, double delta, Tune tn, const double* __restrict__ Xdd, double Kd_div, int d3row) {
    momentum_block<G, E, true, true>(g, S, delta, tn, Xdd, Kd_div, d3row);
}

// ---------------------------------------------------------------------------------------------
// K2 (a5-a9): horizontal divergences of the new momentum, the implicit vertical momentum
// (Eq. 37; two sweeps with the stage's LU factors), density (Eq. 32), rho*theta (Eq. 35, G7) and
// the pressure deviation (Eq. 36).  Fig. 6 small-steps 3-6.  Gathers V*', h, theta from the 6
// neighbours; everything else is column-local.  `first` = 1: p*(tau) is read (first substep of
// stages 2 and 3, p* = p^n - p^[t]); 2: the substep of stage 1, where every deviation is exactly 0 and
// no deviation row is read; 0: p* is re-evaluated from (rho theta)* exactly as the previous
// substep stored it, which saves one row of HBM reads.
//
// vertical_column is the work of one lane group on one column.  `own` points at row 0 (layer k0)
// of the column's own rows F_VAS..F_PT -- in global memory (k_vertical) or in the shared-memory
// stage a TMA bulk copy has filled (k_vertical_tma); neighbours are always gathered from global
// memory (L1/L2 hits).  wdv: the column's 21 divergence weights in shared memory.
// ---------------------------------------------------------------------------------------------
// DD (NEXT-1 with divergence damping on): also emit the 3-D divergence of the momentum this substep
// leaves, D3 = D3^[t] + div_h(V*')/r + D_c[W'], which the next substep's damping needs -- the two
// terms are already in registers here; xd points at row 0 (layer k0) of the column's X record.
template <int G, int E, bool DD = false>
__device__ __forceinline__ void vertical_column(const Geom& g, double* __restrict__ me, const double* own,
                                                const double* const (&nbp)[6], const double* wdv,
                                                int gl, int k0, double delta, int first, double* xd = nullptr) {
    constexpr int NVP = G * E;
    const double gam = g.Cp / (g.Cp - g.Rd), kv = g.Rd / (g.Cp - g.Rd);

    double divV[E], divhV[E], divtV[E], th0[E], h0[E];
    {
        double x[E], y[E];
        ld_rw<E>(own + F_VAS * NVP, x); ld_rw<E>(own + F_VBS * NVP, y);
        ld_rw<E>(own + F_H * NVP, h0);  ld_rw<E>(own + F_TH * NVP, th0);
        const double wa = wdv[0], wb = wdv[1];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = fma(wa, x[e], wb * y[e]);
            divV[e] = d; divhV[e] = h0[e] * d; divtV[e] = th0[e] * d;
        }
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const double* q = nbp[j];
        const double wa = wdv[2 * j + 2], wb = wdv[2 * j + 3];
        double x[E], y[E], hj[E], tj[E];
        ld_rw<E>(q + F_VAS * NVP, x); ld_rw<E>(q + F_VBS * NVP, y);
        ld_rw<E>(q + F_H * NVP, hj);  ld_rw<E>(q + F_TH * NVP, tj);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = fma(wa, x[e], wb * y[e]);
            divV[e] += d;
            divhV[e] = fma(hj[e], d, divhV[e]);
            divtV[e] = fma(tj[e], d, divtV[e]);
        }
    }
    double ri[E], dlo[E], dhi[E], wl[E], wh[E];
    ld_nc<E>(g.rinv + k0, ri); ld_nc<E>(g.dlo + k0, dlo); ld_nc<E>(g.dhi + k0, dhi);
    ld_nc<E>(g.wl + k0, wl);   ld_nc<E>(g.wh + k0, wh);

    double rho_s[E], p_s[E], W_s[E], rts[E], srho[E], sp[E], sW[E], srt[E], pt[E], irt[E];
    if (first == 2) {                     // stage 1: Phi*(0) = 0 exactly, the rows hold nothing yet
#pragma unroll
        for (int e = 0; e < E; ++e) rho_s[e] = W_s[e] = rts[e] = 0.0;
    } else {
        ld_rw<E>(own + F_RHOS * NVP, rho_s); ld_rw<E>(own + F_WS * NVP, W_s); ld_rw<E>(own + F_RTS * NVP, rts);
    }
    ld_rw<E>(own + F_SRHO * NVP, srho);  ld_rw<E>(own + F_SP * NVP, sp);  ld_rw<E>(own + F_SW * NVP, sW);
    ld_rw<E>(own + F_SRT * NVP, srt);    ld_rw<E>(own + F_PT * NVP, pt);
    {   // 1/(rho theta)^[t] from rows already here: h/theta = Cp p/(Rd rho theta)
        const double kap = g.Rd / g.Cp;
#pragma unroll
        for (int e = 0; e < E; ++e) irt[e] = kap * h0[e] / (th0[e] * pt[e]);
    }
    if (first == 2) {
#pragma unroll
        for (int e = 0; e < E; ++e) p_s[e] = 0.0;
    } else if (first) {
        ld_rw<E>(own + F_PS * NVP, p_s);
    } else {
#pragma unroll
        for (int e = 0; e < E; ++e) p_s[e] = eos_dev(rts[e] * irt[e], pt[e], gam, g);
    }
    double pq[E], rq[E], pqb[E], rqb[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double Srho = srho[e] - divV[e] * ri[e];                 // Eq. 41
        const double Sp = sp[e] - kv * divhV[e] * ri[e];               // Eq. 40 (G10)
        pq[e] = fma(delta, Sp, p_s[e]);
        rq[e] = fma(delta, Srho, rho_s[e]);
    }
    below<G, E>(pq, pqb, gl, 0.0); below<G, E>(rq, rqb, gl, 0.0);
    // right-hand side d_k on interior interfaces, already scaled by 1/b'_k (fi = 0 on the ground and on pads)
    double fa[E], fi[E], fc[E], A[E], B[E], zf[E], Wn[E];
    ld_rw<E>(own + F_FA * NVP, fa); ld_rw<E>(own + F_FI * NVP, fi); ld_rw<E>(own + F_FC * NVP, fc);
    {
        double idz[E];
        ld_nc<E>(g.idz + k0, idz);
#pragma unroll
        for (int e = 0; e < E; ++e) {     // G_h and I_h of Eq. 8-9 (k = 1) on the lower interface of layer k
            const double d = W_s[e] + delta * (sW[e] - idz[e] * (pq[e] - pqb[e]) - g.gravity * (wl[e] * rqb[e] + wh[e] * rq[e]));
            A[e] = -fa[e];            // z_k = d_k/b'_k - (a_k/b'_k) z_(k-1)
            B[e] = fi[e] * d;
        }
    }
    affine_scan<G, E, false>(A, B, zf, gl);
#pragma unroll
    for (int e = 0; e < E; ++e) A[e] = -fc[e];                          // x_k = z_k - c'_k x_(k+1)
    affine_scan<G, E, true>(A, zf, Wn, gl);

    double Wup[E], thb[E], X[E], Xup[E];
    above<G, E>(Wn, Wup, gl, 0.0);
    below<G, E>(th0, thb, gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) X[e] = (wl[e] * thb[e] + wh[e] * th0[e]) * Wn[e];  // I_h[theta] W'
    above<G, E>(X, Xup, gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        rho_s[e] = rq[e] - delta * (dhi[e] * Wup[e] - dlo[e] * Wn[e]);                               // Eq. 32
        rts[e] = rts[e] + delta * (srt[e] - divtV[e] * ri[e] - (dhi[e] * Xup[e] - dlo[e] * X[e]));  // Eq. 35
        p_s[e] = eos_dev(rts[e] * irt[e], pt[e], gam, g);                                            // Eq. 36
    }
    st_row<E>(me + F_WS * NVP, Wn);   st_row<E>(me + F_RHOS * NVP, rho_s);
    st_row<E>(me + F_RTS * NVP, rts); st_row<E>(me + F_PS * NVP, p_s);
    if constexpr (DD) {
        double d3[E];
        ld_nc<E>(xd + X_D3T * NVP, d3);
#pragma unroll
        for (int e = 0; e < E; ++e) d3[e] += divV[e] * ri[e] + (dhi[e] * Wup[e] - dlo[e] * Wn[e]);
        st_row<E>(xd + X_D3 * NVP, d3);
    }
}

template <int G, int E, bool DD>
__device__ __forceinline__ void vertical_block(const Geom& g, double* __restrict__ S, double delta, int first, const Tune& tn,
                                               double* __restrict__ Xdd) {
    const Walk wk(tn);
    Map<G, E> L(wk.bid);
    if (wk.ahead_bid >= 0) {                        // only the rows this launch reads (see `first`)
        prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAS, first == 1 ? F_PT + 1 : int(F_PS));
        if (first == 0) prefetch_block_rows<G, E>(S, wk.ahead_bid, F_RHOS, F_PT - F_RHOS + 1);
        if (first == 2) prefetch_block_rows<G, E>(S, wk.ahead_bid, F_SRHO, F_PT - F_SRHO + 1);
#if THOR_GEOMPF
        prefetch_block_geom<G>(g.nbr, wk.ahead_bid, 32); prefetch_block_geom<G>(g.wdiv2, wk.ahead_bid, 128);
        if (DD) prefetch_block_xrows<G, E>(Xdd, wk.ahead_bid, X_D3T, 1);
#endif
    }
    if (wk.in_tail) prefetch_block_rows<G, E>(S, wk.bid, F_SVA, 2);               // the next momentum kernel starts here
    const double* wdv = g.wdiv2 + size_t(L.col) * 16;      // read where used (one 128-byte line per column, L1 hits)
    int nb[6];
    neighbours(g, L.col, nb);
    constexpr size_t REC = Map<G, E>::REC;
    const double* const nbp[6] = {S + size_t(nb[0]) * REC + L.k0, S + size_t(nb[1]) * REC + L.k0, S + size_t(nb[2]) * REC + L.k0,
                                  S + size_t(nb[3]) * REC + L.k0, S + size_t(nb[4]) * REC + L.k0, S + size_t(nb[5]) * REC + L.k0};
    double* me = S + size_t(L.col) * REC + L.k0;
    if constexpr (DD)
        vertical_column<G, E, true>(g, me, me, nbp, wdv, L.gl, L.k0, delta, first, Xdd + size_t(L.col) * (size_t(XF) * Map<G, E>::NVP) + L.k0);
    else
        vertical_column<G, E>(g, me, me, nbp, wdv, L.gl, L.k0, delta, first);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, THOR_K2_MINB)
k_vertical(Geom g, double* __restrict__ S, double delta, int first, Tune tn) {
    vertical_block<G, E, false>(g, S, delta, first, tn, nullptr);
}
// the same kernel with NEXT-1's divergence damping on: also writes D3 for the next substep (vertical_column<.., DD>)
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_vertical_dd(Geom g, double* __restrict__ S, double delta, int first, Tune tn, double* __restrict__ Xdd) {
    vertical_block<G, E, true>(g, S, delta, first, tn, Xdd);
}

// ---------------------------------------------------------------------------------------------
// K2, TMA-staged (NOT the default: measured slower than the direct-load kernel, profiles/r01c_substep_kernels.md;
// selected with THOR_B200_TUNE tma_stages = 1 or 2 and kept as a tested variant): persistent blocks of kTmaWarps warps
// walk tiles of TCOL = kTmaWarps*32/G consecutive columns -- 2x2 / 2x4 / 4x4 patches of the rhombus
// lattice in the Morton device order.  EVERYTHING a tile reads is brought into shared memory by
// cp.async.bulk (TMA) and signalled through an mbarrier: the own rows F_VAS..F_PT of its columns
// (the contiguous head of each record), the gathered rows F_VAS..F_TH of its halo columns (host
// table TileTab::halo, <= hmax per tile), its divergence weights and its neighbour-slot table.
// HBM and L2 requests are therefore in flight without holding registers or stalling a warp, and the
// compute phase touches only shared memory; results go straight to global memory.
// ---------------------------------------------------------------------------------------------
constexpr int kTmaWarps = 4;
constexpr int kOwnRows = F_PT + 1;      // 16
constexpr int kHaloRows = F_TH + 1;     // 4

struct TileTab {
    const int* halo;              // [ntiles][hmax] device columns of the tile's halo (padded with the tile's first column)
    const unsigned char* slots;   // [Npad][8] per column: slot of each of the 6 neighbours (own: 0..TCOL-1, halo: TCOL + i), 2 pad
    int hmax;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return static_cast<unsigned>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <int G, int E, int NSTAGE>
__global__ void __launch_bounds__(kTmaWarps * 32)
k_vertical_staged(Geom g, TileTab tt, double* __restrict__ S, double delta, int first, int ntiles, int rev) {
    constexpr int NVP = G * E, CPW = 32 / G, TCOL = kTmaWarps * CPW;
    constexpr size_t REC = size_t(NF) * NVP;
    const int HM = tt.hmax;
    // one stage: own rows [TCOL][16][NVP] | halo rows [HM][4][NVP] | weights [TCOL][16] | slots [TCOL] x 8 bytes
    const int o_halo = TCOL * kOwnRows * NVP, o_w = o_halo + HM * kHaloRows * NVP, o_sl = o_w + TCOL * 16;
    const int stage_doubles = o_sl + TCOL;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage0 = reinterpret_cast<double*>(smem_raw);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(stage0 + size_t(NSTAGE) * stage_doubles);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int slot = warp * CPW + lane / G;       // column of the tile this lane group owns
    const int gl = lane & (G - 1), k0 = gl * E;
    const int my_tiles = (ntiles - int(blockIdx.x) + int(gridDim.x) - 1) / int(gridDim.x);
    auto tile_of = [&](int i) { const int t = int(blockIdx.x) + i * int(gridDim.x); return rev ? ntiles - 1 - t : t; };
    // producer: the first warp; lane 0 arms the barrier, then the lanes share the copies
    auto issue = [&](int i) {
        if (warp != 0) return;
        const int t = tile_of(i);
        double* st = stage0 + size_t(i % NSTAGE) * stage_doubles;
        unsigned long long* bar = full + i % NSTAGE;
        const unsigned row = NVP * 8u;
        if (lane == 0) {
            mbar_expect_tx(bar, TCOL * (first ? kOwnRows : kOwnRows - 1) * row + HM * kHaloRows * row + TCOL * 16 * 8u + TCOL * 8u);
            bulk_g2s(st + o_w, g.wdiv2 + size_t(t) * TCOL * 16, TCOL * 16 * 8u, bar);
            bulk_g2s(st + o_sl, tt.slots + size_t(t) * TCOL * 8, TCOL * 8u, bar);
        }
        __syncwarp();
        for (int c = lane; c < TCOL; c += 32) {
            const double* src = S + (size_t(t) * TCOL + c) * REC;
            double* dst = st + size_t(c) * kOwnRows * NVP;
            if (first) {
                bulk_g2s(dst, src, kOwnRows * row, bar);
            } else {                                     // skip the p* row: it is re-evaluated from (rho theta)*
                bulk_g2s(dst, src, F_PS * row, bar);
                bulk_g2s(dst + (F_PS + 1) * NVP, src + (F_PS + 1) * NVP, (kOwnRows - F_PS - 1) * row, bar);
            }
        }
        for (int h = lane; h < HM; h += 32) {
            const int c = __ldg(tt.halo + size_t(t) * HM + h);
            bulk_g2s(st + o_halo + size_t(h) * kHaloRows * NVP, S + size_t(c) * REC, kHaloRows * row, bar);
        }
    };
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) mbar_init(full + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    for (int i = 0; i < NSTAGE && i < my_tiles; ++i) issue(i);

    for (int i = 0; i < my_tiles; ++i) {
        const double* st = stage0 + size_t(i % NSTAGE) * stage_doubles;
        mbar_wait(full + i % NSTAGE, (i / NSTAGE) & 1);
        const uint2 sl = *reinterpret_cast<const uint2*>(st + o_sl + slot);
        auto row0 = [&](unsigned b) -> const double* {      // rows F_VAS.. of the column in slot b, at layer k0
            return b < unsigned(TCOL) ? st + size_t(b) * kOwnRows * NVP + k0
                                      : st + o_halo + size_t(b - TCOL) * kHaloRows * NVP + k0;
        };
        const double* const nbp[6] = {row0(sl.x & 255u), row0((sl.x >> 8) & 255u), row0((sl.x >> 16) & 255u),
                                      row0(sl.x >> 24),  row0(sl.y & 255u),        row0((sl.y >> 8) & 255u)};
        const int col = tile_of(i) * TCOL + slot;
        vertical_column<G, E>(g, S + size_t(col) * REC + k0, st + size_t(slot) * kOwnRows * NVP + k0, nbp,
                              st + o_w + slot * 16, gl, k0, delta, first);
        __syncthreads();                                  // every warp has read this stage
        if (i + NSTAGE < my_tiles) issue(i + NSTAGE);
    }
}

// ---------------------------------------------------------------------------------------------
// End of the large step: Phi^(n+1) = Phi^[t] + Phi* (Fig. 6 large-step 4), then the PROFX forcing
// (Eq. 51-52, backward Euler with the large step, R9).
// ---------------------------------------------------------------------------------------------
//
// FIX (NEXT-4, the energy fixer of L215, reading RE1): the step's dynamics are already in the Phi^n rows (a first
// k_finish launch without forcing put them there and the diagnostics kernels summed their mass and energy): bring
// the total energy back to its value before the step with ONE temperature increment for all cells,
// dT = (E - E')/(Cv M), rho unchanged, p <- p + rho Rd dT; then the forcing.  efix: device [M, E, M', E'].
template <int G, int E, bool FIX>
__device__ __forceinline__ void finish_block(const Geom& g, double* __restrict__ S, const Forcing& F, const HeldSuarez& H,
                                             const HotJupiter& J, double dt, const Tune& tn, const double* __restrict__ efix) {
    const Walk wk(tn);
    Map<G, E> L(wk.bid);
    if (wk.ahead_bid >= 0) {
        if (FIX) {
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_RHON, 4); prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PN, 1);
        } else {
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAS, 2);   prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PS, 4);
            prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PT, 1);    prefetch_block_rows<G, E>(S, wk.ahead_bid, F_VAT, 5);
        }
#if THOR_GEOMPF
        prefetch_block_geom<G>(g.frame, wk.ahead_bid, 96);
        if (!H.on && !J.on) {
            prefetch_block_table<G, E>(F.T_eq, wk.ahead_bid); prefetch_block_table<G, E>(F.k_T, wk.ahead_bid);
            prefetch_block_table<G, E>(F.k_v, wk.ahead_bid);
        }
#endif
    }
    constexpr int NVP = Map<G, E>::NVP;
    double* me = S + size_t(L.col) * Map<G, E>::REC + L.k0;
    const size_t to = size_t(L.col) * NVP + L.k0;
    double a[E], d[E], rho[E], p[E], vx[E], vy[E], vz[E];
    auto sum = [&](int ft, int fs, double (&out)[E]) {
        ld_rw<E>(me + ft * NVP, out); ld_rw<E>(me + fs * NVP, d);
#pragma unroll
        for (int e = 0; e < E; ++e) out[e] += d[e];
    };
    const Frame fr = ld_frame(g.frame, L.col);
    if constexpr (FIX) {
        ld_rw<E>(me + F_RHON * NVP, rho); ld_rw<E>(me + F_PN * NVP, p);
        ld_rw<E>(me + F_VXN * NVP, vx);   ld_rw<E>(me + F_VYN * NVP, vy); ld_rw<E>(me + F_VZN * NVP, vz);
        const double dT = (__ldg(efix + 1) - __ldg(efix + 3)) / ((g.Cp - g.Rd) * __ldg(efix + 2));
#pragma unroll
        for (int e = 0; e < E; ++e)
            if (L.k0 + e < g.nv && L.col < g.N) p[e] = p[e] + rho[e] * g.Rd * dT;
    } else {
        sum(F_RHOT, F_RHOS, rho); sum(F_PT, F_PS, p);
        double va[E], vb[E];
        sum(F_VAT, F_VAS, va); sum(F_VBT, F_VBS, vb);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            vx[e] = va[e] * fr.e1.x + vb[e] * fr.e2.x;
            vy[e] = va[e] * fr.e1.y + vb[e] * fr.e2.y;
            vz[e] = va[e] * fr.e1.z + vb[e] * fr.e2.z;
        }
        sum(F_WT, F_WS, a);
        st_row<E>(me + F_WN * NVP, a);
    }
    if (J.on) {
        // Eq. 59-61 (G15, RJ1): T_eq = T_vert(z) + beta_trop(sigma, z) dT_EP cos(lon) cos(lat); cos(lon) cos(lat) = x of the unit vector
        const double p0 = __shfl_sync(kFull, p[0], 0, G), rho0 = __shfl_sync(kFull, rho[0], 0, G);
        const double ps = p0 * exp(g.gravity * __ldg(g.zc) / (g.Rd * (p0 / (rho0 * g.Rd))));
        const double mu = fr.r.x, KT = 1.0 / J.tau_rad;
        double z[E];
        ld_nc<E>(g.zc + L.k0, z);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double sigma = p[e] / ps;
            double Tvert, beta = 0.0;
            if (z[e] <= J.z_stra) {
                const double hz = 0.5 * J.Gamma * (z[e] - J.z_stra);
                Tvert = J.T_surf - J.Gamma * (J.z_stra + 0.5 * (z[e] - J.z_stra)) + sqrt(hz * hz + J.dT_stra * J.dT_stra);
                if (sigma > J.sigma_stra) beta = sin(3.14159265358979323846 * (sigma - J.sigma_stra) / (2.0 * (1.0 - J.sigma_stra)));
            } else {
                Tvert = J.T_surf - J.Gamma * J.z_stra + J.dT_stra;
            }
            const double Teq = Tvert + beta * J.dT_EP * mu;
            double T = p[e] / (rho[e] * g.Rd);
            T = (T + KT * dt * Teq) / (1.0 + KT * dt);                        // Eq. 52
            p[e] = (L.k0 + e < g.nv && L.col < g.N) ? rho[e] * g.Rd * T : p[e];
        }
    } else if (H.on) {
        // sigma = p/p_s with the surface pressure extrapolated hydrostatically and isothermally from the lowest
        // layer centre (L390); K_v (Eq. 53), T_eq (Eq. 54, G14), K_T (Eq. 55, G14); then Eq. 51-52
        const double p0 = __shfl_sync(kFull, p[0], 0, G), rho0 = __shfl_sync(kFull, rho[0], 0, G);
        const double T0 = p0 / (rho0 * g.Rd);
        const double ps = p0 * exp(g.gravity * __ldg(g.zc) / (g.Rd * T0));
        const double sphi = fr.r.z, cphi2 = 1.0 - sphi * sphi, kappa = g.Rd / g.Cp;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double sigma = p[e] / ps;
            const double ramp = fmax(0.0, (sigma - H.sigma_b) / (1.0 - H.sigma_b));
            const double Kv = H.k_f * ramp;
            const double pr = p[e] / H.p_star;
            const double Teq = fmax(H.T_min, (H.T_surf - H.dT_y * sphi * sphi - H.dth_z * log(pr) * cphi2) * pow(pr, kappa));
            const double KT = H.k_a + (H.k_s - H.k_a) * ramp * cphi2 * cphi2;
            const double sv = 1.0 + Kv * dt;
            vx[e] /= sv; vy[e] /= sv; vz[e] /= sv;                            // Eq. 51
            double T = p[e] / (rho[e] * g.Rd);
            T = (T + KT * dt * Teq) / (1.0 + KT * dt);                        // Eq. 52
            p[e] = (L.k0 + e < g.nv && L.col < g.N) ? rho[e] * g.Rd * T : p[e];
        }
    } else if (F.k_v) {
        ld_nc<E>(F.k_v + to, a);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double s = 1.0 + a[e] * dt;
            vx[e] /= s; vy[e] /= s; vz[e] /= s;                               // Eq. 51
        }
    }
    if (!H.on && !J.on && F.k_T && F.T_eq) {
        double te[E];
        ld_nc<E>(F.k_T + to, a); ld_nc<E>(F.T_eq + to, te);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            double T = p[e] / (rho[e] * g.Rd);                                // Eq. 25
            T = (T + a[e] * dt * te[e]) / (1.0 + a[e] * dt);                  // Eq. 52
            p[e] = (L.k0 + e < g.nv && L.col < g.N) ? rho[e] * g.Rd * T : p[e];
        }
    }
    if (!FIX) st_row<E>(me + F_RHON * NVP, rho);
    st_row<E>(me + F_PN * NVP, p);
    st_row<E>(me + F_VXN * NVP, vx);   st_row<E>(me + F_VYN * NVP, vy); st_row<E>(me + F_VZN * NVP, vz);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_finish(Geom g, double* __restrict__ S, Forcing F, HeldSuarez H, HotJupiter J, double dt, Tune tn) {
    finish_block<G, E, false>(g, S, F, H, J, dt, tn, nullptr);
}
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_finish_fix(Geom g, double* __restrict__ S, Forcing F, HeldSuarez H, HotJupiter J, double dt, Tune tn,
             const double* __restrict__ efix) {
    finish_block<G, E, true>(g, S, F, H, J, dt, tn, efix);
}

// Deterministic sum of the per-column partials of k_diag (device order; one block): Neumaier-compensated partial
// sums per thread over a strided range, then a fixed tree in shared memory.  out[0] = mass, out[1] = energy.
__global__ void __launch_bounds__(1024)
k_sum_columns(int N, const double* __restrict__ col_mass, const double* __restrict__ col_energy, double* __restrict__ out) {
    __shared__ double sm[1024], se[1024];
    double m = 0.0, cm = 0.0, en = 0.0, ce = 0.0;
    for (int i = threadIdx.x; i < N; i += 1024) {
        const double x = col_mass[i], y = col_energy[i];
        double t = m + x;
        cm += (fabs(m) >= fabs(x)) ? (m - t) + x : (x - t) + m;
        m = t;
        t = en + y;
        ce += (fabs(en) >= fabs(y)) ? (en - t) + y : (y - t) + en;
        en = t;
    }
    sm[threadIdx.x] = m + cm; se[threadIdx.x] = en + ce;
    __syncthreads();
    for (int s = 512; s >= 1; s >>= 1) {
        if (threadIdx.x < s) { sm[threadIdx.x] += sm[threadIdx.x + s]; se[threadIdx.x] += se[threadIdx.x + s]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sm[0]; out[1] = se[0]; }
}

// ---------------------------------------------------------------------------------------------
// NEXT-1 (section 4 of the paper, Eq. 43-50; readings RD1-RD5 of DESIGN.md): explicit fourth-order
// hyper-diffusion of rho, v_h (Cartesian components), v_r and T per Runge-Kutta stage, and the 3-D
// divergence damping per acoustic substep.  Every nabla_h^2 is the 7-point stencil of L369-L371
// (Geom::wlap).  Work rows live in a second slab X[column][XF][layer], allocated only when a
// diffusion coefficient is set.  The first Laplacians are formed inside the slow-term kernel's gather
// loop (k_slow_terms_hyp), w by the stage-preparation kernel, D3^[t] by the slow-term kernel, D3 per
// substep by the column-solve kernel: the only extra launch per stage is k_diff2 below.
// ---------------------------------------------------------------------------------------------

template <int G, int E>
__device__ __forceinline__ void lap_gather(const double* base, size_t stride, const int (&nb)[6], const double (&w)[6],
                                           int self, int k0, double (&out)[E]) {   // sum_j w_j (s_j - s_self), unit sphere
    double s0[E];
    ld_nc<E>(base + size_t(self) * stride + k0, s0);
#pragma unroll
    for (int e = 0; e < E; ++e) out[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        double sj[E];
        ld_nc<E>(base + size_t(nb[j]) * stride + k0, sj);
#pragma unroll
        for (int e = 0; e < E; ++e) out[e] = fma(w[j], sj[e] - s0[e], out[e]);
    }
}
__device__ __forceinline__ void ld_lap_weights(const Geom& g, int col, int (&nb)[6], double (&w)[6]) {
    neighbours(g, col, nb);
    const double2* wp = reinterpret_cast<const double2*>(g.wlap + size_t(col) * 8);
    const double2 a = __ldg(wp), b = __ldg(wp + 1), c = __ldg(wp + 2);
    w[0] = a.x; w[1] = a.y; w[2] = b.x; w[3] = b.y; w[4] = c.x; w[5] = c.y;
}

// second Laplacian; the fluxes are added to the slow terms of the stage (RD2, RD3); delta1: as in k_slow_terms
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 5)      // 5 blocks per SM: measured, profiles/r02c_variants.md
k_diff2(Geom g, double* __restrict__ S, const double* __restrict__ X, double Kd, Tune tn, double delta1) {
    const Walk wk(tn);
    Map<G, E> L(wk.bid);
    if (wk.ahead_bid >= 0) {
        prefetch_block_rows<G, E>(S, wk.ahead_bid, F_SRHO, 4); prefetch_block_rows<G, E>(S, wk.ahead_bid, F_PT, 3);
#if THOR_GEOMPF
        prefetch_block_geom<G>(g.nbr, wk.ahead_bid, 32); prefetch_block_geom<G>(g.wlap, wk.ahead_bid, 64);
        prefetch_block_geom<G>(g.frame, wk.ahead_bid, 96); prefetch_block_xrows<G, E>(X, wk.ahead_bid, X_Q0, 6);
#endif
    }
    constexpr int NVP = Map<G, E>::NVP;
    constexpr size_t REC = Map<G, E>::REC, XREC = size_t(XF) * NVP;
    int nb[6]; double w[6];
    ld_lap_weights(g, L.col, nb, w);
    double* me = S + size_t(L.col) * REC + L.k0;
    const double gam = g.Cp / (g.Cp - g.Rd);
    double ri[E], rhi[E], q[E], t[E];
    ld_nc<E>(g.rinv + L.k0, ri); ld_nc<E>(g.rhinv + L.k0, rhi);
    auto real = [&](int e) { return (L.k0 + e < g.nv) && (L.col < g.N); };
    // density
    lap_gather<G, E>(X + X_Q0 * NVP, XREC, nb, w, L.col, L.k0, q);
    ld_rw<E>(me + F_SRHO * NVP, t);
#pragma unroll
    for (int e = 0; e < E; ++e) t[e] = real(e) ? t[e] + (-Kd * (q[e] * ri[e] * ri[e])) : 0.0;
    st_row<E>(me + F_SRHO * NVP, t);
    // horizontal momentum: Cartesian flux, Eq. 28, tangent components
    double Fx[E], Fy[E], Fz[E];
    lap_gather<G, E>(X + X_Q1 * NVP, XREC, nb, w, L.col, L.k0, Fx);
    lap_gather<G, E>(X + X_Q2 * NVP, XREC, nb, w, L.col, L.k0, Fy);
    lap_gather<G, E>(X + X_Q3 * NVP, XREC, nb, w, L.col, L.k0, Fz);
    const Frame fr = ld_frame(g.frame, L.col);
    double sa[E], sb[E];
    ld_rw<E>(me + F_SVA * NVP, sa); ld_rw<E>(me + F_SVB * NVP, sb);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double s2 = ri[e] * ri[e];
        double fx = -Kd * (Fx[e] * s2), fy = -Kd * (Fy[e] * s2), fz = -Kd * (Fz[e] * s2);
        const double frr = fx * fr.r.x + fy * fr.r.y + fz * fr.r.z;
        fx -= frr * fr.r.x; fy -= frr * fr.r.y; fz -= frr * fr.r.z;
        sa[e] = real(e) ? sa[e] + (fx * fr.e1.x + fy * fr.e1.y + fz * fr.e1.z) : 0.0;
        sb[e] = real(e) ? sb[e] + (fx * fr.e2.x + fy * fr.e2.y + fz * fr.e2.z) : 0.0;
    }
    st_row<E>(me + F_SVA * NVP, sa); st_row<E>(me + F_SVB * NVP, sb);
    if (delta1 > 0.0) {                              // stage 1 without divergence damping: V*' = delta1 slowV (see k_slow_terms)
#pragma unroll
        for (int e = 0; e < E; ++e) { sa[e] *= delta1; sb[e] *= delta1; }
        st_row<E>(me + F_VAS * NVP, sa); st_row<E>(me + F_VBS * NVP, sb);
    }
    // vertical momentum on interior interfaces
    lap_gather<G, E>(X + X_Q4 * NVP, XREC, nb, w, L.col, L.k0, q);
    ld_rw<E>(me + F_SW * NVP, t);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        t[e] = (k >= 1 && k < g.nv && L.col < g.N) ? t[e] + (-Kd * (q[e] * rhi[e] * rhi[e])) : 0.0;
    }
    st_row<E>(me + F_SW * NVP, t);
    // pressure and, through Eq. 24, rho*theta
    lap_gather<G, E>(X + X_Q5 * NVP, XREC, nb, w, L.col, L.k0, q);
    double p[E], u[E];
    ld_nc<E>(me + F_PT * NVP, p);
    ld_rw<E>(me + F_SP * NVP, t); ld_rw<E>(me + F_SRT * NVP, u);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double Fp = -g.Rd * Kd * (q[e] * ri[e] * ri[e]);
        t[e] = real(e) ? t[e] + Fp : 0.0;
        u[e] = real(e) ? u[e] + Fp * eos_rt(p[e], g.Rd, g.p_ref, 1.0 / gam) / (gam * p[e]) : 0.0;
    }
    st_row<E>(me + F_SP * NVP, t); st_row<E>(me + F_SRT * NVP, u);
}

// ---------------------------------------------------------------------------------------------
// Diagnostics (a12, R10): per-column partial sums of mass and energy; the host finishes the sum.
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_diag(Geom g, const double* __restrict__ S, double* __restrict__ col_mass, double* __restrict__ col_energy) {
    Map<G, E> L;
    constexpr int NVP = Map<G, E>::NVP;
    const double* me = S + size_t(L.col) * Map<G, E>::REC + L.k0;
    const double Cv = g.Cp - g.Rd;
    double rho[E], Vx[E], Vy[E], Vz[E], W[E], Wup[E], p[E], vol[E], zc[E];
    ld_nc<E>(me + F_RHON * NVP, rho); ld_nc<E>(me + F_VXN * NVP, Vx); ld_nc<E>(me + F_VYN * NVP, Vy);
    ld_nc<E>(me + F_VZN * NVP, Vz);   ld_nc<E>(me + F_WN * NVP, W);   ld_nc<E>(me + F_PN * NVP, p);
    ld_nc<E>(g.vol + L.k0, vol);      ld_nc<E>(g.zc + L.k0, zc);
    above<G, E>(W, Wup, L.gl, 0.0);
    double m = 0.0, en = 0.0;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        if (L.k0 + e < g.nv) {
            const double wc = 0.5 * (W[e] + Wup[e]);
            const double ke = 0.5 * (Vx[e] * Vx[e] + Vy[e] * Vy[e] + Vz[e] * Vz[e] + wc * wc) / rho[e];
            m += rho[e] * vol[e];
            en += (Cv * p[e] / g.Rd + ke + rho[e] * g.gravity * zc[e]) * vol[e];
        }
    }
#pragma unroll
    for (int s = G / 2; s >= 1; s >>= 1) {
        m += __shfl_xor_sync(kFull, m, s, G);
        en += __shfl_xor_sync(kFull, en, s, G);
    }
    if (L.col < g.N && L.gl == 0) {
        const double a = __ldg(g.area + L.col);
        col_mass[L.col] = m * a;
        col_energy[L.col] = en * a;
    }
}

// ---------------------------------------------------------------------------------------------
// NEXT-3: one step of the spring dynamics of the grid generator (Eq. 10-12) for all points at once
// (Jacobi: new positions from the old ones), one thread per point.  x, xn: [N][3] unit vectors; v: [N][3] velocities
// (tangent); the twelve pentagon centres stay fixed (L109).  worst: the largest displacement of the step as the bit
// pattern of a non-negative double (atomicMax on the integer order, which is the same).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
k_spring_step(int N, const double* __restrict__ x, double* __restrict__ xn, double* __restrict__ v,
              const int* __restrict__ nbr, const int* __restrict__ deg, double dspr, double kspr, double alpha, double dt,
              unsigned long long* __restrict__ worst) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double moved = 0.0;
    if (i < N) {
        const double px = x[3 * i], py = x[3 * i + 1], pz = x[3 * i + 2];
        if (deg[i] == 5) {
            xn[3 * i] = px; xn[3 * i + 1] = py; xn[3 * i + 2] = pz;
        } else {
            double fx = 0.0, fy = 0.0, fz = 0.0;
            for (int k = 0; k < 6; ++k) {
                const int j = nbr[size_t(i) * 6 + k];
                const double qx = x[3 * j], qy = x[3 * j + 1], qz = x[3 * j + 2];
                const double cx = py * qz - pz * qy, cy = pz * qx - px * qz, cz = px * qy - py * qx;
                const double dt0 = qx * px + qy * py + qz * pz;
                const double d = atan2(sqrt(cx * cx + cy * cy + cz * cz), dt0);             // geodesic distance
                double ex = qx - dt0 * px, ey = qy - dt0 * py, ez = qz - dt0 * pz;           // tangent at P_0 towards P_j
                const double inv = 1.0 / sqrt(ex * ex + ey * ey + ez * ez);
                const double a = kspr * (d - dspr) * inv;
                fx += a * ex; fy += a * ey; fz += a * ez;
            }
            double vx = v[3 * i], vy = v[3 * i + 1], vz = v[3 * i + 2];
            fx -= alpha * vx; fy -= alpha * vy; fz -= alpha * vz;                           // Eq. 10
            vx += dt * fx; vy += dt * fy; vz += dt * fz;
            double nx = px + dt * vx, ny = py + dt * vy, nz = pz + dt * vz;                  // Eq. 11, back onto the sphere
            const double in = 1.0 / sqrt(nx * nx + ny * ny + nz * nz);
            nx *= in; ny *= in; nz *= in;
            const double vr = vx * nx + vy * ny + vz * nz;
            v[3 * i] = vx - vr * nx; v[3 * i + 1] = vy - vr * ny; v[3 * i + 2] = vz - vr * nz;
            xn[3 * i] = nx; xn[3 * i + 1] = ny; xn[3 * i + 2] = nz;
            const double mx = nx - px, my = ny - py, mz = nz - pz;
            moved = sqrt(mx * mx + my * my + mz * mz);
        }
    }
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) moved = fmax(moved, __shfl_xor_sync(kFull, moved, s));
    if ((threadIdx.x & 31) == 0 && moved > 0.0) atomicMax(worst, static_cast<unsigned long long>(__double_as_longlong(moved)));
}

// ---------------------------------------------------------------------------------------------
// Canonical (host order, as uploaded) <-> device rows.  One thread per (device column, layer).
//   rows:   dst[d*dst_col + k] for d < Npad, k < NVP  (a record row: dst_col = NF*NVP; a table: NVP)
//   canon:  src[order[d]*row_len + k*cs + c0]         (real columns and layers only; pads get `pad`)
// ---------------------------------------------------------------------------------------------
__global__ void k_rows_from_canonical(int N, int Npad, int nv, int NVP, const int* __restrict__ order,
                                      const double* __restrict__ src, int row_len, int cs, int c0,
                                      double* __restrict__ dst, size_t dst_col, double pad, int zero_k0) {
    const size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= size_t(Npad) * NVP) return;
    const int d = int(i / NVP), k = int(i % NVP);
    double v = pad;
    if (d < N && k < nv) v = (zero_k0 && k == 0) ? 0.0 : src[size_t(order[d]) * row_len + size_t(k) * cs + c0];
    dst[size_t(d) * dst_col + k] = v;
}
__global__ void k_rows_to_canonical(int N, int nv, int NVP, const int* __restrict__ order,
                                    const double* __restrict__ src, size_t src_col,
                                    int row_len, int cs, int c0, double* __restrict__ dst) {
    const size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= size_t(N) * nv) return;
    const int d = int(i / nv), k = int(i % nv);
    dst[size_t(order[d]) * row_len + size_t(k) * cs + c0] = src[size_t(d) * src_col + k];
}
// plain [N][nv] arrays in canonical <-> device column order (config-1 host wrappers)
__global__ void k_gather_rows(int N, int nv, const int* __restrict__ order, const double* __restrict__ in,
                              int row_len, int cs, int c0, double* __restrict__ out) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= size_t(N) * nv) return;
    const int d = int(i / nv), k = int(i % nv);
    out[i] = in[size_t(order[d]) * row_len + size_t(k) * cs + c0];
}
__global__ void k_scatter_rows(int N, int nv, const int* __restrict__ order, const double* __restrict__ in,
                               int row_len, int cs, int c0, double* __restrict__ out) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= size_t(N) * nv) return;
    const int d = int(i / nv), k = int(i % nv);
    out[size_t(order[d]) * row_len + size_t(k) * cs + c0] = in[i];
}
__global__ void k_fill(size_t n, double* p, double v) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

}  // namespace thor
