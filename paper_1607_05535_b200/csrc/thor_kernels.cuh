// sm_100a kernels of the THOR HE-VI large step (Fig. 6).
//
// Data layout: every field is its own [column][layer] FP64 array, layer
// fastest, columns in the locality-preserving device order.  A column is owned by a group of G
// lanes (G = 8, 16 or 32); each lane holds E consecutive layers (layer = lane_in_group*E + e), so a
// neighbour-column read is one contiguous row (256 B at 32 layers, 512 B at 64) and vertical
// neighbours are either in the same lane or one shuffle away.  W (= rho v_r) is stored on the LOWER
// interface of each layer (slot 0 = ground = 0; the lid above the top layer is an implicit 0), so
// every array has the same stride.
//
// The path is an HBM-bound 7-point gather plus a per-column recurrence: no tensor cores.
#pragma once
#include <cuda_runtime.h>

namespace thor {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kWarpsPerBlock = 8;

struct Geom {                 // device pointers, device column order
    int N, nv;
    const int* nbr;           // [N][6]
    const double* wdiv;       // [N][7][3]
    const double* wgrad;      // [N][6][3]
    const double* rhat;       // [N][3]
    const double* area;       // [N]
    const double* rinv;       // [nv]
    const double* dlo;        // [nv]
    const double* dhi;        // [nv]
    const double* vol;        // [nv]
    const double* zc;         // [nv]
    double dz, omega, gravity, Rd, Cp, p_ref;
};

struct Fields {               // device pointers, each [N][nv]
    // Phi^n (the prognostic state between large steps)
    double *rho_n, *Vx_n, *Vy_n, *Vz_n, *W_n, *p_n, *rt_n;
    // Phi^[t] (reference state of the current Runge-Kutta stage, R1)
    double *rho_t, *Vx_t, *Vy_t, *Vz_t, *W_t, *p_t;
    // stage coefficients (Eq. 38-39) and the factorised tridiagonal matrix of Eq. 37
    double *h, *th, *ux, *uy, *uz, *fa, *fi, *fc;
    // slow terms (RHS of Eq. 32-35, Eq. 42)
    double *sVx, *sVy, *sVz, *srho, *sW, *sp, *srt;
    // deviations Phi* (Eq. 31) and the full rho*theta
    double *rho_s, *Vx_s, *Vy_s, *Vz_s, *W_s, *p_s, *rt;
    // forcing tables (Eq. 51-52), may be null
    const double *T_eq, *k_T, *k_v;
};

// ---------------------------------------------------------------------------------------------
// lane <-> (column, layer) mapping and vertical neighbour access
// ---------------------------------------------------------------------------------------------
template <int G, int E>
struct Lanes {
    int col;        // device column (clamped to N-1 so that every lane takes part in the shuffles)
    bool live;      // col < N
    int gl;         // lane within the group
    int k0;         // first layer of this lane
    __device__ Lanes(int N) {
        const int lane = threadIdx.x & 31;
        const int warp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
        const int c = warp * (32 / G) + lane / G;
        live = c < N;
        col = live ? c : N - 1;
        gl = lane & (G - 1);
        k0 = gl * E;
    }
};

// value at layer k-1 (fill at the bottom)
template <int G, int E>
__device__ __forceinline__ void below(const double (&v)[E], double (&out)[E], int gl, double fill) {
    double prev = __shfl_up_sync(kFull, v[E - 1], 1, G);
    if (gl == 0) prev = fill;
    out[0] = prev;
#pragma unroll
    for (int e = 1; e < E; ++e) out[e] = v[e - 1];
}
// value at layer k+1 (fill above the last lane; masked layers must already hold the fill value)
template <int G, int E>
__device__ __forceinline__ void above(const double (&v)[E], double (&out)[E], int gl, double fill) {
    double next = __shfl_down_sync(kFull, v[0], 1, G);
    if (gl == G - 1) next = fill;
#pragma unroll
    for (int e = 0; e < E - 1; ++e) out[e] = v[e + 1];
    out[E - 1] = next;
}

template <int E>
__device__ __forceinline__ void load_row(const double* __restrict__ base, int k0, int nv, double (&v)[E]) {
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = (k0 + e < nv) ? __ldg(base + k0 + e) : 0.0;
}
template <int E>
__device__ __forceinline__ void load_row_rw(const double* base, int k0, int nv, double (&v)[E]) {
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = (k0 + e < nv) ? base[k0 + e] : 0.0;
}
template <int E>
__device__ __forceinline__ void store_row(double* base, int k0, int nv, bool live, const double (&v)[E]) {
#pragma unroll
    for (int e = 0; e < E; ++e)
        if (live && k0 + e < nv) base[k0 + e] = v[e];
}

// Eq. 24 (L210) and its inverse
__device__ __forceinline__ double eos_p(double rt, double Rd, double p_ref, double gam) {
    return p_ref * pow(Rd * rt / p_ref, gam);
}
__device__ __forceinline__ double eos_rt(double p, double Rd, double p_ref, double inv_gam) {
    return p_ref / Rd * pow(p / p_ref, inv_gam);
}

// ---------------------------------------------------------------------------------------------
// Inclusive scan of the affine recurrence y_k = A_k y_(k-1) + B_k over the layers of a column
// (y_(-1) = 0), upward (DOWN = false) or x_k = A_k x_(k+1) + B_k downward (DOWN = true).
// Work-efficient inside a lane (E serial steps), Kogge-Stone across the G lanes.
// ---------------------------------------------------------------------------------------------
template <int G, int E, bool DOWN>
__device__ __forceinline__ void affine_scan(const double (&A)[E], const double (&B)[E], double (&y)[E], int gl) {
    // compose this lane's E maps into one: y_out = a * y_in + b
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
    // carry entering this lane = inclusive result of the previous lane
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
// Config-1 operators (Eq. 6 and Eq. 7), one row per (column, lane group)
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_div(Geom g, const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
      double* __restrict__ out) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const double* w = g.wdiv + size_t(L.col) * 21;
    double acc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const int c = j == 0 ? L.col : __ldg(g.nbr + size_t(L.col) * 6 + j - 1);
        const double wx = __ldg(w + 3 * j), wy = __ldg(w + 3 * j + 1), wz = __ldg(w + 3 * j + 2);
        double x[E], y[E], z[E];
        load_row<E>(vx + size_t(c) * nv, L.k0, nv, x);
        load_row<E>(vy + size_t(c) * nv, L.k0, nv, y);
        load_row<E>(vz + size_t(c) * nv, L.k0, nv, z);
#pragma unroll
        for (int e = 0; e < E; ++e) acc[e] = fma(wx, x[e], fma(wy, y[e], fma(wz, z[e], acc[e])));
    }
    double ri[E];
    load_row<E>(g.rinv, L.k0, nv, ri);
#pragma unroll
    for (int e = 0; e < E; ++e) acc[e] *= ri[e];
    store_row<E>(out + size_t(L.col) * nv, L.k0, nv, L.live, acc);
}

template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_grad(Geom g, const double* __restrict__ s, double* __restrict__ gx, double* __restrict__ gy,
       double* __restrict__ gz) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const double* w = g.wgrad + size_t(L.col) * 18;
    double s0[E], ax[E], ay[E], az[E];
    load_row<E>(s + size_t(L.col) * nv, L.k0, nv, s0);
#pragma unroll
    for (int e = 0; e < E; ++e) ax[e] = ay[e] = az[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int c = __ldg(g.nbr + size_t(L.col) * 6 + j);
        const double wx = __ldg(w + 3 * j), wy = __ldg(w + 3 * j + 1), wz = __ldg(w + 3 * j + 2);
        double sj[E];
        load_row<E>(s + size_t(c) * nv, L.k0, nv, sj);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = sj[e] - s0[e];
            ax[e] = fma(wx, d, ax[e]); ay[e] = fma(wy, d, ay[e]); az[e] = fma(wz, d, az[e]);
        }
    }
    double ri[E];
    load_row<E>(g.rinv, L.k0, nv, ri);
#pragma unroll
    for (int e = 0; e < E; ++e) { ax[e] *= ri[e]; ay[e] *= ri[e]; az[e] *= ri[e]; }
    store_row<E>(gx + size_t(L.col) * nv, L.k0, nv, L.live, ax);
    store_row<E>(gy + size_t(L.col) * nv, L.k0, nv, L.live, ay);
    store_row<E>(gz + size_t(L.col) * nv, L.k0, nv, L.live, az);
}

// ---------------------------------------------------------------------------------------------
// S1: stage preparation (column-local).  Fig. 6 large-step 4 of the previous stage and
// large-step 1 of this one:  Phi^[t] <- Phi^n (stage 1) or Phi^[t] + Phi* (stages 2, 3);
// h = Cp p/(Rd rho) (Eq. 38, G9), theta, u = (V + I_c[W] r)/rho (L268), g~ (Eq. 39) and the
// LU factors of the tridiagonal matrix of Eq. 37 (coefficients: DESIGN.md "tridiagonal", R8) for
// this stage's substep length delta.  The matrix does not change between the substeps of a
// stage, so its factorisation is done once here and the substeps only run the two sweeps.
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_stage_prepare(Geom g, Fields f, int stage, double delta) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const size_t o = size_t(L.col) * nv;
    const double gam = g.Cp / (g.Cp - g.Rd), kv = g.Rd / (g.Cp - g.Rd);
    double rho[E], Vx[E], Vy[E], Vz[E], W[E], p[E];
    if (stage == 1) {
        load_row_rw<E>(f.rho_n + o, L.k0, nv, rho); load_row_rw<E>(f.Vx_n + o, L.k0, nv, Vx);
        load_row_rw<E>(f.Vy_n + o, L.k0, nv, Vy);   load_row_rw<E>(f.Vz_n + o, L.k0, nv, Vz);
        load_row_rw<E>(f.W_n + o, L.k0, nv, W);     load_row_rw<E>(f.p_n + o, L.k0, nv, p);
    } else {
        double d[E];
        load_row_rw<E>(f.rho_t + o, L.k0, nv, rho); load_row_rw<E>(f.rho_s + o, L.k0, nv, d);
#pragma unroll
        for (int e = 0; e < E; ++e) rho[e] += d[e];
        load_row_rw<E>(f.Vx_t + o, L.k0, nv, Vx); load_row_rw<E>(f.Vx_s + o, L.k0, nv, d);
#pragma unroll
        for (int e = 0; e < E; ++e) Vx[e] += d[e];
        load_row_rw<E>(f.Vy_t + o, L.k0, nv, Vy); load_row_rw<E>(f.Vy_s + o, L.k0, nv, d);
#pragma unroll
        for (int e = 0; e < E; ++e) Vy[e] += d[e];
        load_row_rw<E>(f.Vz_t + o, L.k0, nv, Vz); load_row_rw<E>(f.Vz_s + o, L.k0, nv, d);
#pragma unroll
        for (int e = 0; e < E; ++e) Vz[e] += d[e];
        load_row_rw<E>(f.W_t + o, L.k0, nv, W); load_row_rw<E>(f.W_s + o, L.k0, nv, d);
#pragma unroll
        for (int e = 0; e < E; ++e) W[e] += d[e];
        load_row_rw<E>(f.p_t + o, L.k0, nv, p); load_row_rw<E>(f.p_s + o, L.k0, nv, d);
#pragma unroll
        for (int e = 0; e < E; ++e) p[e] += d[e];
    }
    // masked layers: harmless non-zero values so that nothing divides by zero
#pragma unroll
    for (int e = 0; e < E; ++e)
        if (L.k0 + e >= nv) { rho[e] = 1.0; p[e] = g.p_ref; }

    const double rx = __ldg(g.rhat + 3 * L.col), ry = __ldg(g.rhat + 3 * L.col + 1), rz = __ldg(g.rhat + 3 * L.col + 2);
    double h[E], th[E], rtt[E], Wup[E], ux[E], uy[E], uz[E];
    above<G, E>(W, Wup, L.gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        h[e] = g.Cp * p[e] / (g.Rd * rho[e]);
        rtt[e] = eos_rt(p[e], g.Rd, g.p_ref, 1.0 / gam);
        th[e] = rtt[e] / rho[e];
        const double wc = (L.k0 + e == nv - 1) ? 0.5 * W[e] : 0.5 * (W[e] + Wup[e]);   // I_c[W]
        const double ir = 1.0 / rho[e];
        ux[e] = (Vx[e] + wc * rx) * ir; uy[e] = (Vy[e] + wc * ry) * ir; uz[e] = (Vz[e] + wc * rz) * ir;
    }
    // interface quantities on the lower interface of each layer
    double pb[E], rb[E], hb[E], hh[E], gt[E];
    below<G, E>(p, pb, L.gl, 0.0); below<G, E>(rho, rb, L.gl, 0.0); below<G, E>(h, hb, L.gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        const bool in = k >= 1 && k < nv;                 // interior interface
        hh[e] = in ? 0.5 * (hb[e] + h[e]) : 0.0;          // I_h[h]
        gt[e] = in ? ((p[e] - pb[e]) / g.dz) / (0.5 * (rb[e] + rho[e])) : 0.0;   // Eq. 39
    }
    double hhb[E], hha[E], gtb[E], gta[E], dlo[E], dhi[E], dlob[E], dhib[E];
    below<G, E>(hh, hhb, L.gl, 0.0); above<G, E>(hh, hha, L.gl, 0.0);
    below<G, E>(gt, gtb, L.gl, 0.0); above<G, E>(gt, gta, L.gl, 0.0);
    load_row<E>(g.dlo, L.k0, nv, dlo); load_row<E>(g.dhi, L.k0, nv, dhi);
    below<G, E>(dlo, dlob, L.gl, 0.0); below<G, E>(dhi, dhib, L.gl, 0.0);
    double ta[E], tb[E], tc[E];
    const double d2 = delta * delta, ck = d2 * kv / g.dz, cg = 0.5 * d2 * g.gravity;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        // the top interior interface (k = nv-1) has no unknown above it: hh, g~ there are the lid's 0
        const double hu = (k + 1 < nv) ? hha[e] : 0.0, gu = (k + 1 < nv) ? gta[e] : 0.0;
        tc[e] = -ck * (dhi[e] * hu - 0.5 * gu) - cg * dhi[e];
        ta[e] = -ck * (dlob[e] * hhb[e] + 0.5 * gtb[e]) + cg * dlob[e];
        tb[e] = 1.0 + ck * hh[e] * (dlo[e] + dhib[e]) - cg * (dhib[e] - dlo[e]);
    }
    // Thomas forward elimination of the matrix (L339), serial over the interfaces; every lane of the
    // group follows the same recurrence and keeps the factors of its own interfaces.
    double fa[E], fi[E], fc[E];
#pragma unroll
    for (int e = 0; e < E; ++e) fa[e] = fi[e] = fc[e] = 0.0;
    double cprev = 0.0;
    const int gbase = (threadIdx.x & 31) & ~(G - 1);
    for (int kk = 1; kk < nv; ++kk) {
        const int src = kk / E, ee = kk % E;
        double a_ = 0.0, b_ = 0.0, c_ = 0.0;
#pragma unroll
        for (int e = 0; e < E; ++e)
            if (e == ee) { a_ = ta[e]; b_ = tb[e]; c_ = tc[e]; }
        a_ = __shfl_sync(kFull, a_, gbase + src);
        b_ = __shfl_sync(kFull, b_, gbase + src);
        c_ = __shfl_sync(kFull, c_, gbase + src);
        const double inv = 1.0 / (b_ - a_ * cprev);
        cprev = c_ * inv;
#pragma unroll
        for (int e = 0; e < E; ++e)
            if (L.k0 + e == kk) { fi[e] = inv; fa[e] = a_ * inv; fc[e] = cprev; }
    }
    store_row<E>(f.rho_t + o, L.k0, nv, L.live, rho); store_row<E>(f.Vx_t + o, L.k0, nv, L.live, Vx);
    store_row<E>(f.Vy_t + o, L.k0, nv, L.live, Vy);   store_row<E>(f.Vz_t + o, L.k0, nv, L.live, Vz);
    store_row<E>(f.W_t + o, L.k0, nv, L.live, W);     store_row<E>(f.p_t + o, L.k0, nv, L.live, p);
    store_row<E>(f.h + o, L.k0, nv, L.live, h);       store_row<E>(f.th + o, L.k0, nv, L.live, th);
    store_row<E>(f.ux + o, L.k0, nv, L.live, ux);     store_row<E>(f.uy + o, L.k0, nv, L.live, uy);
    store_row<E>(f.uz + o, L.k0, nv, L.live, uz);
    store_row<E>(f.fa + o, L.k0, nv, L.live, fa);     store_row<E>(f.fi + o, L.k0, nv, L.live, fi);
    store_row<E>(f.fc + o, L.k0, nv, L.live, fc);
    if (stage == 1) store_row<E>(f.rt_n + o, L.k0, nv, L.live, rtt);   // (rho theta)^n, start of every stage
}

// ---------------------------------------------------------------------------------------------
// S2: slow terms of the stage (Fig. 6 large-step 3; RHS of Eq. 32-35 and Eq. 42; O4 with R7) and
// the initial deviations of Eq. 31 (R1: every stage starts from t_n).
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_slow_terms(Geom g, Fields f) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const size_t o = size_t(L.col) * nv;
    const double kv = g.Rd / (g.Cp - g.Rd);
    const double* wd = g.wdiv + size_t(L.col) * 21;
    const double* wg = g.wgrad + size_t(L.col) * 18;

    double p0[E], h0[E], th0[E], rho[E], V0x[E], V0y[E], V0z[E], u0x[E], u0y[E], u0z[E];
    load_row<E>(f.p_t + o, L.k0, nv, p0);
    double divV[E], divhV[E], divtV[E], Ax[E], Ay[E], Az[E], gpx[E], gpy[E], gpz[E];
#pragma unroll
    for (int e = 0; e < E; ++e) divV[e] = divhV[e] = divtV[e] = Ax[e] = Ay[e] = Az[e] = gpx[e] = gpy[e] = gpz[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const int c = j == 0 ? L.col : __ldg(g.nbr + size_t(L.col) * 6 + j - 1);
        const size_t oc = size_t(c) * nv;
        const double wx = __ldg(wd + 3 * j), wy = __ldg(wd + 3 * j + 1), wz = __ldg(wd + 3 * j + 2);
        double x[E], y[E], z[E], hj[E], tj[E], ujx[E], ujy[E], ujz[E], pj[E];
        load_row<E>(f.Vx_t + oc, L.k0, nv, x); load_row<E>(f.Vy_t + oc, L.k0, nv, y); load_row<E>(f.Vz_t + oc, L.k0, nv, z);
        load_row<E>(f.h + oc, L.k0, nv, hj);   load_row<E>(f.th + oc, L.k0, nv, tj);
        load_row<E>(f.ux + oc, L.k0, nv, ujx); load_row<E>(f.uy + oc, L.k0, nv, ujy); load_row<E>(f.uz + oc, L.k0, nv, ujz);
        if (j == 0) {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                V0x[e] = x[e]; V0y[e] = y[e]; V0z[e] = z[e]; h0[e] = hj[e]; th0[e] = tj[e];
                u0x[e] = ujx[e]; u0y[e] = ujy[e]; u0z[e] = ujz[e];
            }
        } else {
            load_row<E>(f.p_t + oc, L.k0, nv, pj);
            const double gx = __ldg(wg + 3 * (j - 1)), gy = __ldg(wg + 3 * (j - 1) + 1), gz = __ldg(wg + 3 * (j - 1) + 2);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const double d = pj[e] - p0[e];
                gpx[e] = fma(gx, d, gpx[e]); gpy[e] = fma(gy, d, gpy[e]); gpz[e] = fma(gz, d, gpz[e]);
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = fma(wx, x[e], fma(wy, y[e], wz * z[e]));      // w_j . V_j
            divV[e] += d;
            divhV[e] = fma(hj[e], d, divhV[e]);
            divtV[e] = fma(tj[e], d, divtV[e]);
            Ax[e] = fma(ujx[e], d, Ax[e]); Ay[e] = fma(ujy[e], d, Ay[e]); Az[e] = fma(ujz[e], d, Az[e]);
        }
    }
    double ri[E], dlo[E], dhi[E];
    load_row<E>(g.rinv, L.k0, nv, ri); load_row<E>(g.dlo, L.k0, nv, dlo); load_row<E>(g.dhi, L.k0, nv, dhi);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        divV[e] *= ri[e]; divhV[e] *= ri[e]; divtV[e] *= ri[e];
        Ax[e] *= ri[e]; Ay[e] *= ri[e]; Az[e] *= ri[e];
        gpx[e] *= ri[e]; gpy[e] *= ri[e]; gpz[e] *= ri[e];
    }
    load_row<E>(f.rho_t + o, L.k0, nv, rho);
#pragma unroll
    for (int e = 0; e < E; ++e)
        if (L.k0 + e >= nv) rho[e] = 1.0;
    double W[E], Wup[E];
    load_row<E>(f.W_t + o, L.k0, nv, W);
    above<G, E>(W, Wup, L.gl, 0.0);

    // vertical flux divergences D_c[W I_h[q]] for q = u_x, u_y, u_z, h, theta, and D_c[W]
    double qb[E], X[E], Xup[E];
    auto vflux = [&](const double (&q)[E], double (&out)[E]) {
        below<G, E>(q, qb, L.gl, 0.0);
#pragma unroll
        for (int e = 0; e < E; ++e) X[e] = W[e] * 0.5 * (qb[e] + q[e]);    // W = 0 on the ground
        above<G, E>(X, Xup, L.gl, 0.0);
#pragma unroll
        for (int e = 0; e < E; ++e) out[e] = dhi[e] * Xup[e] - dlo[e] * X[e];
    };
    double t[E];
    vflux(u0x, t);
#pragma unroll
    for (int e = 0; e < E; ++e) Ax[e] += t[e];
    vflux(u0y, t);
#pragma unroll
    for (int e = 0; e < E; ++e) Ay[e] += t[e];
    vflux(u0z, t);
#pragma unroll
    for (int e = 0; e < E; ++e) Az[e] += t[e];
    double DhW[E], DtW[E], DW[E];
    vflux(h0, DhW);
    vflux(th0, DtW);
#pragma unroll
    for (int e = 0; e < E; ++e) DW[e] = dhi[e] * Wup[e] - dlo[e] * W[e];

    const double rx = __ldg(g.rhat + 3 * L.col), ry = __ldg(g.rhat + 3 * L.col + 1), rz = __ldg(g.rhat + 3 * L.col + 2);
    double sVx[E], sVy[E], sVz[E], Fr[E], srho[E], sp[E], srt[E];
    // g~ W on interfaces, then I_c
    double pb[E], rb[E], Z[E], Zup[E];
    below<G, E>(p0, pb, L.gl, 0.0); below<G, E>(rho, rb, L.gl, 1.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        const double gt = (k >= 1 && k < nv) ? ((p0[e] - pb[e]) / g.dz) / (0.5 * (rb[e] + rho[e])) : 0.0;
        Z[e] = gt * W[e];
    }
    above<G, E>(Z, Zup, L.gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double wc = 0.5 * (W[e] + Wup[e]);
        const double Mx = V0x[e] + wc * rx, My = V0y[e] + wc * ry;
        const double Cx = -2.0 * g.omega * My, Cy = 2.0 * g.omega * Mx;       // 2 Omega z x M
        const double Ar = Ax[e] * rx + Ay[e] * ry + Az[e] * rz;
        const double Cr = Cx * rx + Cy * ry;
        Fr[e] = Ar + Cr;
        sVx[e] = -gpx[e] - (Ax[e] - Ar * rx) - (Cx - Cr * rx);
        sVy[e] = -gpy[e] - (Ay[e] - Ar * ry) - (Cy - Cr * ry);
        sVz[e] = -gpz[e] - (Az[e] - Ar * rz) - (0.0 - Cr * rz);
        srho[e] = -divV[e] - DW[e];
        const double vgp = (V0x[e] * gpx[e] + V0y[e] * gpy[e] + V0z[e] * gpz[e]) / rho[e];
        sp[e] = -kv * (divhV[e] + DhW[e] - vgp - 0.5 * (Z[e] + Zup[e]));
        srt[e] = -divtV[e] - DtW[e];
    }
    double Frb[E], sW[E];
    below<G, E>(Fr, Frb, L.gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = L.k0 + e;
        sW[e] = (k >= 1 && k < nv)
                    ? -(p0[e] - pb[e]) / g.dz - g.gravity * 0.5 * (rb[e] + rho[e]) - 0.5 * (Frb[e] + Fr[e])
                    : 0.0;                                                    // Eq. 42
    }
    store_row<E>(f.sVx + o, L.k0, nv, L.live, sVx); store_row<E>(f.sVy + o, L.k0, nv, L.live, sVy);
    store_row<E>(f.sVz + o, L.k0, nv, L.live, sVz); store_row<E>(f.srho + o, L.k0, nv, L.live, srho);
    store_row<E>(f.sW + o, L.k0, nv, L.live, sW);   store_row<E>(f.sp + o, L.k0, nv, L.live, sp);
    store_row<E>(f.srt + o, L.k0, nv, L.live, srt);

    // Eq. 31: Phi*(0) = Phi^n - Phi^[t]; (rho theta)(0) = (rho theta)^n
    double a[E], d[E];
    load_row<E>(f.rho_n + o, L.k0, nv, a);
#pragma unroll
    for (int e = 0; e < E; ++e) d[e] = a[e] - ((L.k0 + e < nv) ? rho[e] : 0.0);
    store_row<E>(f.rho_s + o, L.k0, nv, L.live, d);
    load_row<E>(f.Vx_n + o, L.k0, nv, a);
#pragma unroll
    for (int e = 0; e < E; ++e) d[e] = a[e] - V0x[e];
    store_row<E>(f.Vx_s + o, L.k0, nv, L.live, d);
    load_row<E>(f.Vy_n + o, L.k0, nv, a);
#pragma unroll
    for (int e = 0; e < E; ++e) d[e] = a[e] - V0y[e];
    store_row<E>(f.Vy_s + o, L.k0, nv, L.live, d);
    load_row<E>(f.Vz_n + o, L.k0, nv, a);
#pragma unroll
    for (int e = 0; e < E; ++e) d[e] = a[e] - V0z[e];
    store_row<E>(f.Vz_s + o, L.k0, nv, L.live, d);
    load_row<E>(f.W_n + o, L.k0, nv, a);
#pragma unroll
    for (int e = 0; e < E; ++e) d[e] = a[e] - W[e];
    store_row<E>(f.W_s + o, L.k0, nv, L.live, d);
    load_row<E>(f.p_n + o, L.k0, nv, a);
#pragma unroll
    for (int e = 0; e < E; ++e) d[e] = a[e] - p0[e];
    store_row<E>(f.p_s + o, L.k0, nv, L.live, d);
    load_row<E>(f.rt_n + o, L.k0, nv, a);
    store_row<E>(f.rt + o, L.k0, nv, L.live, a);
}

// ---------------------------------------------------------------------------------------------
// K1 (a4): explicit horizontal momentum, Eq. 33 (Fig. 6 small-step 2):
//   V*' = V* + delta (-grad_h p* / r + slowV).  Gathers p* from the 6 neighbours.
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_momentum(Geom g, Fields f, double delta) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const size_t o = size_t(L.col) * nv;
    const double* wg = g.wgrad + size_t(L.col) * 18;
    double p0[E], gx[E], gy[E], gz[E];
    load_row<E>(f.p_s + o, L.k0, nv, p0);
#pragma unroll
    for (int e = 0; e < E; ++e) gx[e] = gy[e] = gz[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int c = __ldg(g.nbr + size_t(L.col) * 6 + j);
        const double wx = __ldg(wg + 3 * j), wy = __ldg(wg + 3 * j + 1), wz = __ldg(wg + 3 * j + 2);
        double pj[E];
        load_row<E>(f.p_s + size_t(c) * nv, L.k0, nv, pj);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = pj[e] - p0[e];
            gx[e] = fma(wx, d, gx[e]); gy[e] = fma(wy, d, gy[e]); gz[e] = fma(wz, d, gz[e]);
        }
    }
    double ri[E], v[E], s[E];
    load_row<E>(g.rinv, L.k0, nv, ri);
    load_row_rw<E>(f.Vx_s + o, L.k0, nv, v); load_row<E>(f.sVx + o, L.k0, nv, s);
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = fma(delta, s[e] - gx[e] * ri[e], v[e]);
    store_row<E>(f.Vx_s + o, L.k0, nv, L.live, v);
    load_row_rw<E>(f.Vy_s + o, L.k0, nv, v); load_row<E>(f.sVy + o, L.k0, nv, s);
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = fma(delta, s[e] - gy[e] * ri[e], v[e]);
    store_row<E>(f.Vy_s + o, L.k0, nv, L.live, v);
    load_row_rw<E>(f.Vz_s + o, L.k0, nv, v); load_row<E>(f.sVz + o, L.k0, nv, s);
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = fma(delta, s[e] - gz[e] * ri[e], v[e]);
    store_row<E>(f.Vz_s + o, L.k0, nv, L.live, v);
}

// ---------------------------------------------------------------------------------------------
// K2 (a5-a9): horizontal divergences of the new momentum, the implicit vertical momentum
// (Eq. 37; two sweeps with the stage's LU factors), density (Eq. 32), rho*theta (Eq. 35, G7) and
// the pressure deviation (Eq. 36).  Fig. 6 small-steps 3-6.  Gathers V*', h, theta from the 6
// neighbours; everything else is column-local.
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_vertical(Geom g, Fields f, double delta) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const size_t o = size_t(L.col) * nv;
    const double gam = g.Cp / (g.Cp - g.Rd), kv = g.Rd / (g.Cp - g.Rd);
    const double* wd = g.wdiv + size_t(L.col) * 21;

    double divV[E], divhV[E], divtV[E], th0[E];
#pragma unroll
    for (int e = 0; e < E; ++e) divV[e] = divhV[e] = divtV[e] = 0.0;
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        const int c = j == 0 ? L.col : __ldg(g.nbr + size_t(L.col) * 6 + j - 1);
        const size_t oc = size_t(c) * nv;
        const double wx = __ldg(wd + 3 * j), wy = __ldg(wd + 3 * j + 1), wz = __ldg(wd + 3 * j + 2);
        double x[E], y[E], z[E], hj[E], tj[E];
        load_row<E>(f.Vx_s + oc, L.k0, nv, x); load_row<E>(f.Vy_s + oc, L.k0, nv, y); load_row<E>(f.Vz_s + oc, L.k0, nv, z);
        load_row<E>(f.h + oc, L.k0, nv, hj);   load_row<E>(f.th + oc, L.k0, nv, tj);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double d = fma(wx, x[e], fma(wy, y[e], wz * z[e]));
            divV[e] += d;
            divhV[e] = fma(hj[e], d, divhV[e]);
            divtV[e] = fma(tj[e], d, divtV[e]);
            if (j == 0) th0[e] = tj[e];
        }
    }
    double ri[E], dlo[E], dhi[E];
    load_row<E>(g.rinv, L.k0, nv, ri); load_row<E>(g.dlo, L.k0, nv, dlo); load_row<E>(g.dhi, L.k0, nv, dhi);

    double rho_s[E], p_s[E], W_s[E], srho[E], sp[E], sW[E];
    load_row_rw<E>(f.rho_s + o, L.k0, nv, rho_s); load_row_rw<E>(f.p_s + o, L.k0, nv, p_s);
    load_row_rw<E>(f.W_s + o, L.k0, nv, W_s);
    load_row<E>(f.srho + o, L.k0, nv, srho); load_row<E>(f.sp + o, L.k0, nv, sp); load_row<E>(f.sW + o, L.k0, nv, sW);
    double pq[E], rq[E], pqb[E], rqb[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double Srho = srho[e] - divV[e] * ri[e];                 // Eq. 41
        const double Sp = sp[e] - kv * divhV[e] * ri[e];               // Eq. 40 (G10)
        pq[e] = fma(delta, Sp, p_s[e]);
        rq[e] = fma(delta, Srho, rho_s[e]);
    }
    below<G, E>(pq, pqb, L.gl, 0.0); below<G, E>(rq, rqb, L.gl, 0.0);
    // right-hand side d_k on interior interfaces (0 on the ground), already scaled by 1/b'_k
    double fa[E], fi[E], fc[E], A[E], B[E], zf[E], Wn[E];
    load_row<E>(f.fa + o, L.k0, nv, fa); load_row<E>(f.fi + o, L.k0, nv, fi); load_row<E>(f.fc + o, L.k0, nv, fc);
    const double cdz = delta / g.dz, cg = 0.5 * delta * g.gravity;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const double d = W_s[e] + delta * sW[e] - cdz * (pq[e] - pqb[e]) - cg * (rqb[e] + rq[e]);
        A[e] = -fa[e];            // z_k = d_k/b'_k - (a_k/b'_k) z_(k-1)
        B[e] = fi[e] * d;         // fi = 0 on the ground and on masked layers
    }
    affine_scan<G, E, false>(A, B, zf, L.gl);
#pragma unroll
    for (int e = 0; e < E; ++e) A[e] = -fc[e];                          // x_k = z_k - c'_k x_(k+1)
    affine_scan<G, E, true>(A, zf, Wn, L.gl);

    double Wup[E], thb[E], X[E], Xup[E], rt[E], srt[E], p_t[E];
    above<G, E>(Wn, Wup, L.gl, 0.0);
    below<G, E>(th0, thb, L.gl, 0.0);
#pragma unroll
    for (int e = 0; e < E; ++e) X[e] = 0.5 * (thb[e] + th0[e]) * Wn[e];  // I_h[theta] W'
    above<G, E>(X, Xup, L.gl, 0.0);
    load_row_rw<E>(f.rt + o, L.k0, nv, rt); load_row<E>(f.srt + o, L.k0, nv, srt); load_row<E>(f.p_t + o, L.k0, nv, p_t);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        rho_s[e] = rq[e] - delta * (dhi[e] * Wup[e] - dlo[e] * Wn[e]);                             // Eq. 32
        rt[e] = rt[e] + delta * (srt[e] - divtV[e] * ri[e] - (dhi[e] * Xup[e] - dlo[e] * X[e]));  // Eq. 35
        if (L.k0 + e >= nv) rt[e] = g.p_ref / g.Rd;
        p_s[e] = eos_p(rt[e], g.Rd, g.p_ref, gam) - p_t[e];                                        // Eq. 36
    }
    store_row<E>(f.W_s + o, L.k0, nv, L.live, Wn);   store_row<E>(f.rho_s + o, L.k0, nv, L.live, rho_s);
    store_row<E>(f.rt + o, L.k0, nv, L.live, rt);    store_row<E>(f.p_s + o, L.k0, nv, L.live, p_s);
}

// ---------------------------------------------------------------------------------------------
// End of the large step: Phi^(n+1) = Phi^[t] + Phi* (Fig. 6 large-step 4), then the PROFX forcing
// (Eq. 51-52, backward Euler with the large step, R9).
// ---------------------------------------------------------------------------------------------
__global__ void k_finish(size_t n, Fields f, double dt, double Rd) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double rho = f.rho_t[i] + f.rho_s[i];
    double vx = f.Vx_t[i] + f.Vx_s[i], vy = f.Vy_t[i] + f.Vy_s[i], vz = f.Vz_t[i] + f.Vz_s[i];
    double w = f.W_t[i] + f.W_s[i];
    double p = f.p_t[i] + f.p_s[i];
    if (f.k_v) {
        const double s = 1.0 + f.k_v[i] * dt;
        vx /= s; vy /= s; vz /= s;                                           // Eq. 51
    }
    if (f.k_T && f.T_eq) {
        double T = p / (rho * Rd);                                           // Eq. 25
        T = (T + f.k_T[i] * dt * f.T_eq[i]) / (1.0 + f.k_T[i] * dt);         // Eq. 52
        p = rho * Rd * T;
    }
    f.rho_n[i] = rho; f.Vx_n[i] = vx; f.Vy_n[i] = vy; f.Vz_n[i] = vz; f.W_n[i] = w; f.p_n[i] = p;
}

// ---------------------------------------------------------------------------------------------
// Diagnostics (a12, R10): per-column partial sums of mass and energy; host finishes the sum.
// ---------------------------------------------------------------------------------------------
template <int G, int E>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_diag(Geom g, Fields f, double* __restrict__ col_mass, double* __restrict__ col_energy) {
    Lanes<G, E> L(g.N);
    const int nv = g.nv;
    const size_t o = size_t(L.col) * nv;
    const double Cv = g.Cp - g.Rd;
    double rho[E], Vx[E], Vy[E], Vz[E], W[E], Wup[E], p[E], vol[E], zc[E];
    load_row_rw<E>(f.rho_n + o, L.k0, nv, rho); load_row_rw<E>(f.Vx_n + o, L.k0, nv, Vx);
    load_row_rw<E>(f.Vy_n + o, L.k0, nv, Vy);   load_row_rw<E>(f.Vz_n + o, L.k0, nv, Vz);
    load_row_rw<E>(f.W_n + o, L.k0, nv, W);     load_row_rw<E>(f.p_n + o, L.k0, nv, p);
    load_row<E>(g.vol, L.k0, nv, vol);          load_row<E>(g.zc, L.k0, nv, zc);
    above<G, E>(W, Wup, L.gl, 0.0);
    double m = 0.0, en = 0.0;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        if (L.k0 + e < nv) {
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
    if (L.live && L.gl == 0) {
        const double a = __ldg(g.area + L.col);
        col_mass[L.col] = m * a;
        col_energy[L.col] = en * a;
    }
}

// ---------------------------------------------------------------------------------------------
// Canonical (host order, as uploaded) <-> device order
// ---------------------------------------------------------------------------------------------
// in: canonical [N][nv*stride_in + off...] ; generic row gather: out[d][k] = in[order[d]][k*cs + c0]
__global__ void k_gather_rows(int N, int nv, const int* __restrict__ order, const double* __restrict__ in,
                              int row_len, int cs, int c0, double* __restrict__ out) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= size_t(N) * nv) return;
    const int d = int(i / nv), k = int(i % nv);
    out[i] = in[size_t(order[d]) * row_len + size_t(k) * cs + c0];
}
// out: canonical; out[order[d]][k*cs + c0] = in[d][k]
__global__ void k_scatter_rows(int N, int nv, const int* __restrict__ order, const double* __restrict__ in,
                               int row_len, int cs, int c0, double* __restrict__ out) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= size_t(N) * nv) return;
    const int d = int(i / nv), k = int(i % nv);
    out[size_t(order[d]) * row_len + size_t(k) * cs + c0] = in[i];
}
__global__ void k_zero_ground(int N, int nv, double* W) {
    int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d < N) W[size_t(d) * nv] = 0.0;
}
__global__ void k_fill(size_t n, double* p, double v) {
    size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

}  // namespace thor
