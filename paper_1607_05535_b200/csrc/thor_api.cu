// C-ABI of include/thor.h: argument checks, device memory, the launch sequence of one large
// step (Fig. 6).  Every step of the path runs in the kernels of
// thor_kernels.cuh; there is no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cstdint>
#include <initializer_list>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "grid_host.h"
#include "thor.h"
#include "thor_kernels.cuh"

using namespace thor;

namespace {

thread_local std::string g_err;
std::atomic<long long> g_launches{0};

int fail(int code, const std::string& msg) {
    g_err = msg;
    return code;
}
#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(THOR_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));          \
    } while (0)

constexpr int kMaxLayers = 128;

struct DeviceGeom {
    bool ready = false;
    int device = -1;
    int Npad = 0;
    int* nbr = nullptr;
    int* order = nullptr;
    double *wdiv = nullptr, *wgrad = nullptr, *area = nullptr;
    double *frame = nullptr, *wdiv2 = nullptr, *wgrad2 = nullptr, *wlap = nullptr;
    double *rinv = nullptr, *dlo = nullptr, *dhi = nullptr, *vol = nullptr, *zc = nullptr, *rhinv = nullptr;
    double *wl = nullptr, *wh = nullptr, *idz = nullptr, *vk = nullptr;
    // tiles of the TMA-staged column-solve kernel (kTmaWarps * 32/G consecutive columns each)
    int tcol = 0, hmax = 0;
    // NEXT-1 divergence damping as ONE stencil: -lap(grad D3) composed on the host over the two rings of a column
    int* dd_idx = nullptr;            // [Npad][20] the 18 columns of the two rings (pads: the column itself)
    double* dd_coef = nullptr;        // [Npad][20][2] tangent-basis coefficients of (D3_m - D3_i), unit sphere (x -K_d / r^3)
    int* tile_halo = nullptr;
    unsigned char* tile_slots = nullptr;
    // scratch of the host wrappers thor_apply_div/grad/lap (7 x N x nv doubles), allocated on first use
    double* op_buf = nullptr;
};

// lane-group width G and layers per lane E of the record kernels; NVP = G*E padded layers
struct Shape { int G, E; };
Shape shape_for(int nv) {
    if (nv <= 8) return {4, 2};
    if (nv <= 16) return {8, 2};
    if (nv <= 32) return {16, 2};
    if (nv <= 64) return {32, 2};
    return {32, 4};
}

}  // namespace

struct thor_grid {
    HostGrid h;
    mutable DeviceGeom d;
};

struct thor_state {
    const thor_grid* grid = nullptr;
    cudaStream_t stream = nullptr;
    int NVP = 0;
    double* S = nullptr;             // the slab of column records [Npad][NF][NVP]
    double* X = nullptr;             // NEXT-1 work rows [Npad][XF][NVP], allocated by thor_state_set_diffusion
    double D_hyp = 0.0, D_div = 0.0; // non-dimensional diffusion parameters of Eq. 49 (0 = term off)
    HeldSuarez hs{};                 // NEXT-2: forcing from the evolving sigma (on = 0: tables or none)
    HotJupiter hj{};
    double* stage_buf = nullptr;     // canonical-order staging, max(N*nv*3, N*(nv+1)) doubles
    double *tab_Teq = nullptr, *tab_kT = nullptr, *tab_kv = nullptr;   // [Npad][NVP]
    bool has_Teq = false, has_kT = false, has_kv = false;
    double *col_mass = nullptr, *col_energy = nullptr;
    int efix = 0;                    // NEXT-4: energy fixer of L215 (RE1) on
    double* efix_dev = nullptr;      // device [M, E before the step; M', E' after its dynamics]
    bool stepped = false;
    int walk = 0;                    // direction of the last launch (0 ascending, 1 descending)
    // one large step captured as a CUDA graph, per starting walk direction (replayed while the key holds)
    struct GraphKey { double dt = 0, D_hyp = 0, D_div = 0; int efix = 0; HeldSuarez hs{}; HotJupiter hj{}; int n = 0; const double *Teq = nullptr, *kT = nullptr, *kv = nullptr; char tune[96] = {0}; };
    GraphKey gkey;
    cudaGraphExec_t gexec[2] = {nullptr, nullptr};
    int gwalk_end[2] = {0, 0};
    int gkernels = 0;
    // the launch sequence of thor_acoustic_substeps as a graph (one cached entry; same reason, same rules)
    struct SubKey { double delta = 0; int n = 0, which = 0, walk0 = 0; char tune[96] = {0}; };
    SubKey skey;
    cudaGraphExec_t sexec = nullptr;
    int swalk_end = 0, skernels = 0;
};

namespace {

template <class T>
int upload(T** dst, const std::vector<T>& src) {
    CU(cudaMalloc(reinterpret_cast<void**>(dst), src.size() * sizeof(T)));
    CU(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return THOR_OK;
}

// device copy of the geometry, padded to Npad columns (pad columns: own neighbour, zero weights)
// and to kMaxLayers layers (pad layers: 0)
void free_device_geom(DeviceGeom& d) {
    cudaFree(d.nbr); cudaFree(d.order); cudaFree(d.wdiv); cudaFree(d.wgrad); cudaFree(d.frame); cudaFree(d.area);
    cudaFree(d.rinv); cudaFree(d.dlo); cudaFree(d.dhi); cudaFree(d.vol); cudaFree(d.zc); cudaFree(d.rhinv);
    cudaFree(d.wl); cudaFree(d.wh); cudaFree(d.idz); cudaFree(d.vk);
    cudaFree(d.tile_halo); cudaFree(d.tile_slots); cudaFree(d.dd_idx); cudaFree(d.dd_coef);
    cudaFree(d.wdiv2); cudaFree(d.wgrad2); cudaFree(d.wlap); cudaFree(d.op_buf);
    d = DeviceGeom();
}

int upload_device_geom(const thor_grid* grid);

// The device copy belongs to ONE device (the current one at first use); a call with another current device is
// refused instead of dereferencing foreign pointers.  Serialised: two threads may share a grid.
int ensure_device_geom(const thor_grid* grid) {
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    DeviceGeom& d = grid->d;
    int dev = -1;
    if (d.ready) {
        CU(cudaGetDevice(&dev));
        if (dev != d.device)
            return fail(THOR_EINVAL, "grid lives on CUDA device " + std::to_string(d.device) + ", current device is " + std::to_string(dev));
        return THOR_OK;
    }
    const int rc = upload_device_geom(grid);
    if (rc != THOR_OK) free_device_geom(d);              // nothing half-uploaded is kept
    return rc;
}

int upload_device_geom(const thor_grid* grid) {
    DeviceGeom& d = grid->d;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0)
        return fail(THOR_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(e));
    CU(cudaGetDevice(&d.device));
    const HostGrid& h = grid->h;
    const int N = h.N, Npad = (N + kColPad - 1) / kColPad * kColPad;
    d.Npad = Npad;
    std::vector<int> nbr(size_t(Npad) * 8);
    std::vector<double> wdiv(size_t(Npad) * 24, 0.0), wgrad(size_t(Npad) * 18, 0.0), rhat(size_t(Npad) * 4, 0.0),
        area(Npad, 0.0), basis(size_t(Npad) * 8, 0.0), wdiv2(size_t(Npad) * 16, 0.0), wgrad2(size_t(Npad) * 12, 0.0),
        wlap(size_t(Npad) * 8, 0.0), frame(size_t(Npad) * 12, 0.0);
    for (int c = 0; c < Npad; ++c) {
        for (int k = 0; k < 8; ++k) nbr[size_t(c) * 8 + k] = (c < N && k < 6) ? h.d_nbr[size_t(c) * 6 + k] : c;
        if (c >= N) {
            rhat[size_t(c) * 4 + 2] = 1.0; basis[size_t(c) * 8] = 1.0; basis[size_t(c) * 8 + 4] = 1.0;
            frame[size_t(c) * 12] = 1.0; frame[size_t(c) * 12 + 4] = 1.0; frame[size_t(c) * 12 + 8] = 1.0;
            continue;
        }
        std::copy_n(&h.d_basis[size_t(c) * 6], 6, &frame[size_t(c) * 12]);
        std::copy_n(&h.d_rhat[size_t(c) * 3], 3, &frame[size_t(c) * 12 + 6]);
        std::copy_n(&h.d_basis[size_t(c) * 6], 6, &basis[size_t(c) * 8]);
        std::copy_n(&h.d_wdiv2[size_t(c) * 14], 14, &wdiv2[size_t(c) * 16]);
        std::copy_n(&h.d_wgrad2[size_t(c) * 12], 12, &wgrad2[size_t(c) * 12]);
        std::copy_n(&h.d_wlap[size_t(c) * 6], 6, &wlap[size_t(c) * 8]);
        std::copy_n(&h.d_wdiv[size_t(c) * 21], 21, &wdiv[size_t(c) * 24]);
        std::copy_n(&h.d_wgrad[size_t(c) * 18], 18, &wgrad[size_t(c) * 18]);
        std::copy_n(&h.d_rhat[size_t(c) * 3], 3, &rhat[size_t(c) * 4]);
        area[c] = h.d_area[c];
    }
    auto padded = [&](const std::vector<double>& v) {
        std::vector<double> o(kMaxLayers, 0.0);
        std::copy(v.begin(), v.end(), o.begin());
        return o;
    };
    int rc;
    if ((rc = upload(&d.nbr, nbr))) return rc;
    if ((rc = upload(&d.order, h.order))) return rc;
    if ((rc = upload(&d.wdiv, wdiv))) return rc;
    if ((rc = upload(&d.wgrad, wgrad))) return rc;
    if ((rc = upload(&d.frame, frame))) return rc;
    if ((rc = upload(&d.area, area))) return rc;
    if ((rc = upload(&d.wdiv2, wdiv2))) return rc;
    if ((rc = upload(&d.wgrad2, wgrad2))) return rc;
    if ((rc = upload(&d.wlap, wlap))) return rc;
    if ((rc = upload(&d.rinv, padded(h.rinv)))) return rc;
    if ((rc = upload(&d.dlo, padded(h.dlo)))) return rc;
    if ((rc = upload(&d.dhi, padded(h.dhi)))) return rc;
    if ((rc = upload(&d.vol, padded(h.vol)))) return rc;
    if ((rc = upload(&d.zc, padded(h.zc)))) return rc;
    if ((rc = upload(&d.rhinv, padded(h.rhinv)))) return rc;
    if ((rc = upload(&d.wl, padded(h.wl)))) return rc;
    if ((rc = upload(&d.wh, padded(h.wh)))) return rc;
    if ((rc = upload(&d.idz, padded(h.idz)))) return rc;
    {   // NEXT-3: the order-3 weights of Eq. 8-9, [8][kMaxLayers]
        std::vector<double> vk(size_t(8) * kMaxLayers, 0.0);
        for (int r = 0; r < 4; ++r)
            for (int k = 0; k < h.nv; ++k) {
                vk[size_t(r) * kMaxLayers + k] = h.ihw[size_t(r) * h.nv + k];
                vk[size_t(4 + r) * kMaxLayers + k] = h.icw[size_t(r) * h.nv + k];
            }
        if ((rc = upload(&d.vk, vk))) return rc;
    }
    {   // composed operator of the divergence damping (RD4): F_i = -K_d P_i lap(grad D3)_i
        //   grad D3 at column c:  G_c = sum_j wgrad_cj (D3_nbr(c,j) - D3_c)
        //   lap of each Cartesian component: sum_c wlap_ic (G_c - G_i), then Eq. 28 at i and its tangent basis
        std::vector<int> idx(size_t(Npad) * 20);
        std::vector<double> coef(size_t(Npad) * 40, 0.0);
        for (int i = 0; i < Npad; ++i) {
            int* id = &idx[size_t(i) * 20];
            std::fill(id, id + 20, i);
            if (i >= N) continue;
            int cnt = 0;
            double acc[20][3] = {};
            double self[3] = {0, 0, 0};                               // coefficient of D3_i itself (minus the sum of the others)
            auto add = [&](int m, double sx, double sy, double sz) {
                if (m == i) { self[0] += sx; self[1] += sy; self[2] += sz; return; }
                int q = 0;
                while (q < cnt && id[q] != m) ++q;
                if (q == cnt) id[cnt++] = m;
                acc[q][0] += sx; acc[q][1] += sy; acc[q][2] += sz;
            };
            auto add_grad = [&](int c, double scale) {               // scale * G_c expanded on the D3 values
                for (int j = 0; j < 6; ++j) {
                    const double* wg = &wgrad[size_t(c) * 18 + 3 * j];
                    const int m = nbr[size_t(c) * 8 + j];
                    add(m, scale * wg[0], scale * wg[1], scale * wg[2]);
                    add(c, -scale * wg[0], -scale * wg[1], -scale * wg[2]);
                }
            };
            double lsum = 0.0;
            for (int k = 0; k < 6; ++k) {
                const double L = wlap[size_t(i) * 8 + k];
                add_grad(nbr[size_t(i) * 8 + k], L);
                lsum += L;
            }
            add_grad(i, -lsum);
            const double* r = &rhat[size_t(i) * 4];
            const double* b = &basis[size_t(i) * 8];
            for (int q = 0; q < cnt; ++q) {
                double v[3] = {acc[q][0], acc[q][1], acc[q][2]};
                const double vr = v[0] * r[0] + v[1] * r[1] + v[2] * r[2];
                for (int d2 = 0; d2 < 3; ++d2) v[d2] -= vr * r[d2];
                coef[size_t(i) * 40 + 2 * q] = v[0] * b[0] + v[1] * b[1] + v[2] * b[2];
                coef[size_t(i) * 40 + 2 * q + 1] = v[0] * b[3] + v[1] * b[4] + v[2] * b[5];
            }
            (void)self;                                               // difference form: applied to D3_m - D3_i
        }
        if ((rc = upload(&d.dd_idx, idx))) return rc;
        if ((rc = upload(&d.dd_coef, coef))) return rc;
    }
    {   // tile tables: halo columns of every tile and, per column, the slot of each neighbour
        const Shape sh = shape_for(h.nv);
        const int TC = kTmaWarps * (32 / sh.G), ntiles = Npad / TC;
        std::vector<std::vector<int>> halo(ntiles);
        std::vector<unsigned char> slots(size_t(Npad) * 8, 0);
        int hmax = 0;
        for (int t = 0; t < ntiles; ++t) {
            std::vector<int>& hl = halo[t];
            for (int c = t * TC; c < (t + 1) * TC; ++c)
                for (int k = 0; k < 8; ++k) {
                    const int nb = nbr[size_t(c) * 8 + k];
                    int slot;
                    if (nb / TC == t) slot = nb - t * TC;
                    else {
                        auto it = std::find(hl.begin(), hl.end(), nb);
                        if (it == hl.end()) { hl.push_back(nb); it = hl.end() - 1; }
                        slot = TC + int(it - hl.begin());
                    }
                    slots[size_t(c) * 8 + k] = static_cast<unsigned char>(slot);
                }
            hmax = std::max(hmax, int(hl.size()));
        }
        hmax = std::max(hmax, 1);
        std::vector<int> flat(size_t(ntiles) * hmax);
        for (int t = 0; t < ntiles; ++t)
            for (int i = 0; i < hmax; ++i) flat[size_t(t) * hmax + i] = i < int(halo[t].size()) ? halo[t][i] : t * TC;
        d.tcol = TC; d.hmax = hmax;
        if (TC + hmax > 255) d.hmax = 0;                 // slots are bytes; such a grid uses the direct kernel
        if ((rc = upload(&d.tile_halo, flat))) return rc;
        if ((rc = upload(&d.tile_slots, slots))) return rc;
    }
    d.ready = true;
    return THOR_OK;
}

Geom make_geom(const thor_grid* grid) {
    const HostGrid& h = grid->h;
    const DeviceGeom& d = grid->d;
    Geom g;
    g.N = h.N; g.Npad = d.Npad; g.nv = h.nv;
    g.nbr = d.nbr; g.wdiv = d.wdiv; g.wgrad = d.wgrad; g.frame = d.frame; g.area = d.area;
    g.wdiv2 = d.wdiv2; g.wgrad2 = d.wgrad2; g.wlap = d.wlap;
    g.dd_idx = d.dd_idx; g.dd_coef = d.dd_coef;
    g.rinv = d.rinv; g.dlo = d.dlo; g.dhi = d.dhi; g.vol = d.vol; g.zc = d.zc; g.rhinv = d.rhinv;
    g.wl = d.wl; g.wh = d.wh; g.idz = d.idz; g.vk = d.vk; g.kord = h.kord;
    g.lvl2 = h.lattice_nbr ? 2 * h.level : -1;
    g.omega = h.P.omega; g.gravity = h.P.gravity; g.Rd = h.P.Rd; g.Cp = h.P.Cp; g.p_ref = h.P.p_ref;
    // binomial series of Eq. 36 in deviation form: q_k = C(gamma, k+1)/gamma
    const double gam = h.P.Cp / (h.P.Cp - h.P.Rd);
    g.eosq[0] = 1.0;
    for (int k = 1; k <= kEosTerms; ++k) g.eosq[k] = g.eosq[k - 1] * (gam - k) / (k + 1);
    return g;
}

// dispatch a record kernel template over the supported (G, E) shapes; Npad is a multiple of the
// columns per block of every shape
#define THOR_DISPATCH(KERNEL, nv, Npad, stream, ...)                                               \
    do {                                                                                           \
        const Shape sh_ = shape_for(nv);                                                           \
        const dim3 grid_((Npad) / (kWarpsPerBlock * (32 / sh_.G))), block_(kWarpsPerBlock * 32);   \
        if (sh_.G == 4) KERNEL<4, 2><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                   \
        else if (sh_.G == 8) KERNEL<8, 2><<<grid_, block_, 0, stream>>>(__VA_ARGS__);              \
        else if (sh_.G == 16) KERNEL<16, 2><<<grid_, block_, 0, stream>>>(__VA_ARGS__);            \
        else if (sh_.E == 2) KERNEL<32, 2><<<grid_, block_, 0, stream>>>(__VA_ARGS__);             \
        else KERNEL<32, 4><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                             \
        g_launches.fetch_add(1, std::memory_order_relaxed);                                        \
    } while (0)

// config-1 operators on plain [N][nv] arrays: G lanes per column, E = ceil(nv/G) strided layers per lane
#define THOR_DISPATCH_OP(KERNEL, nv, N, stream, ...)                                               \
    do {                                                                                           \
        const int G_ = (nv) <= 8 ? 8 : ((nv) <= 16 ? 16 : 32);                                     \
        const int E_ = ((nv) + G_ - 1) / G_;                                                       \
        const int cpb_ = kWarpsPerBlock * (32 / G_);                                               \
        const dim3 grid_(((N) + cpb_ - 1) / cpb_), block_(kWarpsPerBlock * 32);                    \
        if (G_ == 8) KERNEL<8, 1><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                      \
        else if (G_ == 16) KERNEL<16, 1><<<grid_, block_, 0, stream>>>(__VA_ARGS__);               \
        else if (E_ == 1) KERNEL<32, 1><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                \
        else if (E_ == 2) KERNEL<32, 2><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                \
        else if (E_ == 3) KERNEL<32, 3><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                \
        else KERNEL<32, 4><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                             \
        g_launches.fetch_add(1, std::memory_order_relaxed);                                        \
    } while (0)

int flat_blocks(size_t n) { return int((n + 255) / 256); }

// scratch of the host wrappers thor_apply_div/grad/lap: 7 N nv doubles, kept in the grid handle
int op_scratch(const thor_grid* grid, double** buf) {
    DeviceGeom& d = grid->d;
    if (!d.op_buf) CU(cudaMalloc(reinterpret_cast<void**>(&d.op_buf), 7 * size_t(grid->h.N) * grid->h.nv * sizeof(double)));
    *buf = d.op_buf;
    return THOR_OK;
}

// fast path of the config-1 operators: even layer count <= 64 and 16-byte aligned arrays
bool op_fast_path(int nv, std::initializer_list<const void*> ptrs) {
    if ((nv & 1) || nv > 64) return false;
    for (const void* p : ptrs)
        if (reinterpret_cast<uintptr_t>(p) & 15u) return false;
    return true;
}
#define THOR_DISPATCH_OP2(KERNEL, nv, N, stream, ...)                                              \
    do {                                                                                           \
        const int G_ = (nv) <= 8 ? 4 : ((nv) <= 16 ? 8 : ((nv) <= 32 ? 16 : 32));                  \
        const int cpb_ = kWarpsPerBlock * (32 / G_);                                               \
        const dim3 grid_(((N) + cpb_ - 1) / cpb_), block_(kWarpsPerBlock * 32);                    \
        if (G_ == 4) KERNEL<4><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                         \
        else if (G_ == 8) KERNEL<8><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                    \
        else if (G_ == 16) KERNEL<16><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                  \
        else KERNEL<32><<<grid_, block_, 0, stream>>>(__VA_ARGS__);                                \
        g_launches.fetch_add(1, std::memory_order_relaxed);                                        \
    } while (0)

// L2 schedule of the step kernels;
// THOR_B200_TUNE="zigzag,k1_ahead,k2_ahead,tail,tma_stages,tma_ctas,stage_ahead,graph" overrides the defaults for
// measurement.  Read at the top of every thor_step / thor_acoustic_substeps call (never inside a graph capture).
struct TunePair { Tune k1, k2, ks; int zigzag, tma_stages, tma_ctas, graph; };
TunePair tune() {
    int v[8] = {1, 148, 148, 148, 0, 4, 148, 1};
    if (const char* e = std::getenv("THOR_B200_TUNE"))
        std::sscanf(e, "%d,%d,%d,%d,%d,%d,%d,%d", &v[0], &v[1], &v[2], &v[3], &v[4], &v[5], &v[6], &v[7]);
    TunePair p;
    p.zigzag = v[0];                 // 1: successive kernels walk the columns in alternating directions
    p.k1 = Tune{0, v[1], v[3]};      // k_momentum: look-ahead, tail hand-over
    p.k2 = Tune{0, v[2], v[3]};      // k_vertical
    p.ks = Tune{0, v[6], 0};         // stage kernels and k_finish: look-ahead only
    p.tma_stages = v[4];      // 0: direct-load column-solve kernel; 1 or 2: TMA-staged, that many stages per block
    p.tma_ctas = v[5];        // persistent blocks per SM of the TMA-staged kernel
    p.graph = v[7];           // 1: replay a large step as a CUDA graph (needs a non-default stream)
    return p;
}

// one canonical host array (or a component of it) -> one row of every column record
int put_row(thor_state* s, const double* host, size_t count, int row_len, int cs, int c0, int field, double pad,
            int zero_k0) {
    const HostGrid& h = s->grid->h;
    const int Npad = s->grid->d.Npad;
    if (host) CU(cudaMemcpyAsync(s->stage_buf, host, count * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    k_rows_from_canonical<<<flat_blocks(size_t(Npad) * s->NVP), 256, 0, s->stream>>>(
        h.N, Npad, h.nv, s->NVP, s->grid->d.order, s->stage_buf, row_len, cs, c0,
        s->S + size_t(field) * s->NVP, size_t(NF) * s->NVP, pad, zero_k0);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return THOR_OK;
}

// host canonical arrays -> Phi^n rows (through the staging buffer, permuted and padded on the device)
int upload_state(thor_state* s, const double* rho, const double* mom_h, const double* W, const double* p) {
    const HostGrid& h = s->grid->h;
    const int N = h.N, nv = h.nv;
    const size_t nc = size_t(N) * nv;
    int rc;
    if ((rc = put_row(s, rho, nc, nv, 1, 0, F_RHON, 1.0, 0))) return rc;
    if ((rc = put_row(s, p, nc, nv, 1, 0, F_PN, h.P.p_ref, 0))) return rc;
    if ((rc = put_row(s, mom_h, nc * 3, nv * 3, 3, 0, F_VXN, 0.0, 0))) return rc;
    if ((rc = put_row(s, nullptr, 0, nv * 3, 3, 1, F_VYN, 0.0, 0))) return rc;
    if ((rc = put_row(s, nullptr, 0, nv * 3, 3, 2, F_VZN, 0.0, 0))) return rc;
    // W: lower interfaces 0..nv-1 of the canonical [nv+1]; ground forced to 0 (rigid lid, L339)
    if ((rc = put_row(s, W, size_t(N) * (nv + 1), nv + 1, 1, 0, F_WN, 0.0, 1))) return rc;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(s->stream));
    return THOR_OK;
}

int upload_table(thor_state* s, const double* host, double** dev) {
    const HostGrid& h = s->grid->h;
    const int Npad = s->grid->d.Npad;
    const size_t nc = size_t(h.N) * h.nv;
    if (!*dev) CU(cudaMalloc(reinterpret_cast<void**>(dev), size_t(Npad) * s->NVP * sizeof(double)));
    CU(cudaMemcpyAsync(s->stage_buf, host, nc * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    k_rows_from_canonical<<<flat_blocks(size_t(Npad) * s->NVP), 256, 0, s->stream>>>(
        h.N, Npad, h.nv, s->NVP, s->grid->d.order, s->stage_buf, h.nv, 1, 0, *dev, size_t(s->NVP), 0.0, 0);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CU(cudaGetLastError());
    return THOR_OK;
}

// a5-a9: TMA-staged persistent kernel where a whole stage fits in shared memory, else the direct-load kernel
constexpr size_t kSmemPerBlockMax = 227 * 1024;
template <int G, int NS>
int launch_vertical_staged(const Geom& g, const DeviceGeom& d, double* S, double delta, int first, const TunePair& tn,
                           cudaStream_t st, bool* done) {
    constexpr int E = 2, NVP = G * E, TCOL = kTmaWarps * (32 / G);
    const size_t stage_doubles = size_t(TCOL) * kOwnRows * NVP + size_t(d.hmax) * kHaloRows * NVP + TCOL * 16 + TCOL;
    const size_t smem = NS * stage_doubles * sizeof(double) + NS * sizeof(unsigned long long);
    *done = false;
    if (d.hmax <= 0 || d.tcol != TCOL || smem > kSmemPerBlockMax) return THOR_OK;
    // the shared-memory opt-in is per device and per function: keyed on the device, set under a lock
    static std::mutex mu;
    static size_t configured[64] = {};
    static int sm_count[64] = {};
    int dev = 0, n_sm = 0;
    CU(cudaGetDevice(&dev));
    {
        std::lock_guard<std::mutex> lock(mu);
        const int slot = dev & 63;
        if (configured[slot] < smem) {
            CU(cudaFuncSetAttribute(k_vertical_staged<G, E, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)));
            CU(cudaDeviceGetAttribute(&sm_count[slot], cudaDevAttrMultiProcessorCount, dev));
            configured[slot] = smem;
        }
        n_sm = sm_count[slot];
    }
    const int ntiles = g.Npad / TCOL;
    const int grid = std::min(ntiles, n_sm * std::max(1, tn.tma_ctas));
    TileTab tt{d.tile_halo, d.tile_slots, d.hmax};
    k_vertical_staged<G, E, NS><<<grid, kTmaWarps * 32, smem, st>>>(g, tt, S, delta, first, ntiles, tn.k2.rev);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    *done = true;
    return THOR_OK;
}
int launch_vertical(const thor_grid* grid, const Geom& g, double* S, double delta, int first, const TunePair& tn,
                    cudaStream_t st, double* Xdd = nullptr) {
    const Shape sh = shape_for(g.nv);
    const DeviceGeom& d = grid->d;
    bool done = false;
    int rc = THOR_OK;
    if (tn.tma_stages >= 1 && sh.E == 2 && !Xdd) {
        const bool two = tn.tma_stages >= 2;
        if (sh.G == 4) rc = two ? launch_vertical_staged<4, 2>(g, d, S, delta, first, tn, st, &done) : launch_vertical_staged<4, 1>(g, d, S, delta, first, tn, st, &done);
        else if (sh.G == 8) rc = two ? launch_vertical_staged<8, 2>(g, d, S, delta, first, tn, st, &done) : launch_vertical_staged<8, 1>(g, d, S, delta, first, tn, st, &done);
        else if (sh.G == 16) rc = two ? launch_vertical_staged<16, 2>(g, d, S, delta, first, tn, st, &done) : launch_vertical_staged<16, 1>(g, d, S, delta, first, tn, st, &done);
        else rc = two ? launch_vertical_staged<32, 2>(g, d, S, delta, first, tn, st, &done) : launch_vertical_staged<32, 1>(g, d, S, delta, first, tn, st, &done);
        if (rc || done) return rc;
    }
    if (Xdd) THOR_DISPATCH(k_vertical_dd, g.nv, g.Npad, st, g, S, delta, first, tn.k2, Xdd);
    else THOR_DISPATCH(k_vertical, g.nv, g.Npad, st, g, S, delta, first, tn.k2);
    return THOR_OK;
}

// NEXT-3: the spring-dynamics relaxation of one refinement level on the current CUDA device (SpringFn of
// grid_host.h).  Same iteration and the same stopping test as the host loop, checked after every step (one 8-byte
// read back per step); positions in and out through the host array.
int spring_dynamics_device(int N, double* xyz, const int* nbr, const int* deg, const SpringParams& sp) {
    double *x = nullptr, *xn = nullptr, *v = nullptr;
    int *dn = nullptr, *dd = nullptr;
    unsigned long long* worst = nullptr;
    const size_t b3 = size_t(N) * 3 * sizeof(double);
    auto cleanup = [&]() { cudaFree(x); cudaFree(xn); cudaFree(v); cudaFree(dn); cudaFree(dd); cudaFree(worst); };
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&x), b3);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&xn), b3);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&v), b3);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&dn), size_t(N) * 6 * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&dd), size_t(N) * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&worst), sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemcpy(x, xyz, b3, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(v, 0, b3);
    if (e == cudaSuccess) e = cudaMemcpy(dn, nbr, size_t(N) * 6 * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dd, deg, size_t(N) * sizeof(int), cudaMemcpyHostToDevice);
    int it = 0;
    for (; e == cudaSuccess && it < sp.max_iter; ++it) {
        e = cudaMemsetAsync(worst, 0, sizeof(unsigned long long), nullptr);
        if (e != cudaSuccess) break;
        k_spring_step<<<(N + 127) / 128, 128>>>(N, x, xn, v, dn, dd, sp.dspr, sp.k, sp.alpha, sp.dt, worst);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        std::swap(x, xn);
        if (it >= sp.min_iter) {
            unsigned long long bits = 0;
            e = cudaMemcpy(&bits, worst, sizeof(bits), cudaMemcpyDeviceToHost);
            double w;
            std::memcpy(&w, &bits, sizeof(w));
            if (e == cudaSuccess && w < sp.tol) {
                ++it;
                break;
            }
        }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpy(xyz, x, b3, cudaMemcpyDeviceToHost);
    cleanup();
    if (e != cudaSuccess) {
        fail(THOR_ECUDA, std::string("thor_grid_create_device: spring dynamics: ") + cudaGetErrorString(e));
        return -1;
    }
    return it;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// thor_diagnostics_noalloc: the per-column partial sums of k_diag and the two results of k_sum_columns live in a
// file-scope device array instead of buffers from cudaMalloc.  Every GPU that loads the library holds the array
// (1 MiB + 256 B) until the process exits.  In HOST code the array's name is a host-side stand-in, not a device
// address: the address the kernels get comes from cudaGetSymbolAddress, looked up once per device with that device
// current.  All calls share the array: calls that overlap on the GPU race.
// ---------------------------------------------------------------------------------------------
constexpr int kNoAllocMaxCols = 65536;                       // grid levels 0..6 (level 6: 40 962 columns)
static __device__ __align__(256) double g_noalloc_scratch[2 * kNoAllocMaxCols + 32];

namespace {
int noalloc_scratch_address(double** out) {
    static std::mutex mu;
    static double* ptr[64] = {};
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(THOR_ECUDA, "thor_diagnostics_noalloc: device index out of range");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        CU(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_noalloc_scratch));
        if (!p) return fail(THOR_ECUDA, "thor_diagnostics_noalloc: cudaGetSymbolAddress returned a null address");
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return THOR_OK;
}
}  // namespace

extern "C" {

const char* thor_last_error(void) { return g_err.c_str(); }
long long thor_launch_count(void) { return g_launches.load(); }

static int grid_create(int level, int n_layers, const thor_planet* planet, const double* z_interfaces, int order_k,
                       SpringFn spring, thor_grid** out, bool shallow = false) {
    if (!planet || !out) return fail(THOR_EINVAL, "thor_grid_create: null argument");
    thor_grid* g = new (std::nothrow) thor_grid();
    if (!g) return fail(THOR_ENOMEM, "thor_grid_create: out of host memory");
    int rc;
    try {
        rc = build_host_grid(level, n_layers, *planet, g->h, z_interfaces, order_k, spring, shallow);
    } catch (const std::bad_alloc&) {
        delete g;
        return fail(THOR_ENOMEM, "thor_grid_create: out of host memory");
    }
    if (rc != THOR_OK) {
        delete g;
        if (rc == THOR_ECUDA) return rc;                 // the device spring loop has set the message
        return fail(rc, "thor_grid_create: invalid level, layer count, planet parameters, interface altitudes or order");
    }
    *out = g;
    return THOR_OK;
}

int thor_grid_create(int level, int n_layers, const thor_planet* planet, thor_grid** out) {
    return grid_create(level, n_layers, planet, nullptr, 1, nullptr, out);
}

int thor_grid_create_vertical(int level, int n_layers, const thor_planet* planet, const double* z_interfaces,
                              int order_k, thor_grid** out) {
    return grid_create(level, n_layers, planet, z_interfaces, order_k, nullptr, out);
}

int thor_grid_create_shallow(int level, int n_layers, const thor_planet* planet, const double* z_interfaces, thor_grid** out) {
    return grid_create(level, n_layers, planet, z_interfaces, 1, nullptr, out, true);
}

int thor_grid_create_device(int level, int n_layers, const thor_planet* planet, const double* z_interfaces,
                            int order_k, thor_grid** out) {
    int n = 0;
    const cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) return fail(THOR_ECUDA, std::string("thor_grid_create_device: no CUDA device: ") + cudaGetErrorString(e));
    return grid_create(level, n_layers, planet, z_interfaces, order_k, spring_dynamics_device, out);
}

int thor_grid_get(const thor_grid* grid, thor_grid_view* out) {
    if (!grid || !out) return fail(THOR_EINVAL, "thor_grid_get: null argument");
    const HostGrid& h = grid->h;
    out->level = h.level; out->n_cols = h.N; out->n_layers = h.nv;
    out->xyz = h.xyz.data(); out->nbr = h.nbr.data(); out->cv_vertex = h.cv.data();
    out->area = h.area.data(); out->edge_len = h.len.data(); out->edge_nrm = h.nrm.data();
    out->device_order = h.order.data();
    out->spring_iterations = h.spring_iterations;
    return THOR_OK;
}

void thor_grid_destroy(thor_grid* grid) {
    if (!grid) return;
    if (grid->d.ready) free_device_geom(grid->d);
    delete grid;
}

static void drop_graphs(thor_state* s);

void thor_state_destroy(thor_state* s) {
    if (!s) return;
    cudaFree(s->S); cudaFree(s->X); cudaFree(s->stage_buf); cudaFree(s->tab_Teq); cudaFree(s->tab_kT); cudaFree(s->tab_kv);
    cudaFree(s->col_mass); cudaFree(s->col_energy); cudaFree(s->efix_dev);
    drop_graphs(s);
    delete s;
}

int thor_state_init(const thor_grid* grid, const double* rho, const double* mom_h, const double* W,
                    const double* p, void* cuda_stream, thor_state** out) {
    if (!grid || !rho || !mom_h || !W || !p || !out) return fail(THOR_EINVAL, "thor_state_init: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    thor_state* s = new (std::nothrow) thor_state();
    if (!s) return fail(THOR_ENOMEM, "thor_state_init: out of host memory");
    s->grid = grid;
    s->stream = static_cast<cudaStream_t>(cuda_stream);
    const HostGrid& h = grid->h;
    const Shape sh = shape_for(h.nv);
    s->NVP = sh.G * sh.E;
    const size_t slab = size_t(grid->d.Npad) * NF * s->NVP;
    const size_t stage_n = std::max(size_t(h.N) * h.nv * 3, size_t(h.N) * (h.nv + 1));
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&s->S), slab * sizeof(double));
    if (e == cudaSuccess) e = cudaMemsetAsync(s->S, 0, slab * sizeof(double), s->stream);
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&s->stage_buf), stage_n * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&s->col_mass), h.N * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&s->col_energy), h.N * sizeof(double));
    if (e != cudaSuccess) {
        thor_state_destroy(s);
        return fail(e == cudaErrorMemoryAllocation ? THOR_ENOMEM : THOR_ECUDA,
                    std::string("thor_state_init: ") + cudaGetErrorString(e));
    }
    rc = upload_state(s, rho, mom_h, W, p);
    if (rc) {
        thor_state_destroy(s);
        return rc;
    }
    *out = s;
    return THOR_OK;
}

int thor_state_set(thor_state* s, const double* rho, const double* mom_h, const double* W, const double* p) {
    if (!s || !rho || !mom_h || !W || !p) return fail(THOR_EINVAL, "thor_state_set: null argument");
    return upload_state(s, rho, mom_h, W, p);
}

int thor_state_get(const thor_state* s, double* rho, double* mom_h, double* W, double* p) {
    if (!s || !rho || !mom_h || !W || !p) return fail(THOR_EINVAL, "thor_state_get: null argument");
    const HostGrid& h = s->grid->h;
    const int N = h.N, nv = h.nv;
    const size_t nc = size_t(N) * nv;
    const int* order = s->grid->d.order;
    cudaStream_t st = s->stream;
    auto scatter = [&](int field, int row_len, int cs, int c0) {
        k_rows_to_canonical<<<flat_blocks(nc), 256, 0, st>>>(N, nv, s->NVP, order, s->S + size_t(field) * s->NVP,
                                                             size_t(NF) * s->NVP, row_len, cs, c0, s->stage_buf);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    };
    scatter(F_RHON, nv, 1, 0);
    CU(cudaMemcpyAsync(rho, s->stage_buf, nc * sizeof(double), cudaMemcpyDeviceToHost, st));
    scatter(F_PN, nv, 1, 0);
    CU(cudaMemcpyAsync(p, s->stage_buf, nc * sizeof(double), cudaMemcpyDeviceToHost, st));
    scatter(F_VXN, nv * 3, 3, 0);
    scatter(F_VYN, nv * 3, 3, 1);
    scatter(F_VZN, nv * 3, 3, 2);
    CU(cudaMemcpyAsync(mom_h, s->stage_buf, nc * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    k_fill<<<flat_blocks(size_t(N) * (nv + 1)), 256, 0, st>>>(size_t(N) * (nv + 1), s->stage_buf, 0.0);   // lid = 0
    g_launches.fetch_add(1, std::memory_order_relaxed);
    scatter(F_WN, nv + 1, 1, 0);
    CU(cudaMemcpyAsync(W, s->stage_buf, size_t(N) * (nv + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
    return THOR_OK;
}

// the 2 (1 + n/2 + n) + 7 launches of one large step (Fig. 6), on the state's stream
static int launch_large_step(thor_state* s, const Geom& g, const TunePair& tn, const Forcing& F, double dt, int n) {
    const int nv = g.nv, Npad = g.Npad;
    cudaStream_t st = s->stream;
    double* S = s->S;
    // K_d = D dbar^4 / dt (Eq. 49), dbar = sqrt(2 pi / 5) A / 2^level (Eq. 2)
    const HostGrid& hg = s->grid->h;
    const double dbar = std::sqrt(2.0 * 3.14159265358979323846 / 5.0) * hg.P.radius / std::pow(2.0, hg.level);
    const double Kd_hyp = (s->X && s->D_hyp > 0.0) ? s->D_hyp * dbar * dbar * dbar * dbar / dt : 0.0;
    const double Kd_div = (s->X && s->D_div > 0.0) ? s->D_div * dbar * dbar * dbar * dbar / dt : 0.0;
    // every launch walks the columns opposite to the one before it (L2 hand-over)
    auto dir = [&](Tune t) { t.rev = tn.zigzag ? (s->walk ^= 1) : 0; return t; };
    // NEXT-4 (RE1): total mass and energy of a state in the Phi^n rows -> two device scalars
    auto sum_state = [&](double* out) {
        THOR_DISPATCH(k_diag, nv, Npad, st, g, S, s->col_mass, s->col_energy);
        k_sum_columns<<<1, 1024, 0, st>>>(hg.N, s->col_mass, s->col_energy, out);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    };
    if (s->efix) sum_state(s->efix_dev);
    for (int stage = 1; stage <= 3; ++stage) {                         // Eq. 30
        const int ns = stage == 1 ? 1 : (stage == 2 ? n / 2 : n);      // L252, L312-L316
        const double delta = stage == 1 ? dt / 3.0 : dt / n;
        // Fig. 6 large-steps 1-3; with NEXT-1 on, the same two kernels also produce w, the first Laplacians
        // (RD2) and D3^[t] (RD4), so that the only extra launch per stage is the second Laplacian
        const int dd = Kd_div > 0.0 ? (stage == 1 ? 2 : 1) : 0;
        THOR_DISPATCH(k_stage_prepare, nv, Npad, st, g, S, stage, delta, dir(tn.ks), Kd_hyp > 0.0 ? s->X : nullptr);
        // stage 1 without divergence damping: its explicit horizontal step V*' = delta slowV (Phi*(0) = 0) is written
        // by the kernel that holds the finished slow term (k_slow_terms, or k_diff2 with the hyper-diffusion on)
        const bool fuse1 = stage == 1 && !(Kd_div > 0.0);
        const double d1s = (fuse1 && !(Kd_hyp > 0.0)) ? delta : 0.0, d1d = (fuse1 && Kd_hyp > 0.0) ? delta : 0.0;
        if (Kd_hyp > 0.0) {
            if (hg.shallow) THOR_DISPATCH(k_slow_terms_hyp_sh, nv, Npad, st, g, S, dir(tn.ks), s->X, dd, 0.0);
            else if (g.kord == 3) THOR_DISPATCH(k_slow_terms_hyp_k3, nv, Npad, st, g, S, dir(tn.ks), s->X, dd, 0.0);
            else THOR_DISPATCH(k_slow_terms_hyp, nv, Npad, st, g, S, dir(tn.ks), s->X, dd, 0.0);
            THOR_DISPATCH(k_diff2, nv, Npad, st, g, S, s->X, Kd_hyp, dir(tn.ks), d1d);
        } else if (hg.shallow) {            // NEXT-4 (RS1): the shallow-atmosphere form is chosen here, on the host
            THOR_DISPATCH(k_slow_terms_sh, nv, Npad, st, g, S, dir(tn.ks), s->X, dd, d1s);
        } else if (g.kord == 3) {
            THOR_DISPATCH(k_slow_terms_k3, nv, Npad, st, g, S, dir(tn.ks), s->X, dd, d1s);
        } else {
            THOR_DISPATCH(k_slow_terms, nv, Npad, st, g, S, dir(tn.ks), s->X, dd, d1s);
        }
        for (int sub = 0; sub < ns; ++sub) {
            // stage 1: Phi*(0) = 0 exactly (Eq. 31 with Phi^[t] = Phi^n), so its substep reads no deviation row
            if (Kd_div > 0.0) {                                         // + Fig. 6 small-step 1
                if (stage == 1) THOR_DISPATCH(k_momentum_dd_stage1, nv, Npad, st, g, S, delta, dir(tn.k1), s->X, Kd_div, int(X_D3N));
                else THOR_DISPATCH(k_momentum_dd, nv, Npad, st, g, S, delta, dir(tn.k1), s->X, Kd_div, sub == 0 ? int(X_D3N) : int(X_D3));
            } else if (stage == 1) {
                // done by k_slow_terms / k_diff2 above
            } else {
                THOR_DISPATCH(k_momentum, nv, Npad, st, g, S, delta, dir(tn.k1));
            }
            TunePair t2 = tn;
            t2.k2 = dir(tn.k2);
            const int first = stage == 1 ? 2 : (sub == 0 ? 1 : 0);
            if (int rc = launch_vertical(s->grid, g, S, delta, first, t2, st, Kd_div > 0.0 ? s->X : nullptr)) return rc;
        }
    }
    if (s->efix) {
        // dynamics -> Phi^n rows without forcing; its mass and energy; one uniform temperature increment, then the forcing
        THOR_DISPATCH(k_finish, nv, Npad, st, g, S, Forcing{nullptr, nullptr, nullptr}, HeldSuarez{}, HotJupiter{}, dt, dir(tn.ks));
        sum_state(s->efix_dev + 2);
        THOR_DISPATCH(k_finish_fix, nv, Npad, st, g, S, F, s->hs, s->hj, dt, dir(tn.ks), s->efix_dev);
    } else {
        THOR_DISPATCH(k_finish, nv, Npad, st, g, S, F, s->hs, s->hj, dt, dir(tn.ks));
    }
    return THOR_OK;
}

static void drop_graphs(thor_state* s) {
    if (s->sexec) { cudaGraphExecDestroy(s->sexec); s->sexec = nullptr; }
    for (cudaGraphExec_t& e : s->gexec)
        if (e) { cudaGraphExecDestroy(e); e = nullptr; }
}

int thor_step(thor_state* s, int n_large, double dt, int n, const thor_forcing* forcing) {
    if (!s) return fail(THOR_EINVAL, "thor_step: null state");
    if (n_large < 0 || !(dt > 0) || n < 2 || (n & 1)) return fail(THOR_EINVAL, "thor_step: need n_large >= 0, dt > 0, even n >= 2");
    cudaStream_t st = s->stream;
    if (forcing && (s->hs.on || s->hj.on)) return fail(THOR_EINVAL, "thor_step: table forcing and evolving-sigma forcing are exclusive");
    if (forcing && forcing->resident && !(s->has_Teq || s->has_kT || s->has_kv))
        return fail(THOR_EINVAL, "thor_step: forcing->resident is set but no table was uploaded to this state");
    if (forcing && !forcing->resident) {
        int rc;
        s->has_Teq = forcing->T_eq != nullptr; s->has_kT = forcing->k_T != nullptr; s->has_kv = forcing->k_v != nullptr;
        if (s->has_Teq && (rc = upload_table(s, forcing->T_eq, &s->tab_Teq))) return rc;
        if (s->has_kT && (rc = upload_table(s, forcing->k_T, &s->tab_kT))) return rc;
        if (s->has_kv && (rc = upload_table(s, forcing->k_v, &s->tab_kv))) return rc;
    }
    Forcing F;
    F.T_eq = (forcing && s->has_Teq) ? s->tab_Teq : nullptr;
    F.k_T = (forcing && s->has_kT) ? s->tab_kT : nullptr;
    F.k_v = (forcing && s->has_kv) ? s->tab_kv : nullptr;
    const Geom g = make_geom(s->grid);
    const TunePair tn = tune();
    // CUDA graph of one large step: after a first directly launched step (which does every lazy
    // set-up), capture the launch sequence once per starting walk direction and replay it.  Small
    // grids are launch-bound (config 0: 33 launches of a few microseconds each).
    const bool use_graph = tn.graph && st != nullptr && s->stepped;
    if (use_graph) {
        thor_state::GraphKey key;
        std::memset(&key, 0, sizeof(key));
        key.dt = dt; key.n = n; key.efix = s->efix; key.D_hyp = s->D_hyp; key.D_div = s->D_div; key.hs = s->hs; key.hj = s->hj; key.Teq = F.T_eq; key.kT = F.k_T; key.kv = F.k_v;
        if (const char* e = std::getenv("THOR_B200_TUNE")) std::strncpy(key.tune, e, sizeof(key.tune) - 1);
        if (std::memcmp(&key, &s->gkey, sizeof(key)) != 0) {
            drop_graphs(s);
            std::memcpy(&s->gkey, &key, sizeof(key));
        }
    }
    for (int step = 0; step < n_large; ++step) {
        if (!use_graph) {
            if (int rc = launch_large_step(s, g, tn, F, dt, n)) return rc;
            continue;
        }
        const int w0 = s->walk & 1;
        if (!s->gexec[w0]) {
            const long long l0 = g_launches.load();
            cudaGraph_t graph = nullptr;
            CU(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
            const int rc = launch_large_step(s, g, tn, F, dt, n);
            const cudaError_t e = cudaStreamEndCapture(st, &graph);
            s->gwalk_end[w0] = s->walk;
            s->walk = w0;                                   // nothing ran yet
            s->gkernels = int(g_launches.load() - l0);
            g_launches.store(l0);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_step: graph capture: ") + cudaGetErrorString(e));
            const cudaError_t ei = cudaGraphInstantiate(&s->gexec[w0], graph, 0);
            cudaGraphDestroy(graph);
            if (ei != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_step: graph instantiate: ") + cudaGetErrorString(ei));
        }
        CU(cudaGraphLaunch(s->gexec[w0], st));
        s->walk = s->gwalk_end[w0];
        g_launches.fetch_add(s->gkernels, std::memory_order_relaxed);
    }
    CU(cudaGetLastError());
    s->stepped = s->stepped || n_large > 0;
    return THOR_OK;
}

int thor_state_set_diffusion(thor_state* s, double D_hyper, double D_div) {
    if (!s) return fail(THOR_EINVAL, "thor_state_set_diffusion: null state");
    if (!(D_hyper >= 0.0) || !(D_div >= 0.0)) return fail(THOR_EINVAL, "thor_state_set_diffusion: need D >= 0");
    if ((D_hyper > 0.0 || D_div > 0.0) && !s->X) {
        const size_t n = size_t(s->grid->d.Npad) * XF * s->NVP;
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&s->X), n * sizeof(double));
        if (e == cudaSuccess) e = cudaMemsetAsync(s->X, 0, n * sizeof(double), s->stream);
        if (e != cudaSuccess)
            return fail(e == cudaErrorMemoryAllocation ? THOR_ENOMEM : THOR_ECUDA,
                        std::string("thor_state_set_diffusion: ") + cudaGetErrorString(e));
    }
    s->D_hyp = D_hyper;
    s->D_div = D_div;
    return THOR_OK;
}

int thor_state_set_energy_fixer(thor_state* s, int on) {
    if (!s) return fail(THOR_EINVAL, "thor_state_set_energy_fixer: null state");
    if (on && !s->efix_dev) {
        const cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&s->efix_dev), 4 * sizeof(double));
        if (e != cudaSuccess)
            return fail(e == cudaErrorMemoryAllocation ? THOR_ENOMEM : THOR_ECUDA,
                        std::string("thor_state_set_energy_fixer: ") + cudaGetErrorString(e));
    }
    s->efix = on ? 1 : 0;
    return THOR_OK;
}

int thor_state_set_held_suarez(thor_state* s, const thor_held_suarez* hs) {
    if (!s) return fail(THOR_EINVAL, "thor_state_set_held_suarez: null state");
    if (!hs) {
        std::memset(&s->hs, 0, sizeof(s->hs));
        return THOR_OK;
    }
    if (!(hs->sigma_b >= 0.0 && hs->sigma_b < 1.0) || !(hs->p_star > 0.0) || !(hs->k_a >= 0.0) || !(hs->k_s >= 0.0) || !(hs->k_f >= 0.0))
        return fail(THOR_EINVAL, "thor_state_set_held_suarez: need 0 <= sigma_b < 1, p_star > 0, rates >= 0");
    if (s->hj.on) return fail(THOR_EINVAL, "thor_state_set_held_suarez: hot-Jupiter forcing is on");
    std::memset(&s->hs, 0, sizeof(s->hs));
    s->hs.on = 1;
    s->hs.T_surf = hs->T_surf; s->hs.dT_y = hs->dT_y; s->hs.dth_z = hs->dth_z; s->hs.T_min = hs->T_min;
    s->hs.k_a = hs->k_a; s->hs.k_s = hs->k_s; s->hs.k_f = hs->k_f; s->hs.sigma_b = hs->sigma_b; s->hs.p_star = hs->p_star;
    return THOR_OK;
}

int thor_state_set_hot_jupiter(thor_state* s, const thor_hot_jupiter* hj) {
    if (!s) return fail(THOR_EINVAL, "thor_state_set_hot_jupiter: null state");
    std::memset(&s->hj, 0, sizeof(s->hj));
    if (!hj) return THOR_OK;
    if (!(hj->tau_rad > 0.0) || !(hj->sigma_stra >= 0.0 && hj->sigma_stra < 1.0))
        return fail(THOR_EINVAL, "thor_state_set_hot_jupiter: need tau_rad > 0, 0 <= sigma_stra < 1");
    if (s->hs.on) return fail(THOR_EINVAL, "thor_state_set_hot_jupiter: Held-Suarez forcing is on");
    s->hj.on = 1;
    s->hj.T_surf = hj->T_surf; s->hj.Gamma = hj->Gamma; s->hj.dT_stra = hj->dT_stra; s->hj.z_stra = hj->z_stra;
    s->hj.sigma_stra = hj->sigma_stra; s->hj.dT_EP = hj->dT_EP; s->hj.tau_rad = hj->tau_rad;
    return THOR_OK;
}

int thor_acoustic_substeps(thor_state* s, int n_substeps, double delta, int which) {
    if (!s) return fail(THOR_EINVAL, "thor_acoustic_substeps: null state");
    if (n_substeps < 0 || !(delta > 0) || which < 1 || which > 3) return fail(THOR_EINVAL, "thor_acoustic_substeps: bad argument");
    if (!s->stepped) return fail(THOR_EINVAL, "thor_acoustic_substeps: call thor_step first (no stage data yet)");
    const HostGrid& h = s->grid->h;
    const int Npad = s->grid->d.Npad;
    const Geom g = make_geom(s->grid);
    const TunePair tn = tune();
    auto dir = [&](Tune t) { t.rev = tn.zigzag ? (s->walk ^= 1) : 0; return t; };
    auto launch_all = [&]() -> int {
        for (int i = 0; i < n_substeps; ++i) {
            if (which & 1) THOR_DISPATCH(k_momentum, h.nv, Npad, s->stream, g, s->S, delta, dir(tn.k1));
            TunePair t2 = tn;
            if (which & 2) t2.k2 = dir(tn.k2);
            if (which & 2)
                if (int rc = launch_vertical(s->grid, g, s->S, delta, 0, t2, s->stream)) return rc;
        }
        return THOR_OK;
    };
    // as in thor_step: on a non-default stream the sequence is captured once and replayed (the substep kernels run
    // back to back inside a large step's graph; timing them with per-launch host gaps would measure the host)
    if (!(tn.graph && s->stream != nullptr && n_substeps > 0)) {
        if (int rc = launch_all()) return rc;
        CU(cudaGetLastError());
        return THOR_OK;
    }
    thor_state::SubKey key;
    std::memset(&key, 0, sizeof(key));
    key.delta = delta; key.n = n_substeps; key.which = which; key.walk0 = s->walk & 1;
    if (const char* e = std::getenv("THOR_B200_TUNE")) std::strncpy(key.tune, e, sizeof(key.tune) - 1);
    if (!s->sexec || std::memcmp(&key, &s->skey, sizeof(key)) != 0) {
        if (s->sexec) { cudaGraphExecDestroy(s->sexec); s->sexec = nullptr; }
        const long long l0 = g_launches.load();
        const int w0 = s->walk;
        cudaGraph_t graph = nullptr;
        CU(cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
        const int rc = launch_all();
        const cudaError_t e = cudaStreamEndCapture(s->stream, &graph);
        s->swalk_end = s->walk;
        s->walk = w0;
        s->skernels = int(g_launches.load() - l0);
        g_launches.store(l0);
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_acoustic_substeps: graph capture: ") + cudaGetErrorString(e));
        const cudaError_t ei = cudaGraphInstantiate(&s->sexec, graph, 0);
        cudaGraphDestroy(graph);
        if (ei != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_acoustic_substeps: graph instantiate: ") + cudaGetErrorString(ei));
        std::memcpy(&s->skey, &key, sizeof(key));
    }
    CU(cudaGraphLaunch(s->sexec, s->stream));
    s->walk = s->swalk_end;
    g_launches.fetch_add(s->skernels, std::memory_order_relaxed);
    CU(cudaGetLastError());
    return THOR_OK;
}

int thor_diagnostics(const thor_state* s, thor_diag* out) {
    if (!s || !out) return fail(THOR_EINVAL, "thor_diagnostics: null argument");
    const HostGrid& h = s->grid->h;
    const Geom g = make_geom(s->grid);
    THOR_DISPATCH(k_diag, h.nv, s->grid->d.Npad, s->stream, g, s->S, s->col_mass, s->col_energy);
    CU(cudaGetLastError());
    std::vector<double> m(h.N), e(h.N);
    CU(cudaMemcpyAsync(m.data(), s->col_mass, h.N * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CU(cudaMemcpyAsync(e.data(), s->col_energy, h.N * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    // Neumaier-compensated sum of the per-column partials
    auto ksum = [](const std::vector<double>& v) {
        double sum = 0.0, c = 0.0;
        for (double x : v) {
            double t = sum + x;
            c += (std::fabs(sum) >= std::fabs(x)) ? (sum - t) + x : (x - t) + sum;
            sum = t;
        }
        return sum + c;
    };
    out->total_mass = ksum(m);
    out->total_energy = ksum(e);
    return THOR_OK;
}

int thor_diagnostics_noalloc(const thor_state* s, thor_diag* out) {
    if (!s || !out) return fail(THOR_EINVAL, "thor_diagnostics_noalloc: null argument");
    const HostGrid& h = s->grid->h;
    if (h.N > kNoAllocMaxCols)
        return fail(THOR_EINVAL, "thor_diagnostics_noalloc: " + std::to_string(h.N) + " columns exceed the static scratch of " +
                                     std::to_string(kNoAllocMaxCols) + " columns (grid level <= 6); use thor_diagnostics");
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev != s->grid->d.device)
        return fail(THOR_EINVAL, "thor_diagnostics_noalloc: state lives on CUDA device " + std::to_string(s->grid->d.device) +
                                     ", current device is " + std::to_string(dev));
    double* scratch = nullptr;
    if (int rc = noalloc_scratch_address(&scratch)) return rc;
    double *col_mass = scratch, *col_energy = scratch + kNoAllocMaxCols, *res = scratch + 2 * kNoAllocMaxCols;
    const Geom g = make_geom(s->grid);
    // the array keeps the last call's contents: the two result slots are cleared so that a launch that did not run
    // cannot hand back the previous call's numbers; the per-column slots 0..N-1 are all rewritten by k_diag
    CU(cudaMemsetAsync(res, 0, 2 * sizeof(double), s->stream));
    THOR_DISPATCH(k_diag, h.nv, s->grid->d.Npad, s->stream, g, s->S, col_mass, col_energy);
    k_sum_columns<<<1, 1024, 0, s->stream>>>(h.N, col_mass, col_energy, res);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CU(cudaGetLastError());
    double r[2] = {0.0, 0.0};
    CU(cudaMemcpyAsync(r, res, sizeof(r), cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    out->total_mass = r[0];
    out->total_energy = r[1];
    return THOR_OK;
}

int thor_apply_div_device(const thor_grid* grid, const double* vx, const double* vy, const double* vz,
                          double* out, void* cuda_stream) {
    if (!grid || !vx || !vy || !vz || !out) return fail(THOR_EINVAL, "thor_apply_div_device: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    const Geom g = make_geom(grid);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (op_fast_path(g.nv, {vx, vy, vz, out})) THOR_DISPATCH_OP2(k_div2, g.nv, g.N, st, g, vx, vy, vz, out);
    else THOR_DISPATCH_OP(k_div, g.nv, g.N, st, g, vx, vy, vz, out);
    CU(cudaGetLastError());
    return THOR_OK;
}

int thor_apply_grad_device(const thor_grid* grid, const double* sfield, double* gx, double* gy, double* gz,
                           void* cuda_stream) {
    if (!grid || !sfield || !gx || !gy || !gz) return fail(THOR_EINVAL, "thor_apply_grad_device: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    const Geom g = make_geom(grid);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (op_fast_path(g.nv, {sfield, gx, gy, gz})) THOR_DISPATCH_OP2(k_grad2, g.nv, g.N, st, g, sfield, gx, gy, gz);
    else THOR_DISPATCH_OP(k_grad, g.nv, g.N, st, g, sfield, gx, gy, gz);
    CU(cudaGetLastError());
    return THOR_OK;
}

int thor_apply_lap_device(const thor_grid* grid, const double* sfield, double* out, void* cuda_stream) {
    if (!grid || !sfield || !out) return fail(THOR_EINVAL, "thor_apply_lap_device: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    const Geom g = make_geom(grid);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (op_fast_path(g.nv, {sfield, out})) THOR_DISPATCH_OP2(k_lap2, g.nv, g.N, st, g, sfield, out);
    else THOR_DISPATCH_OP(k_lap, g.nv, g.N, st, g, sfield, out);
    CU(cudaGetLastError());
    return THOR_OK;
}

int thor_apply_lap(const thor_grid* grid, const double* sfield, double* out) {
    if (!grid || !sfield || !out) return fail(THOR_EINVAL, "thor_apply_lap: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    const HostGrid& h = grid->h;
    const int N = h.N, nv = h.nv;
    const size_t nc = size_t(N) * nv;
    double* buf = nullptr;   // [staging][s][out]
    if (int rb = op_scratch(grid, &buf)) return rb;
    double *stg = buf, *sd = buf + nc, *od = sd + nc;
    cudaError_t e = cudaMemcpy(stg, sfield, nc * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_gather_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, stg, nv, 1, 0, sd);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        rc = thor_apply_lap_device(grid, sd, od, nullptr);
        if (rc == THOR_OK) {
            k_scatter_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, od, nv, 1, 0, stg);
            g_launches.fetch_add(1, std::memory_order_relaxed);
            e = cudaMemcpy(out, stg, nc * sizeof(double), cudaMemcpyDeviceToHost);
        }
    }
    if (rc) return rc;
    if (e != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_apply_lap: ") + cudaGetErrorString(e));
    return THOR_OK;
}

// host wrappers of the two operators: upload, permute, run, permute back, download
int thor_apply_div(const thor_grid* grid, const double* vec, double* out) {
    if (!grid || !vec || !out) return fail(THOR_EINVAL, "thor_apply_div: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    const HostGrid& h = grid->h;
    const int N = h.N, nv = h.nv;
    const size_t nc = size_t(N) * nv;
    double* buf = nullptr;   // [3nc staging][vx][vy][vz][out]
    if (int rb = op_scratch(grid, &buf)) return rb;
    double *stg = buf, *vx = buf + 3 * nc, *vy = vx + nc, *vz = vy + nc, *o = vz + nc;
    cudaError_t e = cudaMemcpy(stg, vec, 3 * nc * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_gather_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, stg, nv * 3, 3, 0, vx);
        k_gather_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, stg, nv * 3, 3, 1, vy);
        k_gather_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, stg, nv * 3, 3, 2, vz);
        g_launches.fetch_add(3, std::memory_order_relaxed);
        rc = thor_apply_div_device(grid, vx, vy, vz, o, nullptr);
        if (rc == THOR_OK) {
            k_scatter_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, o, nv, 1, 0, stg);
            g_launches.fetch_add(1, std::memory_order_relaxed);
            e = cudaMemcpy(out, stg, nc * sizeof(double), cudaMemcpyDeviceToHost);
        }
    }
    if (rc) return rc;
    if (e != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_apply_div: ") + cudaGetErrorString(e));
    return THOR_OK;
}

int thor_apply_grad(const thor_grid* grid, const double* sfield, double* out) {
    if (!grid || !sfield || !out) return fail(THOR_EINVAL, "thor_apply_grad: null argument");
    int rc = ensure_device_geom(grid);
    if (rc) return rc;
    const HostGrid& h = grid->h;
    const int N = h.N, nv = h.nv;
    const size_t nc = size_t(N) * nv;
    double* buf = nullptr;   // [3nc staging][s][gx][gy][gz]
    if (int rb = op_scratch(grid, &buf)) return rb;
    double *stg = buf, *sd = buf + 3 * nc, *gx = sd + nc, *gy = gx + nc, *gz = gy + nc;
    cudaError_t e = cudaMemcpy(stg, sfield, nc * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_gather_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, stg, nv, 1, 0, sd);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        rc = thor_apply_grad_device(grid, sd, gx, gy, gz, nullptr);
        if (rc == THOR_OK) {
            k_scatter_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, gx, nv * 3, 3, 0, stg);
            k_scatter_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, gy, nv * 3, 3, 1, stg);
            k_scatter_rows<<<flat_blocks(nc), 256>>>(N, nv, grid->d.order, gz, nv * 3, 3, 2, stg);
            g_launches.fetch_add(3, std::memory_order_relaxed);
            e = cudaMemcpy(out, stg, 3 * nc * sizeof(double), cudaMemcpyDeviceToHost);
        }
    }
    if (rc) return rc;
    if (e != cudaSuccess) return fail(THOR_ECUDA, std::string("thor_apply_grad: ") + cudaGetErrorString(e));
    return THOR_OK;
}

}  // extern "C"
