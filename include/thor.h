/*
 * thor.h -- C-ABI boundary of the B200-native THOR HE-VI hot path (arXiv 1607.05535).
 *
 * One FP64 large time step of the horizontally-explicit / vertically-implicit split-explicit
 * integrator (Fig. 6) on a spring-smoothed icosahedral grid (L43-L125), the
 * PROFX forcing (Eq. 51-52) and the conserved diagnostics (L190, L200, L339).
 * Citations are PAPER.md:L<line> + equation; R-n / G-n are the readings listed in DESIGN.md.
 *
 * Conventions
 *  - Every function returns THOR_OK (0) or a negative code; nothing is written to outputs on
 *    failure; no exception crosses the boundary; thor_last_error() gives the message of the last
 *    failure on the calling thread.
 *  - Unless a parameter is marked DEVICE, pointers are HOST pointers.  The caller owns every array
 *    it passes in or receives results in; the library copies.  Opaque handles are owned by the
 *    caller and released with the matching _destroy.
 *  - Arrays at the boundary are FP64, C-contiguous, in CANONICAL column order (the grid
 *    generator's numbering), layer index fastest:
 *        rho, p, T_eq, k_T, k_v : [n_cols][n_layers]        at layer centres
 *        mom_h = rho v_h        : [n_cols][n_layers][3]     Cartesian, tangent to the sphere
 *        W     = rho v_r        : [n_cols][n_layers+1]      on layer interfaces, index 0 = bottom;
 *                                 both ends are the rigid lid (L339) and are forced to 0.
 *    The device keeps a different, locality-preserving column order; it is internal
 *    (thor_grid_view.device_order documents it for the *_device entry points).
 *  - Layers are uniform in altitude unless thor_grid_create_vertical says otherwise: dz = z_top / n_layers,
 *    centre k at (k+1/2) dz (R6).
 *  - thor_step and thor_acoustic_substeps are asynchronous on the stream given to thor_state_init;
 *    thor_state_get, thor_state_set and thor_diagnostics synchronise that stream.
 *  - On a non-default stream thor_step replays a large step as a CUDA graph after the first directly
 *    launched one (same kernels, same results).  The environment variable THOR_B200_TUNE
 *    ("zigzag,k1_ahead,k2_ahead,tail,tma_stages,tma_ctas,stage_ahead,graph")
 *    overrides the launch schedule for measurement; it never changes what is computed.
 *  - The library never falls back to the CPU: without a usable CUDA device every device entry
 *    point returns THOR_ECUDA.  thor_grid_create / thor_grid_get are host-only and need no GPU.
 */
#ifndef THOR_H_
#define THOR_H_

#ifdef __cplusplus
extern "C" {
#endif

#define THOR_OK      0
#define THOR_EINVAL (-1)  /* null pointer, level < 0 or > 9, n_layers < 2 or > 128, dt <= 0, odd or < 2 substep count */
#define THOR_ENOMEM (-2)
#define THOR_ECUDA  (-3)  /* CUDA runtime failure or no device */

/* Planet and domain (Table 1; p_ref L213; model top L454).  SI units. */
typedef struct {
    double radius;   /* A, m */
    double omega;    /* rotation rate about the axis through the two polar vertices (L45), 1/s */
    double gravity;  /* constant, radial (L184; R11), m/s^2 */
    double Rd;       /* gas constant, J/kg/K */
    double Cp;       /* specific heat at constant pressure, J/kg/K */
    double p_ref;    /* reference pressure of Eq. 24, Pa */
    double z_top;    /* altitude of the rigid lid, m */
} thor_planet;

typedef struct thor_grid thor_grid;    /* host geometry (+ device copy, made on first device use) */
typedef struct thor_state thor_state;  /* device prognostics, stage arrays and work space */

/* Read-only view of the generated grid; pointers are owned by the grid and live as long as it. */
typedef struct {
    int level, n_cols, n_layers;
    const double *xyz;          /* [n_cols][3] unit-sphere positions P_i after spring dynamics and centroid move */
    const int *nbr;             /* [n_cols][6] neighbours, counter-clockwise seen from outside; pentagons: nbr[5] = -1 */
    const double *cv_vertex;    /* [n_cols][6][3] control-volume vertices C_k (Fig. 2); C_k belongs to the triangle
                                   (P_0, P_nbr[k], P_nbr[k+1]); fixed while P moves (L120) */
    const double *area;         /* [n_cols] unit-sphere control-volume areas A_c (sum = 4 pi) */
    const double *edge_len;     /* [n_cols][6] geodesic arc C_k..C_k+1, l_k of Eq. 4 */
    const double *edge_nrm;     /* [n_cols][6][3] outward unit normal of that arc, n_k of Eq. 4 */
    const int *device_order;    /* [n_cols] canonical index of the column stored at device slot d */
    int spring_iterations;      /* total spring-dynamics steps taken by the generator (all levels) */
} thor_grid_view;

/* PROFX tables (Eq. 51-52; R9: fixed in time).  Any pointer may be NULL = that term is off
 * (Newtonian relaxation needs both T_eq and k_T).  resident != 0: reuse the tables uploaded by
 * the previous thor_step call on this state (no host read, no copy). */
typedef struct {
    const double *T_eq;  /* K   */
    const double *k_T;   /* 1/s */
    const double *k_v;   /* 1/s */
    int resident;
} thor_forcing;

typedef struct { double total_mass, total_energy; } thor_diag;

/* Grid (L43-L125): icosahedron with two polar vertices -> `level` edge bisections (Eq. 1:
 * n_cols = 10*4^level + 2) -> spring dynamics (Eq. 10-12, beta = 1.15) -> centroid move (Eq. 13);
 * then the finite-volume stencil weights of Eq. 4-7 and the device column order.  Host only. */
int thor_grid_create(int level, int n_layers, const thor_planet *planet, thor_grid **out);
/* NEXT-3 (section 2.2, Eq. 8-9): the same grid with layers of unequal thickness and/or the vertical
 * Lagrange interpolation of order k > 1.  z_interfaces: n_layers+1 strictly increasing altitudes, z_interfaces[0] = 0,
 * the last one is the rigid lid and REPLACES planet->z_top; NULL = uniform layers.  Layer centres sit midway between
 * their interfaces.  order_k: 1 (the paper's choice, L94) or 3; it enters the explicit slow terms (vertical fluxes of
 * u, h, theta; I_h[rho] and I_h[F_r] of Eq. 42; I_c[W]; w = W/I_h[rho] of the hyper-diffusion), while the implicit
 * acoustic system keeps k = 1 and stays tridiagonal (reading RV2).  Order 3 uses the two nearest nodes on each side
 * of the target; where the column ends first the missing nodes are dropped (RV1).  Other orders: THOR_EINVAL. */
int thor_grid_create_vertical(int level, int n_layers, const thor_planet *planet, const double *z_interfaces,
                              int order_k, thor_grid **out);
/* NEXT-4 (section 3): the same grid for the SHALLOW-ATMOSPHERE approximation, one of the three the paper says
 * "have been implemented in the model and the user can switch them on and off" (L184) without printing their
 * equations.  Reading RS1: (i) every radius in the discrete operators is the planetary radius A (horizontal
 * operators over A, the vertical divergence without its r^2 factors, cell volume A_c A^2 dz); (ii) Coriolis from the
 * radial component of Omega only, f r x V with f = 2 Omega sin(lat), on the horizontal momentum alone; (iii) no metric
 * coupling between horizontal and vertical motion: the horizontal equation advects the horizontal velocity, the
 * vertical one advects w as a scalar.  States made on this grid are stepped with those equations; everything else
 * (acoustic substeps, NEXT-1, forcings, diagnostics) is the same code reading the changed per-layer tables.
 * z_interfaces as in thor_grid_create_vertical (NULL = uniform layers); the vertical interpolation is linear. */
int thor_grid_create_shallow(int level, int n_layers, const thor_planet *planet, const double *z_interfaces,
                             thor_grid **out);
/* NEXT-3 (section 2.3, Eq. 10-12): the same grid with the spring-dynamics relaxation -- by far the slowest
 * part of set-up from level 6 on -- iterated on the current CUDA device (one kernel launch per step, the same update
 * and the same stopping test as the host loop; positions agree with thor_grid_create's to rounding accumulated over the
 * iteration, far inside the stopping tolerance).  Bisection, centroid move, stencil weights and the device column order
 * stay on the host.  Arguments as thor_grid_create_vertical.  THOR_ECUDA without a usable device. */
int thor_grid_create_device(int level, int n_layers, const thor_planet *planet, const double *z_interfaces,
                            int order_k, thor_grid **out);
int thor_grid_get(const thor_grid *grid, thor_grid_view *out);
void thor_grid_destroy(thor_grid *grid);

/* State: uploads the four prognostic fields (L333) and allocates all stage/work arrays on the
 * current CUDA device.  cuda_stream is a cudaStream_t (NULL = default stream). */
int thor_state_init(const thor_grid *grid, const double *rho, const double *mom_h, const double *W,
                    const double *p, void *cuda_stream, thor_state **out);
int thor_state_set(thor_state *state, const double *rho, const double *mom_h, const double *W, const double *p);
int thor_state_get(const thor_state *state, double *rho, double *mom_h, double *W, double *p);
void thor_state_destroy(thor_state *state);

/* n_large large steps of Fig. 6 (L301-L337): per step three Runge-Kutta stages (Eq. 30) of
 * slow terms (RHS of Eq. 32-35, 42) + 1, n/2, n acoustic substeps (Eq. 33, 37, 32, 35, 36; L252),
 * then the forcing (NULL = none) with the large step dt (L385).  n_acoustic_substeps = n, even, >= 2. */
int thor_step(thor_state *state, int n_large, double dt, int n_acoustic_substeps, const thor_forcing *forcing);

/* NEXT-1 (section 4 of the paper, Eq. 43-50): switch on the explicit fourth-order hyper-diffusion of
 * rho, v_h, v_r and T (per Runge-Kutta stage, Fig. 6 large-step 2) and the 3-D divergence damping
 * (per acoustic substep, Fig. 6 small-step 1) for the following thor_step calls.  D_hyper, D_div are
 * the non-dimensional parameter of Eq. 49, K_d = D dbar^4 / dt with dbar of Eq. 2; the paper uses the
 * same value for both (L367; 0.004837 for its Earth run, 0.01992 for its hot Jupiter, from Table 1).
 * 0 switches a term off; (0, 0), the default, is the base path.  Allocates the work rows on first use. */
int thor_state_set_diffusion(thor_state *state, double D_hyper, double D_div);

/* NEXT-2 (section 7.1, Eq. 51-55): the Held-Suarez forcing with K_v, K_T and T_eq evaluated from the
 * EVOLVING state instead of fixed tables: sigma = p/p_s, p_s extrapolated hydrostatically and
 * isothermally from the lowest layer centre (L390);
 *   K_v = k_f max(0, (sigma - sigma_b)/(1 - sigma_b))                                          (Eq. 53)
 *   T_eq = max{T_min, [T_surf - dT_y sin^2(lat) - dth_z ln(p/p_star) cos^2(lat)] (p/p_star)^(Rd/Cp)}   (Eq. 54)
 *   K_T = k_a + (k_s - k_a) max(0, (sigma - sigma_b)/(1 - sigma_b)) cos^4(lat)                  (Eq. 55)
 * applied with Eq. 51-52 at the end of every large step.  hs = NULL switches it off.  While it is on,
 * thor_step must be called with forcing = NULL (THOR_EINVAL otherwise). */
typedef struct {
    double T_surf, dT_y, dth_z, T_min;   /* K: 315, 60 (L448), (Delta theta)_z (not printed in the paper), 200 */
    double k_a, k_s, k_f;                /* 1/s: 1/(40 d), 1/(4 d), 1/(1 d)  (L438, L448) */
    double sigma_b, p_star;              /* 0.7; reference pressure of Eq. 54, Pa */
} thor_held_suarez;
int thor_state_set_held_suarez(thor_state *state, const thor_held_suarez *hs);

/* NEXT-2, hot Jupiter (section 7.2, Eq. 59-61): T_eq = T_vert(z) + beta_trop(sigma, z) dT_EP cos(lon) cos(lat),
 * beta_trop = sin(pi (sigma - sigma_stra)/(2 (1 - sigma_stra))) below z_stra (clamped at 0), 0 above;
 * T_vert by Eq. 61; K_T = 1/tau_rad; no drag (L512).  The substellar point is on the +x axis.
 * hj = NULL switches it off; exclusive with the tables and with the Held-Suarez forcing. */
typedef struct {
    double T_surf, Gamma, dT_stra, z_stra;   /* 1600 K, 2e-4 K/m, 10 K, 2e6 m  (L527) */
    double sigma_stra, dT_EP, tau_rad;       /* 0.12, 300 K, 1.5e5 s           (L516-L529) */
} thor_hot_jupiter;
int thor_state_set_hot_jupiter(thor_state *state, const thor_hot_jupiter *hj);

/* NEXT-4 (L215): the energy fixer "proposed by Williamson et al. (2009), which globally uniform adjusts the internal
 * energy at all grid points".  Reading RE1: after the dynamics of every large step and before its forcing, the total
 * energy (as thor_diagnostics defines it) is brought back to its value before the step by ONE temperature increment for
 * all cells, dT = (E - E')/(Cv M); rho is unchanged, p <- p + rho Rd dT.  The sums run on the device (k_diag partial
 * sums per column, one-block compensated sum).  on = 0 (the default, and what the paper's runs use): off. */
int thor_state_set_energy_fixer(thor_state *state, int on);

/* Only the hot loop: n_substeps acoustic substeps (steps a4-a9 of DESIGN.md) of length delta on the
 * stage data left by the last thor_step.  which: 1 = explicit horizontal momentum kernel only,
 * 2 = divergence + column-solve kernel only, 3 = both.  For measurement; the state it leaves is
 * not a physical one. */
int thor_acoustic_substeps(thor_state *state, int n_substeps, double delta, int which);

/* Total mass sum(rho A_c r_k^2 dz) and total energy sum((Cv p/Rd + |rho v|^2/(2 rho) + rho g z) A_c r_k^2 dz) (R10). */
int thor_diagnostics(const thor_state *state, thor_diag *out);

/* The same diagnostics for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no cudaMalloc, cudaFree or host allocation in this call.  The per-column partial
 * sums and the two results live in a file-scope device array of the library (1 MiB, held by every GPU that loads the
 * library until the process exits) and are summed on the device (one block, compensated partial sums, fixed order):
 * the result agrees with thor_diagnostics to rounding of the sum (relative 1e-15), not bit for bit.
 * Limit: at most 65 536 columns, i.e. grid levels 0..6; larger grids get THOR_EINVAL (use thor_diagnostics).
 * Every call, on every state, shares that array and it keeps the last call's contents (the call clears what it must):
 * calls that overlap on the GPU (different streams or threads) race -- serialise them.  Synchronises the state's
 * stream; the state must live on the current device. */
int thor_diagnostics_noalloc(const thor_state *state, thor_diag *out);

/* Config-1 operators at radius r_k (unit-sphere operator / r_k): Eq. 6 divergence of vec
 * [n_cols][n_layers][3] -> out [n_cols][n_layers]; Eq. 7 gradient (difference form, projected with
 * Eq. 28) of s [n_cols][n_layers] -> out [n_cols][n_layers][3].  Host arrays, canonical order. */
int thor_apply_div(const thor_grid *grid, const double *vec, double *out);
int thor_apply_grad(const thor_grid *grid, const double *s, double *out);

/* The same two kernels on DEVICE arrays already in device column order, component-separated:
 * each pointer is a DEVICE [n_cols][n_layers] array.  Asynchronous on cuda_stream. */
int thor_apply_div_device(const thor_grid *grid, const double *vx, const double *vy, const double *vz,
                          double *out, void *cuda_stream);
int thor_apply_grad_device(const thor_grid *grid, const double *s, double *gx, double *gy, double *gz,
                           void *cuda_stream);

/* Horizontal Laplacian of L369-L371 (the building block of the paper's fourth-order hyper-diffusion,
 * Eq. 43-48): the Eq. 7 gradient on the primary (triangle) grid, which places a vector at every
 * control-volume corner, then Eq. 6 over the control volume; at radius r_k (unit-sphere operator
 * / r_k^2).  s, out: [n_cols][n_layers]; host arrays in canonical order, or DEVICE arrays in device
 * column order for the _device variant (asynchronous on cuda_stream). */
int thor_apply_lap(const thor_grid *grid, const double *s, double *out);
int thor_apply_lap_device(const thor_grid *grid, const double *s, double *out, void *cuda_stream);

/* Number of kernels this library has launched in the calling process so far. */
long long thor_launch_count(void);

const char *thor_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* THOR_H_ */
