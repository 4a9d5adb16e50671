/* dgvlasov.h -- C ABI of the B200-native tensor-product DG Vlasov-Poisson hot path.
 *
 * Method: D. W. Crews, "Analysis of tensor-product discontinuous Galerkin operators for
 * Vlasov-Poisson simulations and GPU implementation on Python", arXiv 2202.13532.
 * Citations below are "PAPER.md:<line>" (the text under /root/reference) plus the equation.
 *
 * Conventions
 *  - Phase-space dimensions d = 0,1,2 are (x, u, v) = (x, v_x, v_y)  [ndim = 3, 1D2V] or
 *    (x, v) [ndim = 2, 1D1V]; ndim = 1 describes x only (field-solve-only context).
 *  - N_d elements and n_d LGL nodes per element in dimension d; global node index
 *    g_d = a_d * n_d + b_d (element a, node b).  Interface nodes are duplicated.
 *  - The distribution is ONE dense row-major FP64 array f[g_x][g_u][g_v] (f[g_x][g_v] for
 *    ndim = 2): the paper's u[a0,b0,a1,b1,a2,b2] in C order (Section 3.1).
 *  - Every pointer named *_dev is a DEVICE pointer owned by the caller (e.g. a torch
 *    tensor); the library never frees or reallocates it.  Pointers named *_host are host
 *    memory.  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *  - Calls taking a stream only enqueue work on it and never synchronise.  Calls taking
 *    host buffers synchronise before returning.
 *  - Every call returns 0 (DG_OK) or a negative error code; dg_last_error() gives the
 *    message of the calling thread's last failure.  There is NO CPU fallback: a shape the
 *    kernels do not support is DG_ERR_UNSUPPORTED.
 */
#ifndef DGVLASOV_H
#define DGVLASOV_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DG_OK                 0
#define DG_ERR_INVALID_ARG   -1
#define DG_ERR_UNSUPPORTED   -2
#define DG_ERR_CUDA          -3
#define DG_ERR_WORKSPACE     -4

#define DG_MAX_ORDER         10   /* LGL nodes per element per dimension: 2..10 */

typedef struct dg_ctx dg_ctx;

typedef struct {
  int32_t ndim;        /* 1 = x only (field solve), 2 = 1D1V (x,v), 3 = 1D2V (x,vx,vy) */
  int32_t nelem[3];    /* N_d, elements per dimension (unused dims: 0) */
  int32_t order[3];    /* n_d, LGL nodes per element per dimension, 2..DG_MAX_ORDER */
  double  lo[3];       /* lower bounds; x is [lo,hi) periodic */
  double  hi[3];       /* upper bounds */
  int32_t bc[3];       /* 0 periodic (the paper's roll), 1 zero-inflow
                          (exterior state 0); bc[0] must be 0 when the Poisson solve is used.
                          bc[0] = 2 (DG_BC_HALO): this context is an x-slab of a larger grid; the
                          exterior states at its two x faces come from dg_set_xhalo */
  double  omega_c;     /* = B_ext of Eq. 28; ignored for ndim < 3 */
  int32_t pmax;        /* Fourier modes kept, p = 0..pmax; 0 -> nelem[0] */
  int32_t mass_mode;   /* 0 = the paper's exact LGL mass matrix (Eq. 51/53/54);
                          1 = lumped (diagonal) LGL mass: Ups = (w_k/w_j) l_j'(xi_k), Xi = delta/w */
  int32_t device;      /* CUDA device ordinal */
} dg_grid_desc;

/* Host setup (Eq. 45, 53, 54, 63): LGL nodes/weights, Upsilon, Xi, quadrature
 * weights, node coordinates, the DG->Fourier tensor T (Eq. 63) and the synthesis matrix of
 * Eq. 71; uploads them.  *out owns that device memory until dg_destroy. */
int dg_create(const dg_grid_desc* desc, dg_ctx** out);
/* x-only context (field operations: dg_fourier_project, dg_poisson_E, dg_poisson_phi, dg_broken_l2, introspection) whose
 * elements have the explicitly given edges: Eq. 63 with its per-element (Delta x)_m.
 *   edges_host [in] [nelem+1], strictly ascending; x is periodic with L = edges[nelem] - edges[0]
 * Dense kernels only (the FFT factorisation needs equal widths: DG_OPT_FIELD_KERNEL = 4 fails with DG_ERR_UNSUPPORTED). */
int dg_create_field_nonuniform(const double* edges_host, int32_t nelem, int32_t order, int32_t pmax, int32_t device, dg_ctx** out);
int dg_destroy(dg_ctx* ctx);

/* Scratch for dg_ssprk3_* and dg_poisson_E: two stage arrays of the size of f, density
 * partials, rho, c_p, E.  The caller allocates `bytes >= dg_workspace_bytes(ctx)` of device
 * memory (256-byte aligned) and keeps it alive while the context uses it. */
size_t dg_workspace_bytes(const dg_ctx* ctx);
int dg_set_workspace(dg_ctx* ctx, void* ws_dev, size_t bytes);

/* Semi-discrete right-hand side, weak form Eq. 14 reduced by Eq. 20-21
 * with the upwind flux Eq. 23 and the speeds of Eq. 28
 * (PAPER.md:215):  dfdt = sum_d J_d ( a_d Ups_d f - Xi_d Flux_d ).
 *   f_dev    [in]  distribution, layout above
 *   E_dev    [in]  electric field at the x nodes, [N_x*n_x]; NULL means E = 0
 *   dfdt_dev [out] same shape as f; must not alias f_dev */
int dg_rhs(dg_ctx* ctx, const double* f_dev, const double* E_dev, double* dfdt_dev, void* stream);

/* x-slab decomposition (one slab of x-elements per GPU, velocity axes whole).  With bc[0] = DG_BC_HALO
 * the upwind flux of Eq. 23 at the slab's first / last x face takes its exterior
 * state from halo_dev instead of the paper's roll:
 *   halo_dev [in] [2][N_u*n_u][N_v*n_v] (ndim = 3) or [2][N_v*n_v] (ndim = 2):
 *            plane 0 = the left neighbour's LAST x-node plane, plane 1 = the right neighbour's FIRST.
 * The pointer is kept (caller-owned) and read by every later dg_rhs / dg_rk_stage call. */
#define DG_BC_HALO 2
int dg_set_xhalo(dg_ctx* ctx, const double* halo_dev);

/* Fused face-plane exchange for x-slab contexts.  After this call every dg_rk_stage also stores the first x-node plane of
 * out_dev into left_dst_dev and the last one into right_dst_dev, from inside the RHS kernel (a second TMA store of the
 * boundary tiles' rows).  The destinations are planes [G_u][G_v] of the x-NEIGHBOURS' halo buffers: left_dst_dev = plane 1
 * of the left neighbour's buffer (its exterior state right of its last node), right_dst_dev = plane 0 of the right
 * neighbour's -- device pointers into peer memory (NVLink P2P / symmetric memory) or into this device's own memory.
 * The caller double-buffers the halos (the stage that is running still reads the buffer set by dg_set_xhalo) and orders
 * the ranks (the all-gather of the density between two stages does).  NULL disables a side.  16-byte aligned. */
int dg_set_xhalo_push(dg_ctx* ctx, double* left_dst_dev, double* right_dst_dev);

/* One Runge-Kutta stage in Shu-Osher form: out = c0 f_n + c1 (f_s + dt L(f_s; E)).
 *   f_s_dev [in] stage input   f_n_dev [in] step input (NULL when c0 = 0)   E_dev [in] field or NULL
 *   out_dev [out] may alias f_n_dev (each node is read and written by one thread), not f_s_dev
 *   rho_out_dev [out, optional] density (Eq. 27) of out_dev at the own x nodes, [N_x*n_x]: finished from the per-tile
 *           partials of the kernel epilogue (tiled kernel; needs a workspace) instead of another pass over out_dev */
int dg_rk_stage(dg_ctx* ctx, const double* f_s_dev, const double* f_n_dev, const double* E_dev, double* out_dev,
                double c0, double c1, double dt, double* rho_out_dev, void* stream);

/* Shu-Osher SSP-RK3: u1 = u + dt L(u); u2 = 3/4 u + 1/4 (u1 + dt L(u1));
 * u+ = 1/3 u + 2/3 (u2 + dt L(u2)), in place on f_dev.  self_consistent = 1: E is solved from
 * each stage's input (density Eq. 27 -> c_p Eq. 63 -> E Eq. 71); 0: E = 0.  Needs a workspace.
 * dg_ssprk3_run does `nsteps` steps in one call and is what lets the density partials of a
 * stage's output, produced in that stage's epilogue, serve the next stage's field solve. */
int dg_ssprk3_step(dg_ctx* ctx, double* f_dev, double dt, int32_t self_consistent, void* stream);
int dg_ssprk3_run(dg_ctx* ctx, double* f_dev, double dt, int32_t nsteps, int32_t self_consistent, void* stream);
/* Same with a HOST array: copies f in, runs nsteps, copies f back, synchronises. */
int dg_ssprk3_run_host(dg_ctx* ctx, double* f_host, double dt, int32_t nsteps, int32_t self_consistent);
/* The Shu-Osher coefficients of stage `stage` = 0, 1, 2 (its ref. [38]): out = c0 u^n + c1 (u^(s) + dt L(u^(s))),
 * (c0, c1) = (0, 1), (3/4, 1/4), (1/3, 2/3).  For callers that drive dg_rk_stage themselves (the x-slab stepper): the table
 * lives in the library, not in the binding. */
int dg_ssprk3_stage_coeffs(int32_t stage, double* c0_host, double* c1_host);
/* Non-finite guard (the CFL blow-up case: PAPER.md:477 defers the order-dependent limits to its ref. [39]; see
 * dg_max_stable_dt): *flag_dev = 0 if every value of f is finite, 1 if any is Inf or NaN.  One pass over f, asynchronous
 * on `stream`; flag_dev is a device int32 owned by the caller.  x-only contexts check N_x*n_x values. */
int dg_check_finite(dg_ctx* ctx, const double* f_dev, int32_t* flag_dev, void* stream);

/* Zeroth moment Eq. 27 by LGL quadrature: rho[g_x] = sum_{g_u,g_v}
 * (w_{b_u}/J_u)(w_{b_v}/J_v) f.  rho_dev: [N_x*n_x].  Deterministic (no atomics). */
int dg_density(dg_ctx* ctx, const double* f_dev, double* rho_dev, void* stream);

/* c_p = T_p^{mj} rho_mj, Eq. 63, p = 0..pmax.
 *   rho_dev [in]  [batch][N_x*n_x]
 *   c_dev   [out] [batch][pmax+1][2]  (re, im) */
int dg_fourier_project(dg_ctx* ctx, const double* rho_dev, int32_t batch, double* c_dev, void* stream);

/* E from the density by Eq. 63 + Eq. 71: E_mj = sum_{0<|p|<=pmax}
 * -(c_p/(i k_p)) e^{i k_p x_mj}; the p = 0 mode (neutralising background of Eq. 27) is dropped.
 *   rho_dev [in] [batch][N_x*n_x]     E_dev [out] [batch][N_x*n_x]
 * batch > 1 needs workspace room for batch*(pmax+1)*2 doubles (see dg_field_workspace_bytes). */
int dg_poisson_E(dg_ctx* ctx, const double* rho_dev, int32_t batch, double* E_dev, void* stream);
/* Potential instead of field: Phi_mj = sum_{p != 0} -(c_p / k_p^2) e^{i k_p x_mj} (Eq. 70); same
 * arguments, layout and errors as dg_poisson_E.  E = -dPhi/dx. */
int dg_poisson_phi(dg_ctx* ctx, const double* rho_dev, int32_t batch, double* phi_dev, void* stream);
/* Broken l2 norm of Eq. 72 on the x grid: eps_b = (1/N_x) sum_m sqrt( int_m (u_b - v_b)^2 dx ), the integrand
 * being each element's nodal interpolant, integrated exactly with the LGL mass matrix of Eq. 50.
 *   u_dev, v_dev [in] [batch][N_x*n_x]; v_dev may be NULL (norm of u)     eps_dev [out] [batch] */
int dg_broken_l2(dg_ctx* ctx, const double* u_dev, const double* v_dev, int32_t batch, double* eps_dev, void* stream);
/* Domain-integrated electric field energy, the diagnostic of Fig. 10: W_b = (1/2) int E_b(x)^2 dx over the x
 * grid, the integrand being each element's nodal interpolant, integrated exactly with the LGL mass matrix of Eq. 50
 * -- not the lumped sum (1/2) sum w_j E_j^2, which is inexact at degree 2n-2.
 *   E_dev [in] [batch][N_x*n_x]     W_dev [out] [batch]      any context (ndim = 1, 2, 3); deterministic */
int dg_field_energy(dg_ctx* ctx, const double* E_dev, int32_t batch, double* W_dev, void* stream);
size_t dg_field_workspace_bytes(const dg_ctx* ctx, int32_t batch);

/* Introspection (host outputs; any pointer may be NULL to skip it). */
int dg_get_operators(const dg_ctx* ctx, int32_t dim, double* xi_host /*[n]*/, double* w_host /*[n]*/,
                     double* upsilon_host /*[n][n], row j = output node, reference element*/,
                     double* lift_host /*[n][2]: (L,R)*/);
int dg_get_dmatrix(const dg_ctx* ctx, int32_t dim, double* D_host /*[n][n]: D[j][k] = l_k'(xi_j), Eq. 55*/);
int dg_get_nodes(const dg_ctx* ctx, int32_t dim, double* coords_host /*[N_d*n_d]*/);
int dg_get_transform(const dg_ctx* ctx, int32_t p_first, int32_t p_count, double* T_host /*[p_count][N_x*n_x][2]*/);
/* Largest dt with sum_d |a_d| dt / Delta_d <= the SSP-RK3 limit of this order and mass mode
 * at |E| <= E_bound (PAPER.md:477 defers the CFL numbers to its ref. [39]). */
double dg_max_stable_dt(const dg_ctx* ctx, double E_bound);

/* Options and counters. */
#define DG_OPT_RHS_KERNEL   1   /* 0 auto (tiled when supported), 1 generic, 2 tiled (error if unsupported) */
#define DG_OPT_FIELD_KERNEL 2   /* 0 auto, 1 simple kernels (also inside dg_ssprk3_*: three launches per stage instead of the
                                  one-launch field solve), 2 tiled GEMM kernel (FP64 tensor cores, DMMA, when K is even and
                                  the operands are 16-byte aligned; else the DFMA kernel), 3 tiled DFMA GEMM kernel,
                                  4 FFT-factorised kernel (equal-width elements: N_x a power of two, even order; n FFTs of
                                  length N_x per vector in shared memory + a (pmax+1) x n mode table instead of the dense
                                  T and S; DG_ERR_UNSUPPORTED otherwise).  auto takes 4 for batched calls when supported. */
#define DG_OPT_PROFILE      3   /* k = 1: bracket every RHS-kernel launch with CUDA events on its stream (kernels run without
                                  programmatic launches: the kernel alone); k >= 2: bracket every k-th RHS launch only, inside a
                                  normally running sequence (k coprime to 3 visits every RK stage); 0: off */
#define DG_OPT_PDL          4   /* 1 (default): consecutive kernels of dg_ssprk3_* are chained by programmatic dependent
                                  launch (the next kernel's prologue overlaps the previous kernel's tail); 0: plain launches */
#define DG_OPT_FORM         5   /* 0 (default): weak form, Eq. 14: Upsilon F - Xi F*;  1: strong form, Eq. 15
                                  (PAPER.md:102): -D F + Xi (F - F*), D = Eq. 55.  Same scheme (Upsilon + D = Xi_R e_R^T -
                                  Xi_L e_L^T), different rounding; both RHS kernels, every entry point. */
int dg_set_option(dg_ctx* ctx, int32_t key, int64_t value);
/* Profile mode: total device time (ms) and count of the RHS-kernel launches since the last reset.
 * Synchronises on the recorded events. */
int dg_get_profile(dg_ctx* ctx, double* rhs_ms_total_host, int64_t* rhs_launches_host, int32_t reset);
/* The same per RK stage: index 0 = launches outside dg_ssprk3_* (dg_rhs, dg_rk_stage), 1..3 = stages 1..3.
 *   ms_host [out] [4]   launches_host [out] [4] */
int dg_get_profile_stages(dg_ctx* ctx, double* ms_host, int64_t* launches_host, int32_t reset);
int64_t dg_launch_count(const dg_ctx* ctx);      /* kernels launched through this context so far */
const char* dg_last_kernel(const dg_ctx* ctx);   /* name of the RHS kernel variant last used */
const char* dg_last_field_kernel(const dg_ctx* ctx);   /* name of the projection / field-solve kernel last used */
/* Measured FP64 arithmetic peak of `device` in TFLOP/s (2 flop per fused multiply-add): variant 0 = DFMA (vector pipe),
 * 1 = DMMA (mma.sync.m8n8k4.f64, the FP64 tensor path).  Register-resident chains, `iters` iterations (>= 1000 for a stable
 * figure), synchronises.  The roofline denominator of the dense DG->Fourier contraction (Eq. 63). */
int dg_fp64_peak(int32_t device, int32_t variant, int32_t iters, double* tflops_host);
const char* dg_last_error(void);
const char* dg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DGVLASOV_H */
