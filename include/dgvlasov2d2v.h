/* dgvlasov2d2v.h -- C ABI of the 2D2V (four-dimensional phase space) variant of the hot path.
 *
 * The paper states its method for any number of dimensions (Section 2, Eq. 18-21) and
 * runs it in 1D2V; this header is the same path with the second space dimension restored:
 *   phase space (x, y, u, v) = (x, y, v_x, v_y), ONE dense row-major FP64 array f[g_x][g_y][g_u][g_v]
 *   (the paper's u[a0,b0,a1,b1,a2,b2,a3,b3] in C order), g_d = a_d * n_d + b_d;
 *   speeds (Eq. 28, E = -grad Phi, B = omega_c z^):
 *       a_x = u,  a_y = v,  a_u = -E_x(x,y) - omega_c v,  a_v = -E_y(x,y) + omega_c u;
 *   density rho[g_x][g_y] (Eq. 27); field from the tensor product of the DG->Fourier transform of Eq. 63
 *    in x and y and the spectral Poisson solve of Eq. 68/71 with k^2 = k_p^2 + k_q^2.
 * Conventions (pointer naming, streams, error codes, no CPU fallback) are those of dgvlasov.h.
 */
#ifndef DGVLASOV2D2V_H
#define DGVLASOV2D2V_H

#include "dgvlasov.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dg4_ctx dg4_ctx;

typedef struct {
  int32_t nelem[4];    /* N_d, d = x, y, u, v */
  int32_t order[4];    /* LGL nodes per element per dimension, 2..DG_MAX_ORDER (tiled kernel: all four equal to 4) */
  double  lo[4];
  double  hi[4];
  int32_t bc[4];       /* 0 periodic, 1 zero-inflow; bc[0] may be DG_BC_HALO (an x-slab of a larger grid, dg4_set_xhalo);
                          bc[0], bc[1] must be 0 for the self-consistent dg4_ssprk3_run (the Poisson solve is global) */
  double  omega_c;     /* B_ext of Eq. 28 */
  int32_t pmax[2];     /* Fourier modes kept: |p| <= pmax[0] in x, |q| <= pmax[1] in y; 0 -> N_x, N_y */
  int32_t mass_mode;   /* 0 exact LGL mass (Eq. 51/53/54), 1 lumped */
  int32_t device;
} dg4_grid_desc;

int dg4_create(const dg4_grid_desc* desc, dg4_ctx** out);
int dg4_destroy(dg4_ctx* ctx);

/* Scratch for dg4_ssprk3_run and the field solve: two stage arrays, density partials, rho, E_x, E_y, mode buffers.
 * Caller-allocated device memory, 256-byte aligned, kept alive while the context uses it. */
size_t dg4_workspace_bytes(const dg4_ctx* ctx);
int dg4_set_workspace(dg4_ctx* ctx, void* ws_dev, size_t bytes);

/* Weak form Eq. 14 reduced by Eq. 20-21 with the upwind flux of Eq. 23 in four dimensions.
 *   f_dev [in] [G_x][G_y][G_u][G_v]   Ex_dev, Ey_dev [in] [G_x][G_y] or NULL (= 0)   dfdt_dev [out], must not alias f_dev */
int dg4_rhs(dg4_ctx* ctx, const double* f_dev, const double* Ex_dev, const double* Ey_dev, double* dfdt_dev, void* stream);

/* One Shu-Osher stage: out = c0 f_n + c1 (f_s + dt L(f_s; E)); f_n_dev NULL when c0 = 0; out_dev may alias
 * f_n_dev, not f_s_dev.  rho_out_dev [out, optional] [G_x][G_y]: density of out_dev, finished from the kernel's per-tile
 * partials (tiled kernel and a workspace) or by a density pass. */
int dg4_rk_stage(dg4_ctx* ctx, const double* f_s_dev, const double* f_n_dev, const double* Ex_dev, const double* Ey_dev,
                 double* out_dev, double c0, double c1, double dt, double* rho_out_dev, void* stream);

/* x-slab sharding (SURVEY.md 8(e) carried to 2D2V; the contract of dg_set_xhalo): a context created with bc[0] = DG_BC_HALO
 * is a slab of x-elements of a larger grid (y, u, v stay whole, so the density is local).  The upwind flux of Eq. 23
 * at the slab's first / last x face reads the left neighbour's LAST x-node plane / the right neighbour's
 * FIRST one from
 *   halo_dev [in] [2][G_y][G_u][G_v]: plane 0 = exterior state below the slab, plane 1 = above it (zeros for zero inflow);
 * device memory, 16-byte aligned, owned by the caller, read by every later dg4_rhs / dg4_rk_stage until replaced.
 * DG_ERR_INVALID_ARG if the context is not a halo context or the pointer is null or misaligned; dg4_rhs / dg4_rk_stage on a
 * halo context without a halo buffer fail the same way. */
int dg4_set_xhalo(dg4_ctx* ctx, const double* halo_dev);

/* rho[g_x][g_y] = sum_{g_u,g_v} (w_{b_u}/J_u)(w_{b_v}/J_v) f  (Eq. 27).  Deterministic.  Needs a workspace. */
int dg4_density(dg4_ctx* ctx, const double* f_dev, double* rho_dev, void* stream);

/* c_pq = sum T^x_p[g_x] T^y_q[g_y] rho[g_x][g_y] (Eq. 63 in x and in y).
 *   c_dev [out] [pmax_x+1][2 pmax_y+1][2] (re, im): p = 0..pmax_x, second index q + pmax_y for q = -pmax_y..pmax_y
 *   (c_{-p,-q} = conj c_pq for the real density).  Needs a workspace. */
int dg4_fourier_project(dg4_ctx* ctx, const double* rho_dev, double* c_dev, void* stream);

/* (E_x, E_y)[g_x][g_y] = sum_{(p,q) != (0,0)} i (k_p, k_q) c_pq / (k_p^2 + k_q^2) e^{i (k_p x + k_q y)}
 * (Phi_pq = -c_pq/k^2, Eq. 68; E = -grad Phi, Eq. 71).  Needs a workspace. */
int dg4_poisson_E(dg4_ctx* ctx, const double* rho_dev, double* Ex_dev, double* Ey_dev, void* stream);

/* nsteps SSP-RK3 steps in place; self_consistent = 1: the field is solved from each stage's input. */
int dg4_ssprk3_run(dg4_ctx* ctx, double* f_dev, double dt, int32_t nsteps, int32_t self_consistent, void* stream);
/* The same with a HOST array (copy in, run, copy back, synchronise). */
int dg4_ssprk3_run_host(dg4_ctx* ctx, double* f_host, double dt, int32_t nsteps, int32_t self_consistent);

int dg4_get_nodes(const dg4_ctx* ctx, int32_t dim, double* coords_host /*[N_d*n_d]*/);
/* Largest dt with sum_d |a_d| dt / Delta_d within the SSP-RK3 limit of this order and mass mode at |E_x|, |E_y| <= E_bound
 * (as dg_max_stable_dt). */
double dg4_max_stable_dt(const dg4_ctx* ctx, double E_bound);
#define DG4_OPT_RHS_KERNEL 1   /* 0 auto (tiled when all orders are 4 and N_v is even; TMA line kernel for order 8 in all
                                  dimensions; element kernel for equal orders 6; else generic), 1 generic, 2 tiled, 3 element
                                  kernel (equal orders 4, 6, 8), 4 line kernel (order 8); 2, 3 and 4 fail with
                                  DG_ERR_UNSUPPORTED on other shapes */
#define DG4_OPT_PROFILE    3   /* k >= 1: bracket every k-th RHS-kernel launch with CUDA events on its stream (0 off) */
int dg4_set_option(dg4_ctx* ctx, int32_t key, int64_t value);
int dg4_get_profile(dg4_ctx* ctx, double* rhs_ms_total_host, int64_t* rhs_launches_host, int32_t reset);
int64_t dg4_launch_count(const dg4_ctx* ctx);
const char* dg4_last_kernel(const dg4_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* DGVLASOV2D2V_H */
