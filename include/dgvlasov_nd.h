/* dgvlasov_nd.h -- C ABI of the dimension-generic variant of the hot path ("general d").
 *
 * The paper states its method for any number of dimensions (Section 2, Eq. 18-21; PAPER.md:43:
 * "computing the semi-discrete equation in n-dimensions").  This header is the same path for a phase space
 *   (x_1..x_dx, v_1..v_dv),  1 <= dx <= dv <= 3   (1D1V, 1D2V, 1D3V, 2D2V, 2D3V, 3D3V),
 * ONE dense row-major FP64 array f[g_x1]..[g_xdx][g_v1]..[g_vdv] (the paper's u[a0,b0,...] in C order),
 * g_d = a_d * n_d + b_d.  Speeds (Eq. 28, all space dimensions restored; E = -grad Phi, B = omega_c z^):
 *   a_{x_i} = v_i (i < dx);  a_{v_1} = -E_1 - omega_c v_2;  a_{v_2} = -E_2 + omega_c v_1;  a_{v_3} = -E_3
 *   (E_i = 0 for i >= dx; no magnetic term when dv = 1).
 * Density rho[x] over all velocity dimensions (Eq. 27); field from the tensor product of the DG->Fourier
 * transform of Eq. 63 over the space dimensions and the spectral Poisson solve of Eq. 68/71 (PAPER.md:447,
 * 459) with k^2 = sum_i k_{p_i}^2.  One kernel family for every (dx, dv): one thread per node, lines read from global
 * memory -- the tiled / TMA kernels of dgvlasov.h (1D2V) and dgvlasov2d2v.h (2D2V) are the fast paths of their shapes; this
 * one is the general path and their cross-check.
 * Conventions (pointer naming, streams, error codes, no CPU fallback) are those of dgvlasov.h.
 */
#ifndef DGVLASOV_ND_H
#define DGVLASOV_ND_H

#include "dgvlasov.h"

#ifdef __cplusplus
extern "C" {
#endif

#define DGN_MAX_DIM 6

typedef struct dgn_ctx dgn_ctx;

typedef struct {
  int32_t dx, dv;              /* space and velocity dimensions, 1 <= dx <= dv <= 3 */
  int32_t nelem[DGN_MAX_DIM];  /* N_d, dimensions ordered (x_1..x_dx, v_1..v_dv); entries beyond dx + dv ignored */
  int32_t order[DGN_MAX_DIM];  /* LGL nodes per element per dimension, 2..DG_MAX_ORDER */
  double  lo[DGN_MAX_DIM];
  double  hi[DGN_MAX_DIM];
  int32_t bc[DGN_MAX_DIM];     /* 0 periodic, 1 zero-inflow; the space dimensions must be periodic for the Poisson solve */
  double  omega_c;             /* B_ext of Eq. 28 */
  int32_t pmax[3];             /* Fourier modes kept per space dimension, |p_i| <= pmax[i]; 0 -> N_i */
  int32_t mass_mode;           /* 0 exact LGL mass (Eq. 51/53/54), 1 lumped */
  int32_t device;
} dgn_grid_desc;

int dgn_create(const dgn_grid_desc* desc, dgn_ctx** out);
int dgn_destroy(dgn_ctx* ctx);

/* Scratch for dgn_ssprk3_run and the field solve: two stage arrays, rho, dx field components, mode buffers.
 * Caller-allocated device memory, 256-byte aligned, kept alive while the context uses it. */
size_t dgn_workspace_bytes(const dgn_ctx* ctx);
int dgn_set_workspace(dgn_ctx* ctx, void* ws_dev, size_t bytes);

/* Weak form Eq. 14 reduced by Eq. 20-21 with the upwind flux of Eq. 23 in dx + dv dimensions.
 *   f_dev [in]  the phase-space array      E_dev [in] [dx][G_x1]..[G_xdx] (component i at offset i * prod G_x) or NULL (= 0)
 *   dfdt_dev [out], must not alias f_dev */
int dgn_rhs(dgn_ctx* ctx, const double* f_dev, const double* E_dev, double* dfdt_dev, void* stream);

/* One Shu-Osher stage: out = c0 f_n + c1 (f_s + dt L(f_s; E)); f_n_dev NULL when c0 = 0; out_dev may alias
 * f_n_dev, not f_s_dev. */
int dgn_rk_stage(dgn_ctx* ctx, const double* f_s_dev, const double* f_n_dev, const double* E_dev, double* out_dev,
                 double c0, double c1, double dt, void* stream);

/* rho[x] = sum over all velocity nodes of prod_i (w_b/J_{v_i}) f  (Eq. 27).  Deterministic (fixed-order sums). */
int dgn_density(dgn_ctx* ctx, const double* f_dev, double* rho_dev, void* stream);

/* E_i[x] = sum_{p != 0} i k_{p_i} c_p / |k_p|^2 e^{i k_p . x}, c_p the tensor-product projection of rho (Eq. 63, 68, 71).
 *   rho_dev [in] [G_x1]..[G_xdx]    E_dev [out] [dx][G_x1]..[G_xdx].  Needs a workspace. */
int dgn_poisson_E(dgn_ctx* ctx, const double* rho_dev, double* E_dev, void* stream);

/* nsteps SSP-RK3 steps in place; self_consistent = 1: the field is solved from each stage's input. */
int dgn_ssprk3_run(dgn_ctx* ctx, double* f_dev, double dt, int32_t nsteps, int32_t self_consistent, void* stream);

int dgn_get_nodes(const dgn_ctx* ctx, int32_t dim, double* coords_host /*[N_d*n_d]*/);
int64_t dgn_launch_count(const dgn_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* DGVLASOV_ND_H */
