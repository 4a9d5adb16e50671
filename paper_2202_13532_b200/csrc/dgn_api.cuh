// C-ABI entry points of the dimension-generic variant (include/dgvlasov_nd.h).  Included at the end of dg_api.cu (one
// translation unit: it reuses fail / CUDA_TRY / align_up / DeviceGuard, the host setup of dg_setup.cpp and the SSP-RK3 loop of
// dg_stepper.hpp).
#pragma once
#include "../../include/dgvlasov_nd.h"
#include "dgn_kernels.cuh"

struct dgn_ctx {
  dgn_grid_desc desc;
  int ndim = 0, dx = 0, dv = 0;
  int N[6], n[6], G[6];
  double J[6];
  size_t dof = 0;
  long long GX = 1, GV = 1;
  int P[3] = {0, 0, 0};            // modes kept per space dimension
  int M[3] = {1, 1, 1};            // mode-lattice extents: M_0 = P_0 + 1 (p_0 >= 0), M_i = 2 P_i + 1 (i > 0), 1 beyond dx
  double k1[3] = {0, 0, 0};        // 2 pi / L_i
  dgsetup::Basis1D basis[6];
  std::vector<double> coord_h[6];
  void* dev_block = nullptr;
  double *d_ups[6], *d_lift[6], *d_coord[6], *d_wq[6];
  double2 *d_T[3] = {nullptr, nullptr, nullptr};   // [M_i][G_i]: rows of Eq. 63 (negative modes by conjugation)
  double2 *d_W[3] = {nullptr, nullptr, nullptr};   // [G_i][M_i]: e^{i k_p x_g} of Eq. 71
  // workspace
  void* ws = nullptr;
  double *u1 = nullptr, *u2 = nullptr, *rho = nullptr, *E = nullptr;
  double2 *bufA = nullptr, *bufB = nullptr, *Et = nullptr;
  size_t buf_elems = 0;
  int64_t launches = 0;
};

static int checkn(dgn_ctx* ctx, const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
  ctx->launches += 1;
  return DG_OK;
}

static unsigned gridn(long long work) {
  long long b = (work + 255) / 256;
  if (b > 148LL * 32) b = 148LL * 32;
  return (unsigned)(b < 1 ? 1 : b);
}

extern "C" int dgn_create(const dgn_grid_desc* desc, dgn_ctx** out) {
  if (!desc || !out) return fail(DG_ERR_INVALID_ARG, "dgn_create: null argument");
  *out = nullptr;
  if (desc->dx < 1 || desc->dx > 3 || desc->dv < desc->dx || desc->dv > 3)
    return fail(DG_ERR_UNSUPPORTED, "dgn_create: need 1 <= dx <= dv <= 3");
  const int nd = desc->dx + desc->dv;
  for (int d = 0; d < nd; ++d) {
    if (desc->nelem[d] < 1) return fail(DG_ERR_INVALID_ARG, "dgn_create: nelem must be >= 1");
    if (desc->order[d] < 2 || desc->order[d] > DG_MAX_ORDER) return fail(DG_ERR_UNSUPPORTED, "dgn_create: order must be 2..10");
    if (!(desc->hi[d] > desc->lo[d])) return fail(DG_ERR_INVALID_ARG, "dgn_create: hi must exceed lo");
    if (desc->bc[d] != 0 && desc->bc[d] != 1) return fail(DG_ERR_INVALID_ARG, "dgn_create: bc must be 0 or 1");
  }
  if (desc->mass_mode != 0 && desc->mass_mode != 1) return fail(DG_ERR_INVALID_ARG, "dgn_create: mass_mode must be 0 or 1");
  for (int i = 0; i < desc->dx; ++i) if (desc->pmax[i] < 0) return fail(DG_ERR_INVALID_ARG, "dgn_create: pmax must be >= 0");
  if (int rc = check_device(desc->device, "dgn_create")) return rc;
  DeviceGuard guard(desc->device);
  dgn_ctx* ctx = new (std::nothrow) dgn_ctx();
  if (!ctx) return fail(DG_ERR_CUDA, "dgn_create: out of host memory");
  ctx->desc = *desc;
  ctx->ndim = nd; ctx->dx = desc->dx; ctx->dv = desc->dv;
  ctx->dof = 1;
  for (int d = 0; d < nd; ++d) {
    ctx->N[d] = desc->nelem[d]; ctx->n[d] = desc->order[d]; ctx->G[d] = ctx->N[d] * ctx->n[d];
    ctx->J[d] = 2.0 * ctx->N[d] / (desc->hi[d] - desc->lo[d]);
    ctx->dof *= (size_t)ctx->G[d];
    if (d < ctx->dx) ctx->GX *= ctx->G[d]; else ctx->GV *= ctx->G[d];
  }
  const long double two_pi = 6.283185307179586476925286766559L;
  std::vector<double> Tm[3], Wm[3], wq[6];
  try {
    for (int d = 0; d < nd; ++d) ctx->basis[d] = dgsetup::make_basis(ctx->n[d], desc->mass_mode);
    for (int d = 0; d < nd; ++d) {
      const int n = ctx->n[d];
      ctx->coord_h[d].resize(ctx->G[d]);
      wq[d].resize(ctx->G[d]);
      const long double dxl = ((long double)desc->hi[d] - (long double)desc->lo[d]) / ctx->N[d];
      for (int m = 0; m < ctx->N[d]; ++m)
        for (int j = 0; j < n; ++j) {
          ctx->coord_h[d][m * n + j] = (double)((long double)desc->lo[d] + (m + 0.5L) * dxl + 0.5L * dxl * ctx->basis[d].xi_ld[j]);
          wq[d][m * n + j] = (double)(ctx->basis[d].w_ld[j] * dxl * 0.5L);
        }
    }
    for (int i = 0; i < ctx->dx; ++i) {
      const int P = desc->pmax[i] > 0 ? desc->pmax[i] : desc->nelem[i];
      ctx->P[i] = P;
      ctx->M[i] = i == 0 ? P + 1 : 2 * P + 1;
      const long double L = (long double)desc->hi[i] - (long double)desc->lo[i];
      ctx->k1[i] = (double)(two_pi / L);
      std::vector<double> T, S, x;
      dgsetup::make_fourier(ctx->basis[i], ctx->N[i], desc->lo[i], desc->hi[i], P, T, S, x);
      ctx->coord_h[i] = x;
      const int G = ctx->G[i], Mi = ctx->M[i];
      Tm[i].resize((size_t)Mi * G * 2);
      Wm[i].resize((size_t)G * Mi * 2);
      for (int m = 0; m < Mi; ++m) {
        const int p = i == 0 ? m : m - P, pa = p < 0 ? -p : p;
        for (int g = 0; g < G; ++g) {
          Tm[i][((size_t)m * G + g) * 2] = T[(size_t)(2 * pa) * G + g];
          Tm[i][((size_t)m * G + g) * 2 + 1] = (p < 0 ? -1.0 : 1.0) * T[(size_t)(2 * pa + 1) * G + g];      // T_{-p} = conj T_p
          const long double ph = two_pi * p / L * (long double)x[g];
          Wm[i][((size_t)g * Mi + m) * 2] = (double)cosl(ph);
          Wm[i][((size_t)g * Mi + m) * 2 + 1] = (double)sinl(ph);
        }
      }
    }
  } catch (const std::exception& e) {
    delete ctx;
    return fail(DG_ERR_INVALID_ARG, std::string("dgn_create: setup failed: ") + e.what());
  }
  size_t off = 0;
  size_t o_ups[6], o_lift[6], o_coord[6], o_wq[6], o_T[3], o_W[3];
  for (int d = 0; d < nd; ++d) {
    o_ups[d] = off;   off = align_up(off + sizeof(double) * ctx->n[d] * ctx->n[d], 256);
    o_lift[d] = off;  off = align_up(off + sizeof(double) * ctx->n[d] * 2, 256);
    o_coord[d] = off; off = align_up(off + sizeof(double) * ctx->G[d], 256);
    o_wq[d] = off;    off = align_up(off + sizeof(double) * ctx->G[d], 256);
  }
  for (int i = 0; i < ctx->dx; ++i) {
    o_T[i] = off; off = align_up(off + sizeof(double) * Tm[i].size(), 256);
    o_W[i] = off; off = align_up(off + sizeof(double) * Wm[i].size(), 256);
  }
  cudaError_t e = cudaMalloc(&ctx->dev_block, off);
  if (e != cudaSuccess) { delete ctx; return fail(DG_ERR_CUDA, std::string("dgn_create: cudaMalloc: ") + cudaGetErrorString(e)); }
  char* base = (char*)ctx->dev_block;
  bool ok = true;
  auto up = [&](double*& dst, size_t o, const std::vector<double>& src) {
    dst = (double*)(base + o);
    ok = ok && cudaMemcpy(dst, src.data(), sizeof(double) * src.size(), cudaMemcpyHostToDevice) == cudaSuccess;
  };
  for (int d = 0; d < nd; ++d) {
    up(ctx->d_ups[d], o_ups[d], ctx->basis[d].ups);
    up(ctx->d_lift[d], o_lift[d], ctx->basis[d].lift);
    up(ctx->d_coord[d], o_coord[d], ctx->coord_h[d]);
    up(ctx->d_wq[d], o_wq[d], wq[d]);
  }
  for (int i = 0; i < ctx->dx; ++i) {
    double* t; up(t, o_T[i], Tm[i]); ctx->d_T[i] = reinterpret_cast<double2*>(t);
    double* w; up(w, o_W[i], Wm[i]); ctx->d_W[i] = reinterpret_cast<double2*>(w);
  }
  if (!ok) { cudaFree(ctx->dev_block); delete ctx; return fail(DG_ERR_CUDA, "dgn_create: upload failed"); }
  // largest intermediate of the field solve: every axis either still holds nodes or already modes
  ctx->buf_elems = 1;
  for (int i = 0; i < ctx->dx; ++i) ctx->buf_elems *= (size_t)(ctx->M[i] > ctx->G[i] ? ctx->M[i] : ctx->G[i]);
  *out = ctx;
  return DG_OK;
}

extern "C" int dgn_destroy(dgn_ctx* ctx) {
  if (!ctx) return DG_OK;
  DeviceGuard guard(ctx->desc.device);
  if (ctx->dev_block) cudaFree(ctx->dev_block);
  delete ctx;
  return DG_OK;
}

extern "C" size_t dgn_workspace_bytes(const dgn_ctx* ctx) {
  if (!ctx) return 0;
  const size_t modes = (size_t)ctx->M[0] * ctx->M[1] * ctx->M[2];
  size_t b = 2 * align_up(ctx->dof * sizeof(double), 256);
  b += align_up((size_t)ctx->GX * sizeof(double), 256);                         // rho
  b += align_up((size_t)ctx->dx * ctx->GX * sizeof(double), 256);               // E
  b += 2 * align_up(ctx->buf_elems * 2 * sizeof(double), 256);                  // bufA, bufB
  b += align_up((size_t)ctx->dx * modes * 2 * sizeof(double), 256);             // Et
  return b;
}

extern "C" int dgn_set_workspace(dgn_ctx* ctx, void* ws_dev, size_t bytes) {
  if (!ctx) return fail(DG_ERR_INVALID_ARG, "dgn_set_workspace: null context");
  if (!ws_dev || ((uintptr_t)ws_dev & 255) != 0) return fail(DG_ERR_INVALID_ARG, "dgn_set_workspace: pointer must be non-null and 256-byte aligned");
  if (bytes < dgn_workspace_bytes(ctx)) return fail(DG_ERR_WORKSPACE, "dgn_set_workspace: too small, see dgn_workspace_bytes");
  const size_t modes = (size_t)ctx->M[0] * ctx->M[1] * ctx->M[2];
  char* p = (char*)ws_dev;
  auto carve = [&](size_t doubles) { double* d = (double*)p; p += align_up(doubles * sizeof(double), 256); return d; };
  ctx->ws = ws_dev;
  ctx->u1 = carve(ctx->dof); ctx->u2 = carve(ctx->dof);
  ctx->rho = carve((size_t)ctx->GX);
  ctx->E = carve((size_t)ctx->dx * ctx->GX);
  ctx->bufA = reinterpret_cast<double2*>(carve(ctx->buf_elems * 2));
  ctx->bufB = reinterpret_cast<double2*>(carve(ctx->buf_elems * 2));
  ctx->Et = reinterpret_cast<double2*>(carve((size_t)ctx->dx * modes * 2));
  return DG_OK;
}

// ------------------------------------------------------------------------------------------------
// launches
// ------------------------------------------------------------------------------------------------
static int launch_rhsn(dgn_ctx* ctx, const double* f, const double* fn, const double* E, double* out, int mode,
                       double c0, double c1, double dt, cudaStream_t st) {
  dgn::Params p;
  memset(&p, 0, sizeof(p));
  p.ndim = ctx->ndim; p.dx = ctx->dx; p.dv = ctx->dv;
  for (int d = 0; d < ctx->ndim; ++d) {
    p.N[d] = ctx->N[d]; p.n[d] = ctx->n[d]; p.G[d] = ctx->G[d]; p.bc[d] = ctx->desc.bc[d]; p.J[d] = ctx->J[d];
    p.coord[d] = ctx->d_coord[d]; p.ups[d] = ctx->d_ups[d]; p.lift[d] = ctx->d_lift[d];
  }
  p.omega_c = ctx->desc.omega_c;
  p.E = E; p.GX = ctx->GX; p.GV = ctx->GV;
  p.f = f; p.fn = fn; p.out = out; p.c0 = c0; p.c1 = c1; p.dt = dt; p.mode = mode;
  p.dof = (long long)ctx->dof;
  dgn::rhs_nd_kernel<<<gridn((long long)ctx->dof), 256, 0, st>>>(p);
  return checkn(ctx, "rhs_nd_kernel");
}

static int launch_densityn(dgn_ctx* ctx, const double* f, double* rho, cudaStream_t st) {
  const int dx = ctx->dx, dv = ctx->dv;
  const unsigned grid = (unsigned)(ctx->GX < 148LL * 32 ? ctx->GX : 148LL * 32);
  dgn::density_nd_kernel<<<grid, 256, 0, st>>>(f, ctx->d_wq[dx], dv >= 2 ? ctx->d_wq[dx + 1] : nullptr, dv >= 3 ? ctx->d_wq[dx + 2] : nullptr,
                                               dv, ctx->G[dx], dv >= 2 ? ctx->G[dx + 1] : 1, dv >= 3 ? ctx->G[dx + 2] : 1,
                                               ctx->GX, ctx->GV, rho);
  return checkn(ctx, "density_nd_kernel");
}

// rho -> E: Eq. 63 along every space axis, the Poisson factors of Eq. 68 / 71, Eq. 71 back along every axis.
static int launch_fieldn(dgn_ctx* ctx, const double* rho, double* E, cudaStream_t st) {
  const int dx = ctx->dx;
  const int* M = ctx->M;
  const int* G = ctx->G;
  // forward: axis i turns [m_0..m_{i-1}][G_i][G_{i+1}..] into [m_0..m_i][G_{i+1}..]
  const void* src = rho;
  double2* bufs[2] = {ctx->bufA, ctx->bufB};
  int which = 0;
  for (int i = 0; i < dx; ++i) {
    long long pre = 1, post = 1;
    for (int j = 0; j < i; ++j) pre *= M[j];
    for (int j = i + 1; j < dx; ++j) post *= G[j];
    dgn::apply_axis_kernel<<<gridn(pre * M[i] * post), 256, 0, st>>>(ctx->d_T[i], src, i == 0 ? 1 : 0, bufs[which], pre, M[i], G[i], post);
    int rc = checkn(ctx, "apply_axis_kernel");
    if (rc) return rc;
    src = bufs[which];
    which ^= 1;
  }
  const long long modes = (long long)M[0] * M[1] * M[2];
  dgn::poisson_nd_kernel<<<gridn(modes), 256, 0, st>>>(reinterpret_cast<const double2*>(src), dx, M[0], M[1], M[2], ctx->P[1], ctx->P[2],
                                                       ctx->k1[0], ctx->k1[1], ctx->k1[2], ctx->Et);
  int rc = checkn(ctx, "poisson_nd_kernel");
  if (rc) return rc;
  // backward, per component: axes dx-1 .. 1 by apply_axis (modes -> nodes), axis 0 by the real synthesis
  for (int comp = 0; comp < dx; ++comp) {
    const double2* cur = ctx->Et + (long long)comp * modes;
    int w = 0;
    for (int i = dx - 1; i >= 1; --i) {
      long long pre = 1, post = 1;
      for (int j = 0; j < i; ++j) pre *= M[j];
      for (int j = i + 1; j < dx; ++j) post *= G[j];
      dgn::apply_axis_kernel<<<gridn(pre * G[i] * post), 256, 0, st>>>(ctx->d_W[i], cur, 0, bufs[w], pre, G[i], M[i], post);
      rc = checkn(ctx, "apply_axis_kernel");
      if (rc) return rc;
      cur = bufs[w];
      w ^= 1;
    }
    long long post = 1;
    for (int j = 1; j < dx; ++j) post *= G[j];
    dgn::synth0_kernel<<<gridn((long long)G[0] * post), 256, 0, st>>>(ctx->d_W[0], cur, G[0], M[0], post, E + (long long)comp * ctx->GX);
    rc = checkn(ctx, "synth0_kernel");
    if (rc) return rc;
  }
  return DG_OK;
}

// ------------------------------------------------------------------------------------------------
// entry points
// ------------------------------------------------------------------------------------------------
extern "C" int dgn_rhs(dgn_ctx* ctx, const double* f_dev, const double* E_dev, double* dfdt_dev, void* stream) {
  if (!ctx || !f_dev || !dfdt_dev) return fail(DG_ERR_INVALID_ARG, "dgn_rhs: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (f_dev == dfdt_dev) return fail(DG_ERR_INVALID_ARG, "dgn_rhs: dfdt must not alias f");
  return launch_rhsn(ctx, f_dev, nullptr, E_dev, dfdt_dev, 0, 0.0, 1.0, 0.0, (cudaStream_t)stream);
}

extern "C" int dgn_rk_stage(dgn_ctx* ctx, const double* f_s_dev, const double* f_n_dev, const double* E_dev, double* out_dev,
                            double c0, double c1, double dt, void* stream) {
  if (!ctx || !f_s_dev || !out_dev) return fail(DG_ERR_INVALID_ARG, "dgn_rk_stage: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (f_s_dev == out_dev) return fail(DG_ERR_INVALID_ARG, "dgn_rk_stage: out must not alias f_s");
  if (c0 != 0.0 && !f_n_dev) return fail(DG_ERR_INVALID_ARG, "dgn_rk_stage: c0 != 0 needs f_n");
  return launch_rhsn(ctx, f_s_dev, c0 != 0.0 ? f_n_dev : nullptr, E_dev, out_dev, 1, c0, c1, dt, (cudaStream_t)stream);
}

extern "C" int dgn_density(dgn_ctx* ctx, const double* f_dev, double* rho_dev, void* stream) {
  if (!ctx || !f_dev || !rho_dev) return fail(DG_ERR_INVALID_ARG, "dgn_density: null argument");
  DeviceGuard guard(ctx->desc.device);
  return launch_densityn(ctx, f_dev, rho_dev, (cudaStream_t)stream);
}

extern "C" int dgn_poisson_E(dgn_ctx* ctx, const double* rho_dev, double* E_dev, void* stream) {
  if (!ctx || !rho_dev || !E_dev) return fail(DG_ERR_INVALID_ARG, "dgn_poisson_E: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (!ctx->ws) return fail(DG_ERR_WORKSPACE, "dgn_poisson_E: set a workspace first");
  return launch_fieldn(ctx, rho_dev, E_dev, (cudaStream_t)stream);
}

extern "C" int dgn_ssprk3_run(dgn_ctx* ctx, double* f_dev, double dt, int32_t nsteps, int32_t self_consistent, void* stream) {
  if (!ctx || !f_dev) return fail(DG_ERR_INVALID_ARG, "dgn_ssprk3_run: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (nsteps < 0 || !(dt == dt)) return fail(DG_ERR_INVALID_ARG, "dgn_ssprk3_run: bad nsteps or dt");
  if (!ctx->ws) return fail(DG_ERR_WORKSPACE, "dgn_ssprk3_run: set a workspace first");
  if (self_consistent)
    for (int i = 0; i < ctx->dx; ++i)
      if (ctx->desc.bc[i] != 0) return fail(DG_ERR_INVALID_ARG, "dgn_ssprk3_run: the self-consistent field needs periodic space dimensions");
  cudaStream_t st = (cudaStream_t)stream;
  const bool sc = self_consistent != 0;
  return ssprk3_run_loop(
      f_dev, ctx->u1, ctx->u2, nsteps, sc,
      [&](const double* src) {
        int rc = launch_densityn(ctx, src, ctx->rho, st);
        return rc ? rc : launch_fieldn(ctx, ctx->rho, ctx->E, st);
      },
      [&](int, const double* src, const double* fn, double* dst, double c0, double c1) {
        return launch_rhsn(ctx, src, fn, sc ? ctx->E : nullptr, dst, 1, c0, c1, dt, st);
      });
}

extern "C" int dgn_get_nodes(const dgn_ctx* ctx, int32_t dim, double* coords) {
  if (!ctx || dim < 0 || dim >= ctx->ndim || !coords) return fail(DG_ERR_INVALID_ARG, "dgn_get_nodes: bad argument");
  memcpy(coords, ctx->coord_h[dim].data(), sizeof(double) * ctx->G[dim]);
  return DG_OK;
}

extern "C" int64_t dgn_launch_count(const dgn_ctx* ctx) { return ctx ? ctx->launches : 0; }
