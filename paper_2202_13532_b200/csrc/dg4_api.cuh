// C-ABI entry points of the 2D2V variant (include/dgvlasov2d2v.h).  Included at the end of dg_api.cu (one translation
// unit: it reuses fail / CUDA_TRY / align_up and the density kernels of dg_kernels_generic.cuh).
#pragma once
#include "../../include/dgvlasov2d2v.h"
#include "dg4_kernels.cuh"
#include "dg4_kernels_tiled.cuh"
#include "dg4_kernels_elem.cuh"
#include "dg4_kernels_line.cuh"

struct dg4_ctx {
  dg4_grid_desc desc;
  int N[4], n[4], G[4];
  double J[4];
  size_t dof = 0;
  int P1 = 1, Q = 0;               // modes p = 0..P1-1 in x, q = -Q..Q in y
  double kx1 = 0, ky1 = 0;         // 2 pi / L_x, 2 pi / L_y
  dgsetup::Basis1D basis[4];
  std::vector<double> coord_h[4];
  void* dev_block = nullptr;
  double *d_ups[4], *d_lift[4], *d_coord[4], *d_wq[4];
  double *d_Tx = nullptr, *d_Ty = nullptr, *d_Wx = nullptr, *d_Wy = nullptr;
  // workspace
  void* ws = nullptr;
  double *u1 = nullptr, *u2 = nullptr, *partials = nullptr, *rho = nullptr, *Ex = nullptr, *Ey = nullptr;
  double *A = nullptr, *c = nullptr, *Et = nullptr, *B = nullptr;
  size_t partials_doubles = 0;
  double* f_stage = nullptr;
  int64_t launches = 0;
  int opt_kernel = 0, opt_profile = 0;   // opt_profile = k: every k-th RHS launch is bracketed by events
  int64_t prof_seen = 0;
  std::vector<cudaEvent_t> prof_events;
  double prof_ms = 0.0;
  int64_t prof_launches = 0;
  std::string last_kernel = "none";
  std::map<TmapKey, CUtensorMap> tmaps;   // TMA descriptors of the arrays seen so far (line kernel)
  const double* xhalo = nullptr;          // caller-owned exterior x-face planes (bc[0] = DG_BC_HALO)
};

static int check4(dg4_ctx* ctx, const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
  ctx->launches += 1;
  return DG_OK;
}

static int elem_order(const dg4_ctx* ctx) {     // order of the element kernel, 0 = unsupported
  const int n = ctx->n[0];
  for (int d = 1; d < 4; ++d) if (ctx->n[d] != n) return 0;
  if (ctx->N[1] > 65535 || ctx->N[0] > 65535) return 0;
  return (n == 4 || n == 6 || n == 8) ? n : 0;
}

static int tile_kv(const dg4_ctx* ctx) {       // v-elements per tile of the tiled kernel, 0 = unsupported
  for (int d = 0; d < 4; ++d) if (ctx->n[d] != 4) return 0;
  if (ctx->N[3] % 8 == 0) return 8;
  if (ctx->N[3] % 4 == 0) return 4;
  if (ctx->N[3] % 2 == 0) return 2;
  return 0;
}

extern "C" int dg4_create(const dg4_grid_desc* desc, dg4_ctx** out) {
  if (!desc || !out) return fail(DG_ERR_INVALID_ARG, "dg4_create: null argument");
  *out = nullptr;
  for (int d = 0; d < 4; ++d) {
    if (desc->nelem[d] < 1) return fail(DG_ERR_INVALID_ARG, "dg4_create: nelem must be >= 1");
    if (desc->order[d] < 2 || desc->order[d] > DG_MAX_ORDER) return fail(DG_ERR_UNSUPPORTED, "dg4_create: order must be 2..10");
    if (!(desc->hi[d] > desc->lo[d])) return fail(DG_ERR_INVALID_ARG, "dg4_create: hi must exceed lo");
    if (desc->bc[d] != 0 && desc->bc[d] != 1 && !(d == 0 && desc->bc[d] == DG_BC_HALO))
      return fail(DG_ERR_INVALID_ARG, "dg4_create: bc must be 0 or 1 (bc[0] may be DG_BC_HALO)");
  }
  if (desc->mass_mode != 0 && desc->mass_mode != 1) return fail(DG_ERR_INVALID_ARG, "dg4_create: mass_mode must be 0 or 1");
  if (desc->pmax[0] < 0 || desc->pmax[1] < 0) return fail(DG_ERR_INVALID_ARG, "dg4_create: pmax must be >= 0");
  if (int rc = check_device(desc->device, "dg4_create")) return rc;
  DeviceGuard guard(desc->device);      // the caller's current device is restored on return
  dg4_ctx* ctx = new (std::nothrow) dg4_ctx();
  if (!ctx) return fail(DG_ERR_CUDA, "dg4_create: out of host memory");
  ctx->desc = *desc;
  ctx->dof = 1;
  for (int d = 0; d < 4; ++d) {
    ctx->N[d] = desc->nelem[d]; ctx->n[d] = desc->order[d]; ctx->G[d] = ctx->N[d] * ctx->n[d];
    ctx->J[d] = 2.0 * ctx->N[d] / (desc->hi[d] - desc->lo[d]);
    ctx->dof *= (size_t)ctx->G[d];
  }
  const int px = desc->pmax[0] > 0 ? desc->pmax[0] : desc->nelem[0];
  ctx->Q = desc->pmax[1] > 0 ? desc->pmax[1] : desc->nelem[1];
  ctx->P1 = px + 1;
  const long double two_pi = 6.283185307179586476925286766559L;
  ctx->kx1 = (double)(two_pi / ((long double)desc->hi[0] - (long double)desc->lo[0]));
  ctx->ky1 = (double)(two_pi / ((long double)desc->hi[1] - (long double)desc->lo[1]));

  std::vector<double> Tx, Ty, S, x, y, wq[4], Wx, Wy;
  try {
    for (int d = 0; d < 4; ++d) ctx->basis[d] = dgsetup::make_basis(ctx->n[d], desc->mass_mode);
    dgsetup::make_fourier(ctx->basis[0], ctx->N[0], desc->lo[0], desc->hi[0], px, Tx, S, x);
    dgsetup::make_fourier(ctx->basis[1], ctx->N[1], desc->lo[1], desc->hi[1], ctx->Q, Ty, S, y);
  } catch (const std::exception& e) {
    delete ctx;
    return fail(DG_ERR_INVALID_ARG, std::string("dg4_create: setup failed: ") + e.what());
  }
  for (int d = 0; d < 4; ++d) {
    const int n = ctx->n[d];
    ctx->coord_h[d].resize(ctx->G[d]);
    wq[d].resize(ctx->G[d]);
    const long double dx = ((long double)desc->hi[d] - (long double)desc->lo[d]) / ctx->N[d];
    for (int m = 0; m < ctx->N[d]; ++m)
      for (int j = 0; j < n; ++j) {
        ctx->coord_h[d][m * n + j] = (double)((long double)desc->lo[d] + (m + 0.5L) * dx + 0.5L * dx * ctx->basis[d].xi_ld[j]);
        wq[d][m * n + j] = (double)(ctx->basis[d].w_ld[j] * dx * 0.5L);
      }
  }
  ctx->coord_h[0] = x;
  ctx->coord_h[1] = y;
  // synthesis waves e^{i k_p x_g} of Eq. 71 at the node coordinates
  auto waves = [&](int dim, int count, std::vector<double>& W) {
    const int G = ctx->G[dim];
    const long double L = (long double)desc->hi[dim] - (long double)desc->lo[dim];
    W.resize((size_t)count * G * 2);
    for (int p = 0; p < count; ++p)
      for (int g = 0; g < G; ++g) {
        const long double ph = two_pi * p / L * (long double)ctx->coord_h[dim][g];
        W[((size_t)p * G + g) * 2] = (double)cosl(ph);
        W[((size_t)p * G + g) * 2 + 1] = (double)sinl(ph);
      }
  };
  waves(0, ctx->P1, Wx);
  waves(1, ctx->Q + 1, Wy);

  size_t off = 0;
  size_t o_ups[4], o_lift[4], o_coord[4], o_wq[4];
  for (int d = 0; d < 4; ++d) {
    o_ups[d] = off;   off = align_up(off + sizeof(double) * ctx->n[d] * ctx->n[d], 256);
    o_lift[d] = off;  off = align_up(off + sizeof(double) * ctx->n[d] * 2, 256);
    o_coord[d] = off; off = align_up(off + sizeof(double) * ctx->G[d], 256);
    o_wq[d] = off;    off = align_up(off + sizeof(double) * ctx->G[d], 256);
  }
  const size_t o_Tx = off; off = align_up(off + sizeof(double) * Tx.size(), 256);
  const size_t o_Ty = off; off = align_up(off + sizeof(double) * Ty.size(), 256);
  const size_t o_Wx = off; off = align_up(off + sizeof(double) * Wx.size(), 256);
  const size_t o_Wy = off; off = align_up(off + sizeof(double) * Wy.size(), 256);
  cudaError_t e = cudaMalloc(&ctx->dev_block, off);
  if (e != cudaSuccess) { delete ctx; return fail(DG_ERR_CUDA, std::string("dg4_create: cudaMalloc: ") + cudaGetErrorString(e)); }
  char* base = (char*)ctx->dev_block;
  bool ok = true;
  auto up = [&](double*& dst, size_t o, const std::vector<double>& src) {
    dst = (double*)(base + o);
    ok = ok && cudaMemcpy(dst, src.data(), sizeof(double) * src.size(), cudaMemcpyHostToDevice) == cudaSuccess;
  };
  for (int d = 0; d < 4; ++d) {
    up(ctx->d_ups[d], o_ups[d], ctx->basis[d].ups);
    up(ctx->d_lift[d], o_lift[d], ctx->basis[d].lift);
    up(ctx->d_coord[d], o_coord[d], ctx->coord_h[d]);
    up(ctx->d_wq[d], o_wq[d], wq[d]);
  }
  up(ctx->d_Tx, o_Tx, Tx); up(ctx->d_Ty, o_Ty, Ty); up(ctx->d_Wx, o_Wx, Wx); up(ctx->d_Wy, o_Wy, Wy);
  if (!ok) { cudaFree(ctx->dev_block); delete ctx; return fail(DG_ERR_CUDA, "dg4_create: upload failed"); }
  *out = ctx;
  return DG_OK;
}

extern "C" int dg4_destroy(dg4_ctx* ctx) {
  if (!ctx) return DG_OK;
  DeviceGuard guard(ctx->desc.device);
  if (ctx->dev_block) cudaFree(ctx->dev_block);
  if (ctx->f_stage) cudaFree(ctx->f_stage);
  for (cudaEvent_t e : ctx->prof_events) cudaEventDestroy(e);
  delete ctx;
  return DG_OK;
}

static size_t partials4_doubles(const dg4_ctx* ctx) {
  size_t per = 64;                                           // density_partial kernels: chunks per (g_x, g_y)
  const int kv = tile_kv(ctx);
  if (kv && (size_t)ctx->N[2] * (ctx->N[3] / kv) > per) per = (size_t)ctx->N[2] * (ctx->N[3] / kv);
  if (elem_order(ctx) && (size_t)ctx->N[2] * ctx->N[3] > per) per = (size_t)ctx->N[2] * ctx->N[3];
  return (size_t)ctx->G[0] * ctx->G[1] * per;
}

extern "C" size_t dg4_workspace_bytes(const dg4_ctx* ctx) {
  if (!ctx) return 0;
  const size_t gxy = (size_t)ctx->G[0] * ctx->G[1], nq = 2 * (size_t)ctx->Q + 1;
  size_t b = 2 * align_up(ctx->dof * sizeof(double), 256);
  b += align_up(partials4_doubles(ctx) * sizeof(double), 256);
  b += 3 * align_up(gxy * sizeof(double), 256);                                   // rho, Ex, Ey
  b += align_up((size_t)ctx->P1 * ctx->G[1] * 2 * sizeof(double), 256);           // A
  b += align_up((size_t)ctx->P1 * nq * 2 * sizeof(double), 256);                  // c
  b += align_up((size_t)2 * ctx->P1 * nq * 2 * sizeof(double), 256);              // Et
  b += align_up((size_t)2 * ctx->P1 * ctx->G[1] * 2 * sizeof(double), 256);       // B
  return b;
}

extern "C" int dg4_set_workspace(dg4_ctx* ctx, void* ws_dev, size_t bytes) {
  if (!ctx) return fail(DG_ERR_INVALID_ARG, "dg4_set_workspace: null context");
  DeviceGuard guard(ctx->desc.device);
  if (!ws_dev || ((uintptr_t)ws_dev & 255) != 0) return fail(DG_ERR_INVALID_ARG, "dg4_set_workspace: pointer must be non-null and 256-byte aligned");
  if (bytes < dg4_workspace_bytes(ctx)) return fail(DG_ERR_WORKSPACE, "dg4_set_workspace: too small, see dg4_workspace_bytes");
  const size_t gxy = (size_t)ctx->G[0] * ctx->G[1], nq = 2 * (size_t)ctx->Q + 1;
  char* p = (char*)ws_dev;
  auto carve = [&](double*& dst, size_t doubles) { dst = (double*)p; p += align_up(doubles * sizeof(double), 256); };
  ctx->ws = ws_dev;
  carve(ctx->u1, ctx->dof); carve(ctx->u2, ctx->dof);
  ctx->partials_doubles = partials4_doubles(ctx);
  carve(ctx->partials, ctx->partials_doubles);
  carve(ctx->rho, gxy); carve(ctx->Ex, gxy); carve(ctx->Ey, gxy);
  carve(ctx->A, (size_t)ctx->P1 * ctx->G[1] * 2);
  carve(ctx->c, (size_t)ctx->P1 * nq * 2);
  carve(ctx->Et, (size_t)2 * ctx->P1 * nq * 2);
  carve(ctx->B, (size_t)2 * ctx->P1 * ctx->G[1] * 2);
  return DG_OK;
}

// ------------------------------------------------------------------------------------------------
// launches
// ------------------------------------------------------------------------------------------------
// 4-D TMA descriptor of an array f[G0][G1][G2][G3] with box (b0 = v, b1 = u, b2 = y, b3 = x); cached per (base, box).
static bool make_map4(CUtensorMap* m, const void* base, dg4_ctx* ctx, int b0, int b1, int b2, int b3, bool swz64, int outer = 0) {
  const TmapKey key{base, b0, b1, b2 * 16 + b3, swz64 ? 2 : 0, 4 + 16 * outer};
  auto it = ctx->tmaps.find(key);
  if (it != ctx->tmaps.end()) { *m = it->second; return true; }
  dgt::EncodeTiledFn enc = dgt::encode_fn();
  if (!enc) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)ctx->G[3], (cuuint64_t)ctx->G[2], (cuuint64_t)ctx->G[1], (cuuint64_t)(outer > 0 ? outer : ctx->G[0])};
  const cuuint64_t strides[3] = {(cuuint64_t)ctx->G[3] * 8, (cuuint64_t)ctx->G[3] * ctx->G[2] * 8,
                                 (cuuint64_t)ctx->G[3] * ctx->G[2] * ctx->G[1] * 8};
  const cuuint32_t box[4] = {(cuuint32_t)b0, (cuuint32_t)b1, (cuuint32_t)b2, (cuuint32_t)b3};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, swz64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  if (ctx->tmaps.size() >= 512) ctx->tmaps.clear();
  ctx->tmaps[key] = *m;
  return true;
}

// n = 8 in all four dimensions, G_v*8 a multiple of 16 bytes (always), arrays 16-byte aligned: the TMA line kernel
static bool line_supported(const dg4_ctx* ctx) {
  for (int d = 0; d < 4; ++d) if (ctx->n[d] != 8) return false;
  return true;
}

static int launch_rhs4_line(dg4_ctx* ctx, const double* f, const double* fn, const double* Ex, const double* Ey, double* out,
                            int mode, double c0, double c1, double dt, bool want_partials, int* chunks_out, cudaStream_t st) {
  dg4l::LineParams P;
  memset(&P, 0, sizeof(P));
  const bool with_fn = mode != 0 && fn != nullptr;
  bool ok = make_map4(&P.m_main, f, ctx, 8, 8, 8, 8, true) && make_map4(&P.m_out, out, ctx, 8, 8, 8, 8, true) &&
            make_map4(&P.m_xface, f, ctx, 8, 8, 8, 1, false) && make_map4(&P.m_yface, f, ctx, 8, 8, 1, 8, false) &&
            make_map4(&P.m_uface, f, ctx, 8, 1, 8, 8, false) && make_map4(&P.m_vface, f, ctx, 2, 8, 8, 8, false);
  if (ok && with_fn) ok = make_map4(&P.m_fn, fn, ctx, 8, 8, 8, 8, true);
  else P.m_fn = P.m_main;
  if (ok && ctx->desc.bc[0] == DG_BC_HALO) ok = make_map4(&P.m_xhalo, ctx->xhalo, ctx, 8, 8, 8, 1, false, 2);
  else P.m_xhalo = P.m_xface;
  if (!ok) return fail(DG_ERR_CUDA, "dg4: cuTensorMapEncodeTiled failed");
  const dgsetup::Basis1D& b = ctx->basis[0];
  for (int j = 0; j < 4; ++j) {
    for (int k = 0; k < 4; ++k) {
      P.pe[j * 4 + k] = 0.5 * (b.ups[j * 8 + k] + b.ups[j * 8 + 7 - k]);
      P.qo[j * 4 + k] = 0.5 * (b.ups[j * 8 + k] - b.ups[j * 8 + 7 - k]);
    }
    P.la[j] = 0.5 * (b.lift[2 * j] - b.lift[2 * j + 1]);
    P.lb[j] = 0.5 * (b.lift[2 * j] + b.lift[2 * j + 1]);
  }
  for (int j = 0; j < 8; ++j) P.wref[j] = b.w[j];
  P.cu = ctx->d_coord[2]; P.cv = ctx->d_coord[3]; P.Ex = Ex; P.Ey = Ey;
  P.Jx = ctx->J[0]; P.Jy = ctx->J[1]; P.Ju = ctx->J[2]; P.Jv = ctx->J[3]; P.omega_c = ctx->desc.omega_c;
  P.wscale = 1.0 / (ctx->J[2] * ctx->J[3]);
  P.c0 = c0; P.c1 = c1; P.dt = dt; P.mode = mode; P.strong = 0;
  for (int d = 0; d < 4; ++d) { P.N[d] = ctx->N[d]; P.G[d] = ctx->G[d]; P.bc[d] = ctx->desc.bc[d]; }
  P.chunks = ctx->N[2] * ctx->N[3];
  if (want_partials && mode != 0 && ctx->partials && (size_t)ctx->G[0] * ctx->G[1] * P.chunks <= ctx->partials_doubles) {
    P.partials = ctx->partials; P.want_partials = 1;
    if (chunks_out) *chunks_out = P.chunks;
  }
  // x-elements per rasterisation group (as the n = 4 tiled kernel): a power of two <= 8 dividing N_x, grown while the tiles
  // between a tile and its y neighbour (three 32 KB tiles each) stay within ~32 MB, a quarter of the L2
  int bxl = 0;
  while (bxl < 3 && ctx->N[0] % (2 << bxl) == 0 && (double)ctx->N[2] * ctx->N[3] * (2 << bxl) * 3.0 * 32768.0 <= 32e6) ++bxl;
  P.bx_log2 = bxl;
  const long long tiles = (long long)ctx->N[0] * ctx->N[1] * ctx->N[2] * ctx->N[3];
  if (tiles > 0x7fffffffLL) return fail(DG_ERR_UNSUPPORTED, "dg4: too many tiles");
  if (with_fn) {
    CUDA_TRY(ensure_dyn_smem(reinterpret_cast<const void*>(dg4l::rhs4_line_kernel<true>), dg4l::SMEM_BYTES));
    dg4l::rhs4_line_kernel<true><<<(unsigned)tiles, dg4l::NT, dg4l::SMEM_BYTES, st>>>(P);
  } else {
    CUDA_TRY(ensure_dyn_smem(reinterpret_cast<const void*>(dg4l::rhs4_line_kernel<false>), dg4l::SMEM_BYTES));
    dg4l::rhs4_line_kernel<false><<<(unsigned)tiles, dg4l::NT, dg4l::SMEM_BYTES, st>>>(P);
  }
  ctx->last_kernel = "rhs4_line<8>";
  return check4(ctx, "rhs4_line_kernel");
}

static int launch_rhs4_inner(dg4_ctx* ctx, const double* f, const double* fn, const double* Ex, const double* Ey, double* out,
                             int mode, double c0, double c1, double dt, bool want_partials, int* chunks_out, cudaStream_t st) {
  if (chunks_out) *chunks_out = 0;
  if (ctx->desc.bc[0] == DG_BC_HALO && !ctx->xhalo) return fail(DG_ERR_INVALID_ARG, "dg4: bc[0] = DG_BC_HALO needs dg4_set_xhalo first");
  dg4::Params p;
  memset(&p, 0, sizeof(p));
  p.xhalo = ctx->xhalo;
  for (int d = 0; d < 4; ++d) {
    p.N[d] = ctx->N[d]; p.n[d] = ctx->n[d]; p.G[d] = ctx->G[d]; p.bc[d] = ctx->desc.bc[d]; p.J[d] = ctx->J[d];
    p.coord[d] = ctx->d_coord[d]; p.ups[d] = ctx->d_ups[d]; p.lift[d] = ctx->d_lift[d];
  }
  p.omega_c = ctx->desc.omega_c;
  p.Ex = Ex; p.Ey = Ey; p.f = f; p.fn = fn; p.out = out; p.c0 = c0; p.c1 = c1; p.dt = dt; p.mode = mode;
  p.dof = (long long)ctx->dof;
  const int kv = tile_kv(ctx);
  const bool aligned = (((uintptr_t)f | (uintptr_t)out | (uintptr_t)fn) & 15) == 0;
  if (ctx->opt_kernel == 2 && !(kv && aligned))
    return fail(DG_ERR_UNSUPPORTED, "dg4: the tiled kernel needs order 4 in all dimensions, an even N_v and 16-byte aligned arrays");
  if (kv && aligned && (ctx->opt_kernel == 0 || ctx->opt_kernel == 2)) {
    for (int i = 0; i < 16; ++i) p.U[i] = ctx->basis[0].ups[i];
    for (int i = 0; i < 8; ++i) p.Xi[i] = ctx->basis[0].lift[i];
    p.wqu = ctx->d_wq[2]; p.wqv = ctx->d_wq[3];
    const int nvb = ctx->N[3] / kv;
    p.chunks = ctx->N[2] * nvb;
    if (want_partials && mode != 0 && ctx->partials && (size_t)ctx->G[0] * ctx->G[1] * p.chunks <= ctx->partials_doubles) {
      p.partials = ctx->partials;
      if (chunks_out) *chunks_out = p.chunks;
    }
    if (ctx->N[1] > 65535 || ctx->N[0] > 65535) return fail(DG_ERR_UNSUPPORTED, "dg4: more than 65535 elements in x or y");
    // x-elements per rasterisation group: a power of two (<= 8) dividing N_x, grown while the tiles between a tile and its
    // y neighbour (read + read + written bytes) stay within ~32 MB, a quarter of the L2
    int bxl = 0;
    {
      const double tile_bytes = 3.0 * 64 * 4 * kv * 8;
      while (bxl < 3 && ctx->N[0] % (2 << bxl) == 0 && (double)ctx->N[2] * nvb * (2 << bxl) * tile_bytes <= 32e6) ++bxl;
    }
    p.bx_log2 = bxl;
    p.wide_st = (((uintptr_t)out & 31) == 0) ? 1 : 0;      // rows are G_v = 4 N_v doubles: every element row starts on 32 bytes
    const dim3 tiles(nvb * (1 << bxl) * ctx->N[2], ctx->N[1], ctx->N[0] >> bxl);
    const bool with_fn = mode != 0 && fn != nullptr;
    const size_t smem = sizeof(double) * (kv == 8 ? dg4::tile_smem_doubles<8>(with_fn) : kv == 4 ? dg4::tile_smem_doubles<4>(with_fn)
                                                                                              : dg4::tile_smem_doubles<2>(with_fn));
    if (kv == 8) CUDA_TRY(ensure_dyn_smem(reinterpret_cast<const void*>(dg4::rhs4_tile_kernel<8, 5>), sizeof(double) * dg4::tile_smem_doubles<8>(true)));
    if (kv == 8) dg4::rhs4_tile_kernel<8, 5><<<tiles, 128, smem, st>>>(p);
    else if (kv == 4) dg4::rhs4_tile_kernel<4, 1><<<tiles, 64, smem, st>>>(p);
    else dg4::rhs4_tile_kernel<2, 1><<<tiles, 32, smem, st>>>(p);
    ctx->last_kernel = kv == 8 ? "rhs4_tile<8>" : (kv == 4 ? "rhs4_tile<4>" : "rhs4_tile<2>");
    return check4(ctx, "rhs4_tile_kernel");
  }
  if (ctx->opt_kernel == 4 && !(line_supported(ctx) && aligned))
    return fail(DG_ERR_UNSUPPORTED, "dg4: the line kernel needs order 8 in all dimensions and 16-byte aligned arrays");
  if (line_supported(ctx) && aligned && (ctx->opt_kernel == 0 || ctx->opt_kernel == 4))
    return launch_rhs4_line(ctx, f, fn, Ex, Ey, out, mode, c0, c1, dt, want_partials, chunks_out, st);
  const int ne = elem_order(ctx);
  if (ctx->opt_kernel == 3 && !(ne && aligned))
    return fail(DG_ERR_UNSUPPORTED, "dg4: the element kernel needs equal orders 4, 6 or 8 and 16-byte aligned arrays");
  if (ne && aligned && (ctx->opt_kernel == 3 || (ctx->opt_kernel == 0 && ne != 4))) {
    for (int i = 0; i < ne * ne; ++i) p.Un[i] = ctx->basis[0].ups[i];
    for (int i = 0; i < 2 * ne; ++i) p.Xin[i] = ctx->basis[0].lift[i];
    p.wqu = ctx->d_wq[2]; p.wqv = ctx->d_wq[3];
    p.chunks = ctx->N[2] * ctx->N[3];
    if (want_partials && mode != 0 && ctx->partials && (size_t)ctx->G[0] * ctx->G[1] * p.chunks <= ctx->partials_doubles) {
      p.partials = ctx->partials;
      if (chunks_out) *chunks_out = p.chunks;
    }
    const dim3 grid(ctx->N[3] * ctx->N[2], ctx->N[1], ctx->N[0]);
    if (ne == 8) {
      const size_t smem = sizeof(double) * dg4::elem_smem_doubles<8>();
      CUDA_TRY(ensure_dyn_smem(reinterpret_cast<const void*>(dg4::rhs4_elem_kernel<8>), smem));
      dg4::rhs4_elem_kernel<8><<<grid, 512, smem, st>>>(p);
    } else if (ne == 6) dg4::rhs4_elem_kernel<6><<<grid, 216, sizeof(double) * dg4::elem_smem_doubles<6>(), st>>>(p);
    else dg4::rhs4_elem_kernel<4><<<grid, 64, sizeof(double) * dg4::elem_smem_doubles<4>(), st>>>(p);
    ctx->last_kernel = ne == 8 ? "rhs4_elem<8>" : (ne == 6 ? "rhs4_elem<6>" : "rhs4_elem<4>");
    return check4(ctx, "rhs4_elem_kernel");
  }
  long long blocks = ((long long)ctx->dof + 255) / 256;
  if (blocks > 148LL * 64) blocks = 148LL * 64;
  dg4::rhs4_generic_kernel<<<(unsigned)blocks, 256, 0, st>>>(p);
  ctx->last_kernel = "rhs4_generic";
  return check4(ctx, "rhs4_generic_kernel");
}

static int launch_rhs4(dg4_ctx* ctx, const double* f, const double* fn, const double* Ex, const double* Ey, double* out,
                       int mode, double c0, double c1, double dt, bool want_partials, int* chunks_out, cudaStream_t st) {
  if (!(ctx->opt_profile > 0 && (ctx->prof_seen++ % ctx->opt_profile) == 0)) return launch_rhs4_inner(ctx, f, fn, Ex, Ey, out, mode, c0, c1, dt, want_partials, chunks_out, st);
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  CUDA_TRY(cudaEventRecord(e0, st));
  int rc = launch_rhs4_inner(ctx, f, fn, Ex, Ey, out, mode, c0, c1, dt, want_partials, chunks_out, st);
  CUDA_TRY(cudaEventRecord(e1, st));
  ctx->prof_events.push_back(e0);
  ctx->prof_events.push_back(e1);
  return rc;
}

// Density partials of f over the (u, v) plane of every (g_x, g_y): the 1D2V density kernels with (g_x, g_y) flattened.
static int launch_density4_partials(dg4_ctx* ctx, const double* f, int* nchunks_out, cudaStream_t st) {
  const int GXY = ctx->G[0] * ctx->G[1], G2 = ctx->G[2], G3 = ctx->G[3];
  if (!ctx->partials) return fail(DG_ERR_WORKSPACE, "dg4: set a workspace first");
  const size_t plane = (size_t)G2 * G3;
  int nchunks, rows;
  if (G3 % 2 == 0 && ((uintptr_t)f & 15) == 0) {
    int CP = 1;
    while (CP < G3 / 2 && CP < 256) CP *= 2;
    const int RL = 256 / CP;
    rows = 32 * RL;
    while (rows > 8 * RL && (long long)((G2 + rows - 1) / rows) * GXY < 148LL * 16) rows /= 2;
    nchunks = (G2 + rows - 1) / rows;
    if ((size_t)nchunks * GXY <= ctx->partials_doubles) {
      for (int g0 = 0; g0 < GXY; g0 += 65535) {            // grid.y is limited to 65535 (g_x, g_y) pairs per launch
        dim3 grid(nchunks, GXY - g0 < 65535 ? GXY - g0 : 65535);
        dgk::density_partial_vec_kernel<8><<<grid, 256, 0, st>>>(f + g0 * plane, ctx->d_wq[2], ctx->d_wq[3], G2, G3, rows, CP,
                                                                 ctx->partials + (size_t)g0 * nchunks);
        int rc = check4(ctx, "density_partial_vec_kernel");
        if (rc) return rc;
      }
      *nchunks_out = nchunks;
      return DG_OK;
    }
  }
  rows = G2; nchunks = 1;
  for (int g0 = 0; g0 < GXY; g0 += 65535) {
    dim3 grid(nchunks, GXY - g0 < 65535 ? GXY - g0 : 65535);
    dgk::density_partial_kernel<<<grid, 256, 0, st>>>(f + g0 * plane, ctx->d_wq[2], ctx->d_wq[3], G2, G3, rows, ctx->partials + g0);
    int rc = check4(ctx, "density_partial_kernel");
    if (rc) return rc;
  }
  *nchunks_out = nchunks;
  return DG_OK;
}

static int launch_density4_finish(dg4_ctx* ctx, int nchunks, double* rho, cudaStream_t st) {
  const int GXY = ctx->G[0] * ctx->G[1];
  dgk::density_finish_kernel<<<(GXY + 3) / 4, 128, 0, st>>>(ctx->partials, nchunks, GXY, rho);
  return check4(ctx, "density_finish_kernel");
}

static int launch_project4(dg4_ctx* ctx, const double* rho, double* c, double* Et, cudaStream_t st) {
  const int G0 = ctx->G[0], G1 = ctx->G[1], NQ = 2 * ctx->Q + 1;
  dg4::proj_x_kernel<<<dim3((G1 + 31) / 32, ctx->P1), 256, 0, st>>>(ctx->d_Tx, rho, G0, G1, ctx->A);
  int rc = check4(ctx, "proj_x_kernel");
  if (rc) return rc;
  dg4::proj_y_poisson_kernel<<<(ctx->P1 * NQ + 3) / 4, 128, 0, st>>>(ctx->d_Ty, ctx->A, G1, ctx->P1, ctx->Q, ctx->kx1, ctx->ky1, c, Et);
  return check4(ctx, "proj_y_poisson_kernel");
}

static int launch_field4(dg4_ctx* ctx, const double* rho, double* Ex, double* Ey, cudaStream_t st) {
  const int G0 = ctx->G[0], G1 = ctx->G[1];
  int rc = launch_project4(ctx, rho, nullptr, ctx->Et, st);
  if (rc) return rc;
  dg4::synth_y_kernel<<<dim3((G1 + 31) / 32, ctx->P1, 2), 256, 0, st>>>(ctx->Et, ctx->d_Wy, G1, ctx->P1, ctx->Q, ctx->B);
  rc = check4(ctx, "synth_y_kernel");
  if (rc) return rc;
  if (G0 > 65535) return fail(DG_ERR_UNSUPPORTED, "dg4: G_x above 65535");
  dg4::synth_x_kernel<<<dim3((G1 + 31) / 32, G0, 2), 128, 0, st>>>(ctx->B, ctx->d_Wx, G0, G1, ctx->P1, Ex, Ey);
  return check4(ctx, "synth_x_kernel");
}

// ------------------------------------------------------------------------------------------------
// entry points
// ------------------------------------------------------------------------------------------------
extern "C" int dg4_rhs(dg4_ctx* ctx, const double* f_dev, const double* Ex_dev, const double* Ey_dev, double* dfdt_dev, void* stream) {
  if (!ctx || !f_dev || !dfdt_dev) return fail(DG_ERR_INVALID_ARG, "dg4_rhs: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (f_dev == dfdt_dev) return fail(DG_ERR_INVALID_ARG, "dg4_rhs: dfdt must not alias f");
  return launch_rhs4(ctx, f_dev, nullptr, Ex_dev, Ey_dev, dfdt_dev, 0, 0.0, 1.0, 0.0, false, nullptr, (cudaStream_t)stream);
}

extern "C" int dg4_density(dg4_ctx* ctx, const double* f_dev, double* rho_dev, void* stream) {
  if (!ctx || !f_dev || !rho_dev) return fail(DG_ERR_INVALID_ARG, "dg4_density: null argument");
  DeviceGuard guard(ctx->desc.device);
  int nchunks = 0;
  int rc = launch_density4_partials(ctx, f_dev, &nchunks, (cudaStream_t)stream);
  if (rc) return rc;
  return launch_density4_finish(ctx, nchunks, rho_dev, (cudaStream_t)stream);
}

extern "C" int dg4_rk_stage(dg4_ctx* ctx, const double* f_s_dev, const double* f_n_dev, const double* Ex_dev, const double* Ey_dev,
                            double* out_dev, double c0, double c1, double dt, double* rho_out_dev, void* stream) {
  if (!ctx || !f_s_dev || !out_dev) return fail(DG_ERR_INVALID_ARG, "dg4_rk_stage: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (f_s_dev == out_dev) return fail(DG_ERR_INVALID_ARG, "dg4_rk_stage: out must not alias f_s");
  if (c0 != 0.0 && !f_n_dev) return fail(DG_ERR_INVALID_ARG, "dg4_rk_stage: c0 != 0 needs f_n");
  cudaStream_t st = (cudaStream_t)stream;
  int chunks = 0;
  int rc = launch_rhs4(ctx, f_s_dev, c0 != 0.0 ? f_n_dev : nullptr, Ex_dev, Ey_dev, out_dev, 1, c0, c1, dt, rho_out_dev != nullptr, &chunks, st);
  if (rc || !rho_out_dev) return rc;
  if (chunks > 0) return launch_density4_finish(ctx, chunks, rho_out_dev, st);
  return dg4_density(ctx, out_dev, rho_out_dev, stream);
}

extern "C" int dg4_set_xhalo(dg4_ctx* ctx, const double* halo_dev) {
  if (!ctx) return fail(DG_ERR_INVALID_ARG, "dg4_set_xhalo: null context");
  if (ctx->desc.bc[0] != DG_BC_HALO) return fail(DG_ERR_INVALID_ARG, "dg4_set_xhalo: the context was not created with bc[0] = DG_BC_HALO");
  if (!halo_dev || ((uintptr_t)halo_dev & 15) != 0) return fail(DG_ERR_INVALID_ARG, "dg4_set_xhalo: pointer must be non-null and 16-byte aligned");
  ctx->xhalo = halo_dev;
  return DG_OK;
}

extern "C" int dg4_fourier_project(dg4_ctx* ctx, const double* rho_dev, double* c_dev, void* stream) {
  if (!ctx || !rho_dev || !c_dev) return fail(DG_ERR_INVALID_ARG, "dg4_fourier_project: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (!ctx->ws) return fail(DG_ERR_WORKSPACE, "dg4_fourier_project: set a workspace first");
  return launch_project4(ctx, rho_dev, c_dev, nullptr, (cudaStream_t)stream);
}

extern "C" int dg4_poisson_E(dg4_ctx* ctx, const double* rho_dev, double* Ex_dev, double* Ey_dev, void* stream) {
  if (!ctx || !rho_dev || !Ex_dev || !Ey_dev) return fail(DG_ERR_INVALID_ARG, "dg4_poisson_E: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (!ctx->ws) return fail(DG_ERR_WORKSPACE, "dg4_poisson_E: set a workspace first");
  return launch_field4(ctx, rho_dev, Ex_dev, Ey_dev, (cudaStream_t)stream);
}

static int field4_from_partials_or_f(dg4_ctx* ctx, const double* f, int chunks, cudaStream_t st) {
  int rc;
  if (chunks <= 0) { rc = launch_density4_partials(ctx, f, &chunks, st); if (rc) return rc; }
  rc = launch_density4_finish(ctx, chunks, ctx->rho, st);
  if (rc) return rc;
  return launch_field4(ctx, ctx->rho, ctx->Ex, ctx->Ey, st);
}

extern "C" int dg4_ssprk3_run(dg4_ctx* ctx, double* f_dev, double dt, int32_t nsteps, int32_t self_consistent, void* stream) {
  if (!ctx || !f_dev) return fail(DG_ERR_INVALID_ARG, "dg4_ssprk3_run: null argument");
  DeviceGuard guard(ctx->desc.device);
  if (nsteps < 0 || !(dt == dt)) return fail(DG_ERR_INVALID_ARG, "dg4_ssprk3_run: bad nsteps or dt");
  if (!ctx->ws) return fail(DG_ERR_WORKSPACE, "dg4_ssprk3_run: set a workspace first");
  // An x-slab context reads its exterior x faces from the planes of dg4_set_xhalo, which belong to ONE stage input: a whole
  // step in one call would feed stages 2 and 3 the faces of the step input.  Slabs step stage by stage (dg4_rk_stage).
  if (ctx->desc.bc[0] == DG_BC_HALO)
    return fail(DG_ERR_INVALID_ARG, "dg4_ssprk3_run: an x-slab context (bc[0] = DG_BC_HALO) steps stage by stage through dg4_rk_stage");
  if (self_consistent && (ctx->desc.bc[0] != 0 || ctx->desc.bc[1] != 0))
    return fail(DG_ERR_INVALID_ARG, "dg4_ssprk3_run: the self-consistent field needs periodic x and y");
  cudaStream_t st = (cudaStream_t)stream;
  const bool sc = self_consistent != 0;
  const double *Ex = sc ? ctx->Ex : nullptr, *Ey = sc ? ctx->Ey : nullptr;
  int chunks = 0;          // > 0: ctx->partials holds density partials of the current stage input
  return ssprk3_run_loop(
      f_dev, ctx->u1, ctx->u2, nsteps, sc,
      [&](const double* src) { return field4_from_partials_or_f(ctx, src, chunks, st); },
      [&](int, const double* src, const double* fn, double* dst, double c0, double c1) {
        return launch_rhs4(ctx, src, fn, Ex, Ey, dst, 1, c0, c1, dt, sc, &chunks, st);
      });
}

extern "C" int dg4_ssprk3_run_host(dg4_ctx* ctx, double* f_host, double dt, int32_t nsteps, int32_t self_consistent) {
  if (!ctx || !f_host) return fail(DG_ERR_INVALID_ARG, "dg4_ssprk3_run_host: null argument");
  DeviceGuard guard(ctx->desc.device);
  const size_t bytes = ctx->dof * sizeof(double);
  if (!ctx->f_stage) CUDA_TRY(cudaMalloc(&ctx->f_stage, bytes));
  CUDA_TRY(cudaMemcpyAsync(ctx->f_stage, f_host, bytes, cudaMemcpyHostToDevice, 0));
  int rc = dg4_ssprk3_run(ctx, ctx->f_stage, dt, nsteps, self_consistent, nullptr);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(f_host, ctx->f_stage, bytes, cudaMemcpyDeviceToHost, 0));
  CUDA_TRY(cudaStreamSynchronize(0));
  return DG_OK;
}

extern "C" int dg4_get_nodes(const dg4_ctx* ctx, int32_t dim, double* coords) {
  if (!ctx || dim < 0 || dim > 3 || !coords) return fail(DG_ERR_INVALID_ARG, "dg4_get_nodes: bad argument");
  memcpy(coords, ctx->coord_h[dim].data(), sizeof(double) * ctx->G[dim]);
  return DG_OK;
}

extern "C" double dg4_max_stable_dt(const dg4_ctx* ctx, double E_bound) {
  if (!ctx) return 0.0;
  // per-dimension limits add: sum_d |a_d|_max / (nu_d Delta_d) * dt <= 1, nu_d = the SSP-RK3 limit of the 1-D upwind operator
  auto vmax = [&](int d) { return std::fmax(std::fabs(ctx->desc.lo[d]), std::fabs(ctx->desc.hi[d])); };
  const double w = std::fabs(ctx->desc.omega_c), e = std::fabs(E_bound);
  const double amax[4] = {vmax(2), vmax(3), e + w * vmax(3), e + w * vmax(2)};
  double sum = 0.0;
  for (int d = 0; d < 4; ++d) {
    const double nu = dgsetup::rk3_cfl_limit(ctx->basis[d]);
    sum += amax[d] / (nu * (ctx->desc.hi[d] - ctx->desc.lo[d]) / ctx->N[d]);
  }
  return sum > 0.0 ? 1.0 / sum : INFINITY;
}

extern "C" int dg4_set_option(dg4_ctx* ctx, int32_t key, int64_t value) {
  if (!ctx) return fail(DG_ERR_INVALID_ARG, "dg4_set_option: null context");
  if (key == DG4_OPT_RHS_KERNEL && value >= 0 && value <= 4) { ctx->opt_kernel = (int)value; return DG_OK; }
  if (key == DG4_OPT_PROFILE && value >= 0 && value <= 1000000) { ctx->opt_profile = (int)value; ctx->prof_seen = 0; return DG_OK; }
  return fail(DG_ERR_INVALID_ARG, "dg4_set_option: unknown key or value");
}

extern "C" int dg4_get_profile(dg4_ctx* ctx, double* ms_total, int64_t* launches, int32_t reset) {
  if (!ctx) return fail(DG_ERR_INVALID_ARG, "dg4_get_profile: null context");
  DeviceGuard guard(ctx->desc.device);
  for (size_t i = 0; i + 1 < ctx->prof_events.size(); i += 2) {
    CUDA_TRY(cudaEventSynchronize(ctx->prof_events[i + 1]));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, ctx->prof_events[i], ctx->prof_events[i + 1]));
    ctx->prof_ms += ms;
    ctx->prof_launches += 1;
    cudaEventDestroy(ctx->prof_events[i]);
    cudaEventDestroy(ctx->prof_events[i + 1]);
  }
  ctx->prof_events.clear();
  if (ms_total) *ms_total = ctx->prof_ms;
  if (launches) *launches = ctx->prof_launches;
  if (reset) { ctx->prof_ms = 0.0; ctx->prof_launches = 0; }
  return DG_OK;
}

extern "C" int64_t dg4_launch_count(const dg4_ctx* ctx) { return ctx ? ctx->launches : 0; }
extern "C" const char* dg4_last_kernel(const dg4_ctx* ctx) { return ctx ? ctx->last_kernel.c_str() : "none"; }
