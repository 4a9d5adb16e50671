// Internal context of the C-ABI library (not part of the public boundary).
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <cstdint>
#include <map>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "../../include/dgvlasov.h"
#include "dg_setup.hpp"

// Every entry point runs with the context's device current and restores the caller's on return (a process may hold
// contexts on several GPUs).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device property of a kernel: remember the largest value set per
// (kernel, device) instead of a process-wide flag.  Call with the target device current.
inline cudaError_t ensure_dyn_smem(const void* func, size_t bytes) {
  static std::mutex mu;
  static std::map<std::pair<const void*, int>, size_t> done;
  if (bytes <= 48 * 1024) return cudaSuccess;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  size_t& cur = done[std::make_pair(func, dev)];
  if (bytes <= cur) return cudaSuccess;
  e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess) cur = bytes;
  return e;
}

// key of a cached TMA descriptor: base pointer + box + swizzle + outer extent
struct TmapKey {
  const void* base; int b0, b1, b2, swz, outer;
  bool operator<(const TmapKey& o) const {
    if (base != o.base) return base < o.base;
    if (b0 != o.b0) return b0 < o.b0;
    if (b1 != o.b1) return b1 < o.b1;
    if (b2 != o.b2) return b2 < o.b2;
    if (swz != o.swz) return swz < o.swz;
    return outer < o.outer;
  }
};

struct ProfRecord { cudaEvent_t e0, e1; int stage; };

struct dg_ctx {
  dg_grid_desc desc;
  int ndim = 0;
  int N[3] = {0, 0, 0};       // elements per dim
  int n[3] = {0, 0, 0};       // nodes per element per dim
  int G[3] = {1, 1, 1};       // flat nodes per dim (1 for unused dims)
  size_t dof = 0;             // prod G over used dims (0 for ndim == 1)
  int pmax = 0, P1 = 1;
  double J[3] = {0, 0, 0};    // 2 / Delta_d                                     (Eq. 61)
  dgsetup::Basis1D basis[3];
  std::vector<double> coord_h[3];
  std::vector<double> T_h;    // kept on the host only until uploaded, then for dg_get_transform

  // device constants (one allocation, carved)
  void* dev_block = nullptr;
  double* d_ups[3] = {nullptr, nullptr, nullptr};    // reference Upsilon [n][n]
  double* d_lift[3] = {nullptr, nullptr, nullptr};   // reference Xi [n][2]
  double* d_negD[3] = {nullptr, nullptr, nullptr};   // -D [n][n] (Eq. 55): the volume operator of the strong form, Eq. 15
  double* d_coord[3] = {nullptr, nullptr, nullptr};  // node coordinates [G_d]
  double* d_wq[3] = {nullptr, nullptr, nullptr};     // quadrature weight w_b / J_d per flat node [G_d]
  double* d_T = nullptr;      // [2*P1][G0]   rows 2p / 2p+1 = Re / Im of T_p (Eq. 63)
  double* d_S = nullptr;      // [G0][2*P1]   synthesis rows of Eq. 71 with -1/(i k_p) folded in
  void* dense_block = nullptr;  // T and S when built on first use (large x-only contexts served by the FFT kernel)
  // FFT-factorised field solve (field_fft_kernel): nullptr when the grid does not qualify
  double* d_AD = nullptr;     // [P1][2][n0] complex: A_p^j, D_p^j
  double* d_W = nullptr;      // [N0/2] complex twiddles
  int sm_count = 148;
  std::vector<double> edges;  // element edges of a non-uniform x-only context (dg_create_field_nonuniform), else empty
  double* d_half_dx = nullptr;  // [N0] half widths of such a context
  double* d_wg = nullptr;     // [2][n0]: w_j and w_j P_{n-1}(xi_j) of the x basis (broken l2 norm, Eq. 50 / 72)
  // one-launch field solve (field_fused_kernel): per-CTA shares of c_q
  double* d_cpart = nullptr;  // [2*P1][fused_grid]
  int fused_rows = 0, fused_grid = 0;

  // caller-provided workspace
  void* ws = nullptr;
  size_t ws_bytes = 0;
  double *u1 = nullptr, *u2 = nullptr, *partials = nullptr, *rho = nullptr, *E = nullptr, *cbuf = nullptr;
  size_t cbuf_doubles = 0, partials_doubles = 0;

  const double* xhalo = nullptr;   // caller-owned exterior x-face planes (bc[0] = DG_BC_HALO)
  double* push_left = nullptr;     // dg_set_xhalo_push: where dg_rk_stage also stores the first / last x plane of out
  double* push_right = nullptr;

  // library-owned staging for the host entry point
  double* f_stage = nullptr;

  int64_t launches = 0;
  int opt_rhs_kernel = 0, opt_field_kernel = 0, opt_profile = 0, opt_pdl = 1;
  int opt_form = 0;           // 0 weak form (Eq. 14), 1 strong form (Eq. 15)
  // profile mode: (start, stop) event pairs around RHS launches, tagged with the RK stage (0 = not inside dg_ssprk3_*)
  std::vector<ProfRecord> prof_events;
  int64_t prof_seen = 0;      // RHS launches since profile mode was set (every opt_profile-th one is bracketed)
  int cur_stage = 0;          // stage tag of the launch being issued
  double prof_ms[4] = {0, 0, 0, 0};
  int64_t prof_n[4] = {0, 0, 0, 0};
  std::map<TmapKey, CUtensorMap> tmaps;   // TMA descriptors of the arrays seen so far (f, u1, u2, halos: a handful)
  std::string last_kernel = "none";
  std::string last_field_kernel = "none";
  double cfl_limit = -1.0;    // lazily computed
};
