// 2D2V element kernel for equal even orders n = 4, 6, 8 in all four dimensions (sm_100a): the orders the n = 4 tiled
// kernel does not take (the paper runs n = 8).
//
// One CTA per element (n^4 nodes), n^3 threads, thread = (x node, y node, u node) owns the v line through it (n contiguous
// doubles: 128-bit global loads and stores) and keeps its n sums in registers for the whole kernel:
//   v direction  registers only (operator entries are compile-time indexed kernel parameters);
//   u, y, x      the line through each of the thread's nodes runs over n v-lines of other threads: the CTA's lines sit in
//                shared memory (row pitch chosen so that the n lanes that differ in the u node hit distinct bank groups),
//                the thread walks the n rows of the direction with its own operator row (n per-thread coefficients);
//   faces        the upwind neighbour rows of the element (x: the side the sign of u selects; y, u: both sides, the sign
//                changes inside a row) are staged in shared memory by the first 5 n^2 threads, the v face is one scalar
//                per thread;
//   epilogue     stage combination, LGL-weighted line sums reduced over the u nodes in a fixed order -> one density
//                partial per (g_x, g_y, element).
// Shared-memory traffic is 3 n reads per node (the price of general n in four dimensions), so the kernel is bound by
// shared-memory bandwidth, not HBM; it replaces the one-thread-per-node kernel, which reads every line from L1/L2.
#pragma once
#include "dg4_kernels.cuh"

namespace dg4 {

template <int n>
constexpr int elem_pitch() { return n == 8 ? 10 : n; }            // doubles per shared-memory row
template <int n>
constexpr int elem_smem_doubles() { return n * n * n * elem_pitch<n>() + 5 * n * n * elem_pitch<n>() + n * n * n + 2 * n + n * (n + 1) + (n * (n + 1)) % 2; }

template <int n>
__global__ void __launch_bounds__(n * n * n, 1) rhs4_elem_kernel(const Params p) {
  constexpr int NT = n * n * n, RP = elem_pitch<n>(), H = n / 2;
  extern __shared__ double2 esm_raw[];
  double* T = reinterpret_cast<double*>(esm_raw);                 // [n^3][RP] v lines of the element
  double* hx = T + NT * RP;                                       // [n^2 (jy, ju)][RP]
  double* hy = hx + n * n * RP;                                   // [2][n^2 (jx, ju)][RP]
  double* hu = hy + 2 * n * n * RP;                               // [2][n^2 (jx, jy)][RP]
  double* red = hu + 2 * n * n * RP;                              // [n^3]
  double* Xs = red + n * n * n;                                   // [n][2] lift
  double* Us = Xs + 2 * n;                                   // [n][n+1]: the per-thread operator rows (padded: conflict-free)
  const int tid = threadIdx.x;
  const int ju = tid % n, jy = (tid / n) % n, jx = tid / (n * n);
  const int eu = blockIdx.x / p.N[3], ev = blockIdx.x - eu * p.N[3], ey = blockIdx.y, ex = blockIdx.z;
  const int gx0 = ex * n, gy0 = ey * n, gu0 = eu * n, gv0 = ev * n;
  const long long s2 = p.G[3], s1 = s2 * p.G[2], s0 = s1 * p.G[1];
  const long long elem_off = gx0 * s0 + gy0 * s1 + gu0 * s2 + gv0;
  const long long line_off = elem_off + jx * s0 + jy * s1 + ju * s2;
  const bool use_fn = p.mode != 0 && p.fn != nullptr;

  // own line, f_n line
  double fo[n], fnl[n];
  {
    const double2* q = reinterpret_cast<const double2*>(p.f + line_off);
#pragma unroll
    for (int c = 0; c < H; ++c) { const double2 a = __ldg(q + c); fo[2 * c] = a.x; fo[2 * c + 1] = a.y; }
    if (use_fn) {
      const double2* qn = reinterpret_cast<const double2*>(p.fn + line_off);
#pragma unroll
      for (int c = 0; c < H; ++c) { const double2 a = __ldcs(qn + c); fnl[2 * c] = a.x; fnl[2 * c + 1] = a.y; }
    }
  }
  // face rows: r < n^2: x face; then y lo, y hi, u lo, u hi
  for (int r = tid; r < 5 * n * n; r += NT) {
    const int which = r / (n * n), rr = r - which * n * n, a = rr / n, b = rr - a * n;
    long long src = -1;
    double* dst;
    if (which == 0) {                                             // (jy, ju) = (a, b): side by the sign of u
      const double u = p.coord[2][gu0 + b];
      int g = -1;
      if (u > 0.0) g = ex > 0 ? gx0 - 1 : (p.bc[0] == 0 ? p.G[0] - 1 : -1);
      else if (u < 0.0) g = ex < p.N[0] - 1 ? gx0 + n : (p.bc[0] == 0 ? 0 : -1);
      if (g >= 0) src = g * s0 + (gy0 + a) * s1 + (gu0 + b) * s2 + gv0;
      dst = hx + rr * RP;
    } else if (which <= 2) {                                      // (jx, ju) = (a, b)
      const int g = which == 1 ? (ey > 0 ? gy0 - 1 : (p.bc[1] == 0 ? p.G[1] - 1 : -1))
                               : (ey < p.N[1] - 1 ? gy0 + n : (p.bc[1] == 0 ? 0 : -1));
      if (g >= 0) src = (gx0 + a) * s0 + g * s1 + (gu0 + b) * s2 + gv0;
      dst = hy + ((which - 1) * n * n + rr) * RP;
    } else {                                                      // (jx, jy) = (a, b)
      const int g = which == 3 ? (eu > 0 ? gu0 - 1 : (p.bc[2] == 0 ? p.G[2] - 1 : -1))
                               : (eu < p.N[2] - 1 ? gu0 + n : (p.bc[2] == 0 ? 0 : -1));
      if (g >= 0) src = (gx0 + a) * s0 + (gy0 + b) * s1 + g * s2 + gv0;
      dst = hu + ((which - 3) * n * n + rr) * RP;
    }
    double2* d2 = reinterpret_cast<double2*>(dst);
    if (src >= 0) {
      const double2* q = reinterpret_cast<const double2*>(p.f + src);
#pragma unroll
      for (int c = 0; c < H; ++c) d2[c] = __ldg(q + c);
    } else {
#pragma unroll
      for (int c = 0; c < H; ++c) d2[c] = make_double2(0.0, 0.0);
    }
  }
  // speeds
  const long long gxy = (long long)(gx0 + jx) * p.G[1] + gy0 + jy;
  const double exf = p.Ex ? __ldg(p.Ex + gxy) : 0.0, eyf = p.Ey ? __ldg(p.Ey + gxy) : 0.0;
  const double uu = p.coord[2][gu0 + ju];
  double vv[n];
#pragma unroll
  for (int j = 0; j < n; ++j) vv[j] = p.coord[3][gv0 + j];
  const double a_v = -eyf + p.omega_c * uu;
  // v face: one scalar
  double vface = 0.0;
  {
    int g = -1;
    if (a_v > 0.0) g = ev > 0 ? gv0 - 1 : (p.bc[3] == 0 ? p.G[3] - 1 : -1);
    else if (a_v < 0.0) g = ev < p.N[3] - 1 ? gv0 + n : (p.bc[3] == 0 ? 0 : -1);
    if (g >= 0) vface = __ldg(p.f + line_off - gv0 + g);
  }
  if (tid < n * n) Us[(tid / n) * (n + 1) + tid % n] = p.Un[tid];
  if (tid < 2 * n) Xs[tid] = p.Xin[tid];
  // own line to shared memory
  {
    double2* t2 = reinterpret_cast<double2*>(T + tid * RP);
#pragma unroll
    for (int c = 0; c < H; ++c) t2[c] = make_double2(fo[2 * c], fo[2 * c + 1]);
  }
  __syncthreads();

  double rhs[n];
  // v direction: the thread's own line
  {
    const double uL = a_v > 0.0 ? vface : fo[0], uR = a_v > 0.0 ? fo[n - 1] : vface;
    const double sv = p.J[3] * a_v;
#pragma unroll
    for (int j = 0; j < n; ++j) {
      double v = p.Xin[2 * j] * uL;
      v = fma(-p.Xin[2 * j + 1], uR, v);
#pragma unroll
      for (int k = 0; k < n; ++k) v = fma(p.Un[j * n + k], fo[k], v);
      rhs[j] = sv * v;
    }
  }
  // u, y, x: walk the n rows of the direction
#pragma unroll
  for (int d = 2; d >= 0; --d) {
    const int jd = d == 2 ? ju : (d == 1 ? jy : jx);
    const int row0 = d == 2 ? tid - ju : (d == 1 ? tid - jy * n : tid - jx * n * n);
    const int rstep = d == 2 ? 1 : (d == 1 ? n : n * n);
    double acc[n], first[n], last[n], cf[n];
#pragma unroll
    for (int k = 0; k < n; ++k) cf[k] = Us[jd * (n + 1) + k];
#pragma unroll
    for (int j = 0; j < n; ++j) acc[j] = 0.0;
#pragma unroll
    for (int k = 0; k < n; ++k) {
      const double c = cf[k];
      const double2* t2 = reinterpret_cast<const double2*>(T + (row0 + k * rstep) * RP);
#pragma unroll
      for (int h = 0; h < H; ++h) {
        const double2 a = t2[h];
        acc[2 * h] = fma(c, a.x, acc[2 * h]); acc[2 * h + 1] = fma(c, a.y, acc[2 * h + 1]);
        if (k == 0) { first[2 * h] = a.x; first[2 * h + 1] = a.y; }
        if (k == n - 1) { last[2 * h] = a.x; last[2 * h + 1] = a.y; }
      }
    }
    const double xl = Xs[2 * jd], xr = Xs[2 * jd + 1];
    const double* lo = d == 2 ? hu + (jx * n + jy) * RP : (d == 1 ? hy + (jx * n + ju) * RP : hx + (jy * n + ju) * RP);
    const double* hi = d == 0 ? lo : lo + n * n * RP;
    double flo[n], fhi[n];
#pragma unroll
    for (int h = 0; h < H; ++h) {
      const double2 a = reinterpret_cast<const double2*>(lo)[h], b = reinterpret_cast<const double2*>(hi)[h];
      flo[2 * h] = a.x; flo[2 * h + 1] = a.y; fhi[2 * h] = b.x; fhi[2 * h + 1] = b.y;
    }
#pragma unroll
    for (int j = 0; j < n; ++j) {
      const double a = d == 2 ? -exf - p.omega_c * vv[j] : (d == 1 ? vv[j] : uu);
      const double uL = a > 0.0 ? flo[j] : first[j], uR = a > 0.0 ? last[j] : fhi[j];
      rhs[j] = fma(p.J[d] * a, acc[j] - xr * uR + xl * uL, rhs[j]);
    }
  }
  // stage combination, store, density partial
  double dens = 0.0;
  {
    double o[n];
#pragma unroll
    for (int j = 0; j < n; ++j) {
      if (p.mode == 0) o[j] = rhs[j];
      else {
        o[j] = p.c1 * fma(p.dt, rhs[j], fo[j]);
        if (use_fn) o[j] = fma(p.c0, fnl[j], o[j]);
      }
    }
    double2* q = reinterpret_cast<double2*>(p.out + line_off);
#pragma unroll
    for (int c = 0; c < H; ++c) __stcs(q + c, make_double2(o[2 * c], o[2 * c + 1]));
    if (p.partials) {
#pragma unroll
      for (int j = 0; j < n; ++j) dens = fma(p.wqv[gv0 + j], o[j], dens);
      dens *= p.wqu[gu0 + ju];
    }
  }
  if (p.partials) {
    red[tid] = dens;
    __syncthreads();
    if (ju == 0) {
      double s = 0.0;
#pragma unroll
      for (int k = 0; k < n; ++k) s += red[tid + k];
      p.partials[gxy * p.chunks + eu * p.N[3] + ev] = s;
    }
  }
}

}  // namespace dg4
