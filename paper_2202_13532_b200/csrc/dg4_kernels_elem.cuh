// 2D2V element kernel for equal even orders n = 4, 6, 8 in all four dimensions (sm_100a): the orders the n = 4 tiled
// kernel does not take (the paper runs n = 8).
//
// One CTA per element (n^4 nodes, n^3 threads), four line phases over two shared-memory copies of the element (the values
// f and the running sums), every phase with one line of n nodes per thread and the lanes of a warp along v, so that all
// shared-memory traffic is unit-stride 64-bit words (no bank conflicts, no redundant reads):
//   phase v  thread = (x, y, u) node: its v line comes straight from global memory (128-bit loads) and goes to shared
//            memory for the other phases; v contraction + lift in registers, sums to shared memory;
//   phase u  thread = (x, y, v) node: u line from shared memory, sums += ;      phase y  thread = (x, u, v): the same in y;
//   phase x  thread = (y, u, v) node: x line, final sums, stage combination with f_n, stores (lanes along v: full 32-byte
//            sectors), LGL-weighted sums -> one density partial per (g_x, g_y, element) by a fixed-order reduction.
// The upwind neighbour value of a line is one scalar per thread, read from global memory (L2) by the sign of the line's
// speed.  Per node: 4 shared-memory reads of f, 3 read-modify-writes of the sums -- a third of the traffic of walking the
// rows of a direction per owner thread -- and about 50 registers per thread (two CTAs per SM at n = 8).
#pragma once
#include "dg4_kernels.cuh"

namespace dg4 {

// Shared-memory position of element j of v line (row) r.  n = 8: one 64-byte pad after every 8 rows (rows 8 apart -- the
// lines of two neighbouring (x, y) nodes in the u phase -- then sit in opposite halves of a 128-byte bank line) and the 16-byte
// chunks of a row XORed with (r / 2) mod 4 (the 8 rows a quarter-warp stores in the v phase hit 8 distinct bank groups); the
// lanes of every other access run along j inside one row, where any permutation is conflict-free.
template <int n>
__device__ __forceinline__ int eaddr(int r, int j) {
  if (n == 8) return r * 8 + (r >> 3) * 8 + ((((j >> 1) ^ (r >> 1)) & 3) << 1) + (j & 1);
  return r * n + j;
}
template <int n>
constexpr int elem_array_doubles() { return n == 8 ? n * n * n * n + n * n * n : n * n * n * n; }
template <int n>
constexpr int elem_smem_doubles() { return 2 * elem_array_doubles<n>(); }

// Contraction + lift of one line: out[j] = s * ( sum_k U[j][k] f[k] - XiR[j] uR + XiL[j] uL ).
template <int n>
__device__ __forceinline__ void line_op(const Params& p, const double (&f)[n], double a, double J, double ext, double (&out)[n]) {
  const double uL = a > 0.0 ? ext : f[0], uR = a > 0.0 ? f[n - 1] : ext;
  const double s = J * a;
#pragma unroll
  for (int j = 0; j < n; ++j) {
    double v = p.Xin[2 * j] * uL;
    v = fma(-p.Xin[2 * j + 1], uR, v);
#pragma unroll
    for (int k = 0; k < n; ++k) v = fma(p.Un[j * n + k], f[k], v);
    out[j] = s * v;
  }
}

// Index of the upwind neighbour node of an element in dimension d (global node index), or -1 (zero inflow / no flux).
__device__ __forceinline__ int upwind_index(const Params& p, int d, int e, int n, double a) {
  if (a > 0.0) return e > 0 ? e * n - 1 : (p.bc[d] == 0 ? p.G[d] - 1 : -1);
  if (a < 0.0) return e < p.N[d] - 1 ? e * n + n : (p.bc[d] == 0 ? 0 : -1);
  return -1;
}

template <int n>
__global__ void __launch_bounds__(n * n * n, (n == 8 ? 2 : (n == 6 ? 4 : 8))) rhs4_elem_kernel(const Params p) {
  constexpr int H = n / 2, n2 = n * n;
  extern __shared__ double2 esm_raw[];
  double* T = reinterpret_cast<double*>(esm_raw);                 // [jx][jy][ju][jv] values of f
  double* A = T + elem_array_doubles<n>();                        // the running sums, same layout
  const int tid = threadIdx.x;
  const int c0 = tid % n, c1 = (tid / n) % n, c2 = tid / n2;      // c0 fastest
  const int eu = blockIdx.x / p.N[3], ev = blockIdx.x - eu * p.N[3], ey = blockIdx.y, ex = blockIdx.z;
  const int gx0 = ex * n, gy0 = ey * n, gu0 = eu * n, gv0 = ev * n;
  const long long s2 = p.G[3], s1 = s2 * p.G[2], s0 = s1 * p.G[1];
  const long long elem_off = gx0 * s0 + gy0 * s1 + gu0 * s2 + gv0;
  const bool use_fn = p.mode != 0 && p.fn != nullptr;

  // ---- phase v: thread = (jx, jy, ju) = (c2, c1, c0) ----------------------------------------------------------------
  {
    const long long line_off = elem_off + c2 * s0 + c1 * s1 + c0 * s2;
    double f[n], o[n];
    const double2* q = reinterpret_cast<const double2*>(p.f + line_off);
#pragma unroll
    for (int c = 0; c < H; ++c) { const double2 a = __ldg(q + c); f[2 * c] = a.x; f[2 * c + 1] = a.y; }
    const double eyf = p.Ey ? __ldg(p.Ey + (long long)(gx0 + c2) * p.G[1] + gy0 + c1) : 0.0;
    const double a = -eyf + p.omega_c * p.coord[2][gu0 + c0];
    const int g = upwind_index(p, 3, ev, n, a);
    const double ext = g >= 0 ? __ldg(p.f + line_off - gv0 + g) : 0.0;
#pragma unroll
    for (int c = 0; c < H; ++c) *reinterpret_cast<double2*>(T + eaddr<n>(tid, 2 * c)) = make_double2(f[2 * c], f[2 * c + 1]);
    line_op<n>(p, f, a, p.J[3], ext, o);
#pragma unroll
    for (int c = 0; c < H; ++c) *reinterpret_cast<double2*>(A + eaddr<n>(tid, 2 * c)) = make_double2(o[2 * c], o[2 * c + 1]);
  }
  __syncthreads();

  // ---- phase u: thread = (jx, jy, jv) = (c2, c1, c0); line over ju at stride n ---------------------------------------
  {
    const int row = (c2 * n + c1) * n;                                // + k
    double f[n], o[n];
#pragma unroll
    for (int k = 0; k < n; ++k) f[k] = T[eaddr<n>(row + k, c0)];
    const long long gxy = (long long)(gx0 + c2) * p.G[1] + gy0 + c1;
    const double exf = p.Ex ? __ldg(p.Ex + gxy) : 0.0;
    const double a = -exf - p.omega_c * p.coord[3][gv0 + c0];
    const int g = upwind_index(p, 2, eu, n, a);
    const double ext = g >= 0 ? __ldg(p.f + elem_off - gu0 * s2 + c2 * s0 + c1 * s1 + g * s2 + c0) : 0.0;
    line_op<n>(p, f, a, p.J[2], ext, o);
#pragma unroll
    for (int k = 0; k < n; ++k) A[eaddr<n>(row + k, c0)] += o[k];
  }
  __syncthreads();

  // ---- phase y: thread = (jx, ju, jv) = (c2, c1, c0); line over jy at stride n^2 -------------------------------------
  {
    const int row = c2 * n2 + c1;                                     // + k n
    double f[n], o[n];
#pragma unroll
    for (int k = 0; k < n; ++k) f[k] = T[eaddr<n>(row + k * n, c0)];
    const double a = p.coord[3][gv0 + c0];
    const int g = upwind_index(p, 1, ey, n, a);
    const double ext = g >= 0 ? __ldg(p.f + elem_off - gy0 * s1 + c2 * s0 + g * s1 + c1 * s2 + c0) : 0.0;
    line_op<n>(p, f, a, p.J[1], ext, o);
#pragma unroll
    for (int k = 0; k < n; ++k) A[eaddr<n>(row + k * n, c0)] += o[k];
  }
  __syncthreads();

  // ---- phase x: thread = (jy, ju, jv) = (c2, c1, c0); line over jx at stride n^3; epilogue ---------------------------
  {
    const int row = c2 * n + c1;                                      // + k n^2
    double f[n], o[n];
#pragma unroll
    for (int k = 0; k < n; ++k) f[k] = T[eaddr<n>(row + k * n2, c0)];
    const double a = p.coord[2][gu0 + c1];
    const int g = upwind_index(p, 0, ex, n, a);
    const long long node_off = elem_off + c2 * s1 + c1 * s2 + c0;          // + jx * s0
    double ext = g >= 0 ? __ldg(p.f + node_off - gx0 * s0 + g * s0) : 0.0;
    if (p.bc[0] == 2) {        // x-slab: at the slab's two x faces the exterior state comes from the halo planes
      if (a > 0.0 && ex == 0) ext = __ldg(p.xhalo + node_off - gx0 * s0);
      else if (a < 0.0 && ex == p.N[0] - 1) ext = __ldg(p.xhalo + s0 + node_off - gx0 * s0);
    }
    double fnv[n];
    if (use_fn) {
#pragma unroll
      for (int k = 0; k < n; ++k) fnv[k] = __ldcs(p.fn + node_off + k * s0);
    }
    line_op<n>(p, f, a, p.J[0], ext, o);
    const double w = p.partials ? p.wqu[gu0 + c1] * p.wqv[gv0 + c0] : 0.0;
#pragma unroll
    for (int k = 0; k < n; ++k) {
      double r = o[k] + A[eaddr<n>(row + k * n2, c0)];
      if (p.mode != 0) {
        r = p.c1 * fma(p.dt, r, f[k]);
        if (use_fn) r = fma(p.c0, fnv[k], r);
      }
      __stcs(p.out + node_off + k * s0, r);
      o[k] = w * r;
    }
    if (p.partials) {
      // density of the element at (jx, jy): sum over (ju, jv) in a fixed order
      // (each thread overwrites the sums it has just consumed: A becomes the weighted outputs, [jx][jy][ju*n + jv])
#pragma unroll
      for (int k = 0; k < n; ++k) A[eaddr<n>(row + k * n2, c0)] = o[k];
      __syncthreads();
      if (tid < n2) {
        double s = 0.0;
        for (int i = 0; i < n2; ++i) s += A[eaddr<n>(tid * n + i / n, i % n)];
        const int jx = tid / n, jy = tid - jx * n;
        p.partials[((long long)(gx0 + jx) * p.G[1] + gy0 + jy) * p.chunks + eu * p.N[3] + ev] = s;
      }
    }
  }
}

}  // namespace dg4
