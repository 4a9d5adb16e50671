// Generic (any order 2..10, per-dimension orders, 1D1V or 1D2V) kernels: one thread per node,
// lines read straight from global memory.  Correct for every supported shape; the tiled sm_100a
// kernels in dg_kernels_tiled.cuh replace them on the 1D2V equal-order fast path.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace dgk {

struct GenericParams {
  int ndim;
  int N[3], n[3], G[3], bc[3];
  const double* ups[3];     // reference Upsilon [n][n]
  const double* lift[3];    // reference Xi [n][2]
  const double* coord[3];   // node coordinates
  double J[3];
  double omega_c;
  const double* E;          // [G0] or nullptr
  const double* xhalo;      // exterior x-face planes [2][G1*G2] (bc[0] = 2) or nullptr
  const double* f;          // stage input
  const double* fn;         // f_n for the stage combination (mode 1) or nullptr
  double* out;
  double c0, c1, dt;        // out = c0*fn + c1*(f + dt*rhs)   (mode 1);   out = rhs (mode 0)
  int mode;
  double* push_left;        // x-slab face push: plane [G1*G2] in the left neighbour's halo for this slab's first x plane of out
  double* push_right;       // ... and in the right neighbour's halo for the last x plane (mode 1 only), or nullptr
  int strong;               // 1: strong form Eq. 15 -- ups holds -D and the lift acts on (upwind state - own face value)
  long long dof;
};

// Weak form Eq. 14 reduced by Eq. 20-21, upwind flux Eq. 23,
// speeds Eq. 28, optional Shu-Osher stage combination.
__global__ void __launch_bounds__(256) rhs_generic_kernel(const GenericParams p) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < p.dof; idx += stride) {
    int g[3] = {0, 0, 0};
    long long r = idx;
    for (int d = p.ndim - 1; d >= 0; --d) { g[d] = (int)(r % p.G[d]); r /= p.G[d]; }
    long long strd[3];
    strd[p.ndim - 1] = 1;
    for (int d = p.ndim - 2; d >= 0; --d) strd[d] = strd[d + 1] * p.G[d + 1];
    const double Ex = p.E ? p.E[g[0]] : 0.0;
    double a[3];
    if (p.ndim == 2) {
      a[0] = p.coord[1][g[1]];
      a[1] = -Ex;
    } else {
      a[0] = p.coord[1][g[1]];
      a[1] = -Ex - p.omega_c * p.coord[2][g[2]];
      a[2] = p.omega_c * p.coord[1][g[1]];
    }
    double rhs = 0.0;
    for (int d = 0; d < p.ndim; ++d) {
      const int n = p.n[d], N = p.N[d];
      const int e = g[d] / n, j = g[d] - e * n;
      const long long base = idx - (long long)j * strd[d];        // node 0 of this line
      const double* U = p.ups[d] + j * n;
      double vol = 0.0;
      for (int k = 0; k < n; ++k) vol = fma(U[k], p.f[base + k * strd[d]], vol);
      const double own0 = p.f[base], own1 = p.f[base + (long long)(n - 1) * strd[d]];
      double uL = 0.0, uR = 0.0;                                  // upwind states at the two faces
      if (a[d] > 0.0) {
        uR = own1;
        if (e > 0) uL = p.f[base - strd[d]];
        else if (p.bc[d] == 0) uL = p.f[base + ((long long)(N - 1) * n + (n - 1)) * strd[d]];
        else if (p.bc[d] == 2) uL = p.xhalo[idx % strd[0]];                       // left neighbour's last x plane
      } else if (a[d] < 0.0) {
        uL = own0;
        if (e < N - 1) uR = p.f[base + (long long)n * strd[d]];
        else if (p.bc[d] == 0) uR = p.f[base - (long long)e * n * strd[d]];
        else if (p.bc[d] == 2) uR = p.xhalo[strd[0] + idx % strd[0]];             // right neighbour's first x plane
      }
      if (p.strong) { uL -= own0; uR -= own1; }                  // Eq. 15: Xi (F - F*) with -D F
      const double xl = p.lift[d][2 * j], xr = p.lift[d][2 * j + 1];
      rhs += (p.J[d] * a[d]) * (vol - xr * uR + xl * uL);
    }
    if (p.mode == 0) p.out[idx] = rhs;
    else {
      const double v = p.f[idx] + p.dt * rhs;
      const double o = (p.fn ? p.c0 * p.fn[idx] : 0.0) + p.c1 * v;
      p.out[idx] = o;
      if (p.push_left && g[0] == 0) p.push_left[idx % strd[0]] = o;
      if (p.push_right && g[0] == p.G[0] - 1) p.push_right[idx % strd[0]] = o;
    }
  }
}

// Non-finite guard for the CFL blow-up case (the stable time step depends on the order):
// flag[0] becomes 1 if any of the n values is Inf or NaN (the caller zeroes it first).  8 B per value, HBM-bound.
__global__ void __launch_bounds__(256) check_finite_kernel(const double* __restrict__ f, long long n, int* __restrict__ flag) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  const long long i0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if ((reinterpret_cast<uintptr_t>(f) & 15) == 0) {
    const double2* f2 = reinterpret_cast<const double2*>(f);
    const long long n2 = n >> 1;
    for (long long i = i0; i < n2; i += stride) {
      const double2 v = __ldcs(f2 + i);
      bad |= !(fabs(v.x) <= 1.7976931348623157e308) | !(fabs(v.y) <= 1.7976931348623157e308);
    }
    if ((n & 1) && i0 == 0) bad |= !(fabs(f[n - 1]) <= 1.7976931348623157e308);
  } else {
    for (long long i = i0; i < n; i += stride) bad |= !(fabs(f[i]) <= 1.7976931348623157e308);
  }
  if (__syncthreads_or(bad ? 1 : 0) && threadIdx.x == 0) atomicOr(flag, 1);
}

// Deterministic block reduction (fixed tree): every thread passes its partial, thread 0 gets the sum.
template <int THREADS>
__device__ __forceinline__ double block_reduce_sum(double v, double* smem) {
  const int tid = threadIdx.x;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
  if ((tid & 31) == 0) smem[tid >> 5] = v;
  __syncthreads();
  double tot = 0.0;
  if (tid < 32) {
    tot = (tid < THREADS / 32) ? smem[tid] : 0.0;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) tot += __shfl_down_sync(0xffffffffu, tot, off);
  }
  __syncthreads();
  return tot;
}

// Eq. 27: partial[gx][chunk] = sum over this chunk of the velocity plane of
// wq1[g1] * wq2[g2] * f.  grid = (chunks, G0).  plane = G1*G2 (G2 = 1 for 1D1V).
__global__ void __launch_bounds__(256) density_partial_kernel(const double* __restrict__ f, const double* __restrict__ wq1,
                                                              const double* __restrict__ wq2, int G1, int G2,
                                                              int rows_per_chunk, double* __restrict__ partial) {
  __shared__ double red[8];
  const int gx = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int r0 = chunk * rows_per_chunk;
  const int r1 = min(G1, r0 + rows_per_chunk);
  const double* plane = f + (size_t)gx * G1 * G2;
  double acc = 0.0;
  if (G2 == 1) {
    for (int i = r0 + threadIdx.x; i < r1; i += 256) acc = fma(wq1[i], plane[i], acc);
  } else {
    for (int r = r0; r < r1; ++r) {
      const double* row = plane + (size_t)r * G2;
      double racc = 0.0;
      for (int i = threadIdx.x; i < G2; i += 256) racc = fma(wq2[i], row[i], racc);
      acc = fma(wq1[r], racc, acc);
    }
  }
  const double tot = block_reduce_sum<256>(acc, red);
  if (threadIdx.x == 0) partial[(size_t)gx * nchunks + chunk] = tot;
}

// Same sum for even G2 and a 16-byte aligned f, shaped for HBM bandwidth: thread = (row lane, column pair),
// 128-bit loads, UNR rows in flight per thread; the weight of the column pair is applied once at the end.
// CP = column pairs covered per pass (power of two <= 256), 256 / CP row lanes.  Fixed association: deterministic.
template <int UNR>
__global__ void __launch_bounds__(256) density_partial_vec_kernel(const double* __restrict__ f, const double* __restrict__ wq1,
                                                                  const double* __restrict__ wq2, int G1, int G2, int rows_per_chunk,
                                                                  int CP, double* __restrict__ partial) {
  __shared__ double red[8];
  const int gx = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int r0 = chunk * rows_per_chunk;
  const int r1 = min(G1, r0 + rows_per_chunk);
  const int ncol2 = G2 >> 1;
  const int cp0 = threadIdx.x & (CP - 1), rl = threadIdx.x / CP, RL = 256 / CP;
  const double2* plane = reinterpret_cast<const double2*>(f + (size_t)gx * G1 * G2);
  double acc = 0.0;
  for (int cp = cp0; cp < ncol2; cp += CP) {
    const double2 w2 = *reinterpret_cast<const double2*>(wq2 + 2 * cp);
    const double2* col = plane + cp;
    double a0 = 0.0, a1 = 0.0;
    int r = r0 + rl;
    for (; r + (UNR - 1) * RL < r1; r += UNR * RL) {
      double2 v[UNR];
      double w[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) { v[u] = __ldcs(col + (size_t)(r + u * RL) * ncol2); w[u] = wq1[r + u * RL]; }
#pragma unroll
      for (int u = 0; u < UNR; ++u) { a0 = fma(w[u], v[u].x, a0); a1 = fma(w[u], v[u].y, a1); }
    }
    for (; r < r1; r += RL) {
      const double2 v = __ldcs(col + (size_t)r * ncol2);
      const double w = wq1[r];
      a0 = fma(w, v.x, a0); a1 = fma(w, v.y, a1);
    }
    acc = fma(w2.x, a0, fma(w2.y, a1, acc));
  }
  const double tot = block_reduce_sum<256>(acc, red);
  if (threadIdx.x == 0) partial[(size_t)gx * nchunks + chunk] = tot;
}

// rho[gx] = sum_c partial[gx][c] in index order (deterministic).  One warp per gx.
__global__ void __launch_bounds__(128) density_finish_kernel(const double* __restrict__ partial, int nchunks, int G0,
                                                             double* __restrict__ rho) {
  const int gx = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (gx >= G0) return;
  double acc = 0.0;
  for (int c = lane; c < nchunks; c += 32) acc += partial[(size_t)gx * nchunks + c];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
  if (lane == 0) rho[gx] = acc;
}

// c[b][p] = sum_g T_p[g] rho[b][g], Eq. 63.  grid = (P1, batch), 128 threads.
__global__ void __launch_bounds__(128) project_simple_kernel(const double* __restrict__ T, const double* __restrict__ rho,
                                                             int G, int P1, double* __restrict__ c) {
  __shared__ double red[8];
  const int p = blockIdx.x, b = blockIdx.y;
  const double* tr = T + (size_t)(2 * p) * G;
  const double* ti = tr + G;
  const double* r = rho + (size_t)b * G;
  double are = 0.0, aim = 0.0;
  for (int g = threadIdx.x; g < G; g += 128) {
    const double v = r[g];
    are = fma(tr[g], v, are);
    aim = fma(ti[g], v, aim);
  }
  const double sre = block_reduce_sum<128>(are, red);
  const double sim = block_reduce_sum<128>(aim, red);
  if (threadIdx.x == 0) {
    c[((size_t)b * P1 + p) * 2] = sre;
    c[((size_t)b * P1 + p) * 2 + 1] = sim;
  }
}

// E[b][g] = sum_{q} S[g][q] c[b][q], q = 2p + {re,im}: Eq. 71 with the Poisson factor
// folded into S and the p = 0 columns zero.  One warp per output node.
__global__ void __launch_bounds__(128) synth_simple_kernel(const double* __restrict__ S, const double* __restrict__ c,
                                                           int G, int Q, double* __restrict__ E) {
  const int g = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31, b = blockIdx.y;
  if (g >= G) return;
  const double* s = S + (size_t)g * Q;
  const double* cb = c + (size_t)b * Q;
  double acc = 0.0;
  for (int q = lane; q < Q; q += 32) acc = fma(s[q], cb[q], acc);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
  if (lane == 0) E[(size_t)b * G + g] = acc;
}

// Broken l2 norm of Eq. 72 of the difference of two nodal vectors on the x grid:
//   eps = (1/N) sum_m sqrt( int_m (u - v)^2 dx ),  the integrand being the element's degree-(n-1) interpolant, integrated
// exactly by the LGL mass matrix of Eq. 50: d^T M d = sum_j w_j d_j^2 - alpha (sum_j w_j P_{n-1}(xi_j) d_j)^2.
// One CTA per vector; elements in a fixed order per thread, fixed shared-memory tree: deterministic.
__global__ void __launch_bounds__(256) broken_l2_kernel(const double* __restrict__ u, const double* __restrict__ v,
                                                        const double* __restrict__ wg /*[2][n]: w_j, w_j P_{n-1}(xi_j)*/,
                                                        const double* __restrict__ half_dx_m /*[N] or nullptr: equal widths*/,
                                                        int N, int n, double alpha, double half_dx, double* __restrict__ eps) {
  __shared__ double red[256];
  const size_t off = (size_t)blockIdx.x * N * n;
  double acc = 0.0;
  for (int m = threadIdx.x; m < N; m += 256) {
    double s2 = 0.0, sp = 0.0;
    for (int j = 0; j < n; ++j) {
      const size_t g = off + (size_t)m * n + j;
      const double d = u[g] - (v ? v[g] : 0.0);
      s2 = fma(wg[j] * d, d, s2);
      sp = fma(wg[n + j], d, sp);
    }
    acc += sqrt(fmax(0.0, fma(-alpha * sp, sp, s2)) * (half_dx_m ? half_dx_m[m] : half_dx));
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) eps[blockIdx.x] = red[0] / (double)N;
}

// Domain-integrated field energy (Fig. 10): W = (1/2) int E^2 dx, each element's interpolant integrated exactly
// by the mass matrix of Eq. 50 in the same rank-one form as above.  One CTA per vector, fixed order: deterministic.
__global__ void __launch_bounds__(256) field_energy_kernel(const double* __restrict__ E, const double* __restrict__ wg,
                                                           const double* __restrict__ half_dx_m, int N, int n, double alpha,
                                                           double half_dx, double* __restrict__ W) {
  __shared__ double red[256];
  const size_t off = (size_t)blockIdx.x * N * n;
  double acc = 0.0;
  for (int m = threadIdx.x; m < N; m += 256) {
    double s2 = 0.0, sp = 0.0;
    for (int j = 0; j < n; ++j) {
      const double e = E[off + (size_t)m * n + j];
      s2 = fma(wg[j] * e, e, s2);
      sp = fma(wg[n + j], e, sp);
    }
    acc = fma(fma(-alpha * sp, sp, s2), half_dx_m ? half_dx_m[m] : half_dx, acc);
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) W[blockIdx.x] = 0.5 * red[0];
}

}  // namespace dgk
