// 2D2V kernels (include/dgvlasov2d2v.h): the four-dimensional RHS + stage, and the small kernels of the 2-D field solve.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace dg4 {

struct Params {
  int N[4], n[4], G[4], bc[4];
  double J[4];
  const double* coord[4];    // node coordinates per dimension
  const double* ups[4];      // reference Upsilon [n][n] (generic kernel)
  const double* lift[4];     // reference Xi [n][2]
  double U[16], Xi[8];       // the same operators for n = 4 (tiled kernel: kernel-parameter constant bank)
  double Un[64], Xin[16];    // ... and for the element kernel's order n <= 8: Un[j*n + k], Xin[2*j + {L,R}]
  double omega_c;
  const double* Ex;          // [G0*G1] or nullptr
  const double* Ey;
  const double* f;           // stage input
  const double* fn;          // step input for the stage combination, or nullptr
  double* out;
  double c0, c1, dt;         // mode 1: out = c0*fn + c1*(f + dt*rhs);  mode 0: out = rhs
  int mode;
  const double* wqu;         // quadrature weights w_b/J per flat u / v node (density partials)
  const double* wqv;
  double* partials;          // [G0*G1][chunks] per-tile density partials of out, or nullptr
  int chunks;
  int bx_log2;               // tiled kernel: log2 of the x-elements per rasterisation group
  int wide_st;               // tiled kernel: out is 32-byte aligned (256-bit stores)
  const double* xhalo;       // bc[0] = DG_BC_HALO: exterior x-face planes [2][G1][G2][G3] of an x-slab (dg4_set_xhalo)
  long long dof;
};

// One thread per node, lines read straight from global memory: any orders 2..10, any element counts.
// Weak form Eq. 14 reduced by Eq. 20-21, upwind flux Eq. 23, speeds Eq. 28.
__global__ void __launch_bounds__(256) rhs4_generic_kernel(const Params p) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  long long strd[4];
  strd[3] = 1;
  for (int d = 2; d >= 0; --d) strd[d] = strd[d + 1] * p.G[d + 1];
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < p.dof; idx += stride) {
    int g[4];
    long long r = idx;
    for (int d = 3; d >= 0; --d) { g[d] = (int)(r % p.G[d]); r /= p.G[d]; }
    const long long gxy = (long long)g[0] * p.G[1] + g[1];
    const double ex = p.Ex ? p.Ex[gxy] : 0.0, ey = p.Ey ? p.Ey[gxy] : 0.0;
    const double u = p.coord[2][g[2]], v = p.coord[3][g[3]];
    const double a[4] = {u, v, -ex - p.omega_c * v, -ey + p.omega_c * u};
    double rhs = 0.0;
    for (int d = 0; d < 4; ++d) {
      const int n = p.n[d], N = p.N[d];
      const int e = g[d] / n, j = g[d] - e * n;
      const long long base = idx - (long long)j * strd[d];
      const double* U = p.ups[d] + j * n;
      double vol = 0.0;
      for (int k = 0; k < n; ++k) vol = fma(U[k], p.f[base + k * strd[d]], vol);
      double uL = 0.0, uR = 0.0;
      if (a[d] > 0.0) {
        uR = p.f[base + (long long)(n - 1) * strd[d]];
        if (e > 0) uL = p.f[base - strd[d]];
        else if (p.bc[d] == 0) uL = p.f[base + ((long long)(N - 1) * n + (n - 1)) * strd[d]];
        else if (p.bc[d] == 2) uL = p.xhalo[idx - (long long)g[0] * strd[0]];                   // x-slab: the left neighbour's last plane
      } else if (a[d] < 0.0) {
        uL = p.f[base];
        if (e < N - 1) uR = p.f[base + (long long)n * strd[d]];
        else if (p.bc[d] == 0) uR = p.f[base - (long long)e * n * strd[d]];
        else if (p.bc[d] == 2) uR = p.xhalo[strd[0] + idx - (long long)g[0] * strd[0]];         // the right neighbour's first plane
      }
      rhs += (p.J[d] * a[d]) * (vol - p.lift[d][2 * j + 1] * uR + p.lift[d][2 * j] * uL);
    }
    if (p.mode == 0) p.out[idx] = rhs;
    else p.out[idx] = (p.fn ? p.c0 * p.fn[idx] : 0.0) + p.c1 * (p.f[idx] + p.dt * rhs);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Field solve in two dimensions: separable passes, all tiny (G_x G_y densities, (P+1)(2Q+1) modes).
// T rows: T[(2p+c)*G + g], c = 0 real / 1 imaginary part of Eq. 63.  Waves: W[(p*G + g)*2 + c] = e^{i k_p x_g}.
// ---------------------------------------------------------------------------------------------------------------

// A[p][gy] = sum_gx T^x_p[gx] rho[gx][gy].  grid (ceil(G1/32), P+1), 256 threads = 32 g_y x 8 slices of g_x; the slices
// are summed in a fixed order (deterministic).
__global__ void __launch_bounds__(256) proj_x_kernel(const double* __restrict__ Tx, const double* __restrict__ rho, int G0, int G1,
                                                      double* __restrict__ A) {
  __shared__ double red[2][8][32];
  const int gl = threadIdx.x & 31, sl = threadIdx.x >> 5;
  const int gy = blockIdx.x * 32 + gl, p = blockIdx.y;
  const double* tr = Tx + (size_t)(2 * p) * G0;
  const double* ti = tr + G0;
  double are = 0.0, aim = 0.0;
  if (gy < G1) {
    for (int gx = sl; gx < G0; gx += 8) {
      const double r = rho[(size_t)gx * G1 + gy];
      are = fma(tr[gx], r, are);
      aim = fma(ti[gx], r, aim);
    }
  }
  red[0][sl][gl] = are; red[1][sl][gl] = aim;
  __syncthreads();
  if (threadIdx.x < 64) {
    const int c = threadIdx.x >> 5;
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) v += red[c][k][gl];
    if (gy < G1) A[((size_t)p * G1 + gy) * 2 + c] = v;
  }
}

// c[p][q'] = sum_gy T^y_q[gy] A[p][gy], q = q' - Q (T_{-q} = conj T_q), and the Poisson factors of Eq. 68/71:
// Et[0|1][p][q'] = i (k_p | k_q) c / (k_p^2 + k_q^2), zero at (0,0).  One warp per (p, q').
__global__ void __launch_bounds__(128) proj_y_poisson_kernel(const double* __restrict__ Ty, const double* __restrict__ A, int G1, int P1,
                                                              int Q, double kx1, double ky1, double* __restrict__ c,
                                                              double* __restrict__ Et) {
  const int NQ = 2 * Q + 1;
  const int w = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (w >= P1 * NQ) return;
  const int p = w / NQ, qi = w - p * NQ, q = qi - Q, qa = q < 0 ? -q : q;
  const double sgn = q < 0 ? -1.0 : 1.0;
  const double* tr = Ty + (size_t)(2 * qa) * G1;
  const double* ti = tr + G1;
  double cre = 0.0, cim = 0.0;
  for (int gy = lane; gy < G1; gy += 32) {
    const double ar = A[((size_t)p * G1 + gy) * 2], ai = A[((size_t)p * G1 + gy) * 2 + 1];
    const double yr = tr[gy], yi = sgn * ti[gy];
    cre += yr * ar - yi * ai;
    cim += yr * ai + yi * ar;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    cre += __shfl_down_sync(0xffffffffu, cre, off);
    cim += __shfl_down_sync(0xffffffffu, cim, off);
  }
  if (lane == 0) {
    if (c) { c[(size_t)w * 2] = cre; c[(size_t)w * 2 + 1] = cim; }
    if (Et) {
      const double kp = kx1 * p, kq = ky1 * q;
      const double k2 = kp * kp + kq * kq;
      const double fx = (p == 0 && q == 0) ? 0.0 : kp / k2, fy = (p == 0 && q == 0) ? 0.0 : kq / k2;
      const size_t half = (size_t)P1 * NQ * 2;
      Et[(size_t)w * 2] = -fx * cim;          // i * fx * (cre + i cim)
      Et[(size_t)w * 2 + 1] = fx * cre;
      Et[half + (size_t)w * 2] = -fy * cim;
      Et[half + (size_t)w * 2 + 1] = fy * cre;
    }
  }
}

// B[s][p][gy] = sum_q' Et[s][p][q'] e^{i k_q y_gy}.  grid (ceil(G1/32), P1, 2), 256 threads = 32 g_y x 8 slices of q'.
__global__ void __launch_bounds__(256) synth_y_kernel(const double* __restrict__ Et, const double* __restrict__ Wy, int G1, int P1, int Q,
                                                       double* __restrict__ B) {
  __shared__ double red[2][8][32];
  const int gl = threadIdx.x & 31, sl = threadIdx.x >> 5;
  const int gy = blockIdx.x * 32 + gl, p = blockIdx.y, s = blockIdx.z;
  const int NQ = 2 * Q + 1;
  const double* e = Et + ((size_t)s * P1 + p) * NQ * 2;
  double bre = 0.0, bim = 0.0;
  if (gy < G1) {
    for (int qi = sl; qi < NQ; qi += 8) {
      const int q = qi - Q, qa = q < 0 ? -q : q;
      const double wr = Wy[((size_t)qa * G1 + gy) * 2], wi = (q < 0 ? -1.0 : 1.0) * Wy[((size_t)qa * G1 + gy) * 2 + 1];
      bre += e[2 * qi] * wr - e[2 * qi + 1] * wi;
      bim += e[2 * qi] * wi + e[2 * qi + 1] * wr;
    }
  }
  red[0][sl][gl] = bre; red[1][sl][gl] = bim;
  __syncthreads();
  if (threadIdx.x < 64) {
    const int c = threadIdx.x >> 5;
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) v += red[c][k][gl];
    if (gy < G1) B[(((size_t)s * P1 + p) * G1 + gy) * 2 + c] = v;
  }
}

// E_s[gx][gy] = Re B[s][0][gy] + 2 Re sum_{p>=1} B[s][p][gy] e^{i k_p x_gx}.  grid (ceil(G1/32), G0, 2), 128 threads =
// 32 g_y x 4 slices of p.
__global__ void __launch_bounds__(128) synth_x_kernel(const double* __restrict__ B, const double* __restrict__ Wx, int G0, int G1, int P1,
                                                       double* __restrict__ Ex, double* __restrict__ Ey) {
  __shared__ double red[4][32];
  const int gl = threadIdx.x & 31, sl = threadIdx.x >> 5;
  const int gy = blockIdx.x * 32 + gl, gx = blockIdx.y, s = blockIdx.z;
  double acc = 0.0;
  if (gy < G1) {
    for (int p = 1 + sl; p < P1; p += 4) {
      const double br = B[(((size_t)s * P1 + p) * G1 + gy) * 2], bi = B[(((size_t)s * P1 + p) * G1 + gy) * 2 + 1];
      acc += br * Wx[((size_t)p * G0 + gx) * 2] - bi * Wx[((size_t)p * G0 + gx) * 2 + 1];
    }
  }
  red[sl][gl] = acc;
  __syncthreads();
  if (threadIdx.x < 32 && gy < G1) {
    const double v = B[(((size_t)s * P1) * G1 + gy) * 2] + 2.0 * (((red[0][gl] + red[1][gl]) + red[2][gl]) + red[3][gl]);
    (s == 0 ? Ex : Ey)[(size_t)gx * G1 + gy] = v;
  }
}

}  // namespace dg4
