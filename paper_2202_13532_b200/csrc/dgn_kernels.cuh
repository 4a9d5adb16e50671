// Dimension-generic kernels (include/dgvlasov_nd.h): phase space (x_1..x_dx, v_1..v_dv), 1 <= dx <= dv <= 3.
// One thread per node for the RHS, one CTA per space node for the density, and a field solve made of one complex
// "contract along an axis" kernel applied once per space dimension each way.  The general path and on-device cross-check of
// the tiled kernels; sized for correctness on any shape, not for the HBM roofline.
#pragma once
#include <cuda_runtime.h>

namespace dgn {

constexpr int MAXD = 6;

struct Params {
  int ndim, dx, dv;
  int N[MAXD], n[MAXD], G[MAXD], bc[MAXD];
  double J[MAXD];
  const double* coord[MAXD];   // node coordinates per dimension
  const double* ups[MAXD];     // reference Upsilon [n][n]   (Eq. 53)
  const double* lift[MAXD];    // reference Xi [n][2]        (Eq. 54)
  double omega_c;
  const double* E;             // [dx][GX] or nullptr
  long long GX, GV;            // nodes of the space / velocity sub-grids
  const double* f;
  const double* fn;            // or nullptr
  double* out;
  double c0, c1, dt;           // mode 1: out = c0*fn + c1*(f + dt*rhs);  mode 0: out = rhs
  int mode;
  long long dof;
};

// Weak form Eq. 14 reduced by Eq. 20-21, upwind flux Eq. 23, speeds Eq. 28 in dx + dv
// dimensions: a_{x_i} = v_i, a_{v_1} = -E_1 - omega_c v_2, a_{v_2} = -E_2 + omega_c v_1, a_{v_3} = -E_3.
__global__ void __launch_bounds__(256) rhs_nd_kernel(const Params p) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  long long strd[MAXD];
  strd[p.ndim - 1] = 1;
  for (int d = p.ndim - 2; d >= 0; --d) strd[d] = strd[d + 1] * p.G[d + 1];
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < p.dof; idx += stride) {
    int g[MAXD];
    long long r = idx;
    for (int d = p.ndim - 1; d >= 0; --d) { g[d] = (int)(r % p.G[d]); r /= p.G[d]; }
    const long long gx = idx / p.GV;                       // flat index of the space node
    double v[3] = {0.0, 0.0, 0.0}, e[3] = {0.0, 0.0, 0.0};
    for (int i = 0; i < p.dv; ++i) v[i] = p.coord[p.dx + i][g[p.dx + i]];
    if (p.E) for (int i = 0; i < p.dx; ++i) e[i] = p.E[(long long)i * p.GX + gx];
    double a[MAXD];
    for (int i = 0; i < p.dx; ++i) a[i] = v[i];
    a[p.dx] = -e[0] - (p.dv >= 2 ? p.omega_c * v[1] : 0.0);
    if (p.dv >= 2) a[p.dx + 1] = -e[1] + p.omega_c * v[0];
    if (p.dv >= 3) a[p.dx + 2] = -e[2];
    double rhs = 0.0;
    for (int d = 0; d < p.ndim; ++d) {
      const int n = p.n[d], N = p.N[d];
      const int el = g[d] / n, j = g[d] - el * n;
      const long long base = idx - (long long)j * strd[d];
      const double* U = p.ups[d] + j * n;
      double vol = 0.0;
      for (int k = 0; k < n; ++k) vol = fma(U[k], p.f[base + k * strd[d]], vol);
      double uL = 0.0, uR = 0.0;
      if (a[d] > 0.0) {
        uR = p.f[base + (long long)(n - 1) * strd[d]];
        if (el > 0) uL = p.f[base - strd[d]];
        else if (p.bc[d] == 0) uL = p.f[base + ((long long)(N - 1) * n + (n - 1)) * strd[d]];
      } else if (a[d] < 0.0) {
        uL = p.f[base];
        if (el < N - 1) uR = p.f[base + (long long)n * strd[d]];
        else if (p.bc[d] == 0) uR = p.f[base - (long long)el * n * strd[d]];
      }
      rhs += (p.J[d] * a[d]) * (vol - p.lift[d][2 * j + 1] * uR + p.lift[d][2 * j] * uL);
    }
    if (p.mode == 0) p.out[idx] = rhs;
    else p.out[idx] = (p.fn ? p.c0 * p.fn[idx] : 0.0) + p.c1 * (p.f[idx] + p.dt * rhs);
  }
}

// rho[gx] = sum over the velocity nodes of prod_i wq_i[g_vi] f  (Eq. 27).  One CTA per space node (grid-stride), each thread
// a fixed subset of the velocity nodes in index order, then a fixed-order tree over the 256 partial sums: deterministic.
__global__ void __launch_bounds__(256) density_nd_kernel(const double* __restrict__ f, const double* __restrict__ wq0,
                                                          const double* __restrict__ wq1, const double* __restrict__ wq2, int dv,
                                                          int Gv0, int Gv1, int Gv2, long long GX, long long GV,
                                                          double* __restrict__ rho) {
  __shared__ double red[256];
  for (long long gx = blockIdx.x; gx < GX; gx += gridDim.x) {
    const double* row = f + gx * GV;
    double s = 0.0;
    for (long long j = threadIdx.x; j < GV; j += 256) {
      long long r = j;
      double w = 1.0;
      if (dv >= 3) { w *= wq2[r % Gv2]; r /= Gv2; }
      if (dv >= 2) { w *= wq1[r % Gv1]; r /= Gv1; }
      w *= wq0[r];
      s = fma(w, row[j], s);
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int off = 128; off > 0; off >>= 1) {
      if (threadIdx.x < off) red[threadIdx.x] += red[threadIdx.x + off];
      __syncthreads();
    }
    if (threadIdx.x == 0) rho[gx] = red[0];
    __syncthreads();
  }
}

// out[pre][m][post] = sum_g M[m][g] in[pre][g][post]: one contraction along one axis of a complex array (in_real: the input
// holds doubles, imaginary part 0).  M: [rows][cols] complex.  One thread per output element, the sum in index order.
__global__ void __launch_bounds__(256) apply_axis_kernel(const double2* __restrict__ M, const void* __restrict__ in, int in_real,
                                                          double2* __restrict__ out, long long pre, int rows, int cols, long long post) {
  const long long total = pre * rows * post;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (long long)gridDim.x * blockDim.x) {
    const long long po = o % post, t = o / post;
    const int m = (int)(t % rows);
    const long long pr = t / rows;
    const double2* Mr = M + (long long)m * cols;
    double re = 0.0, im = 0.0;
    if (in_real) {
      const double* src = reinterpret_cast<const double*>(in) + pr * cols * post + po;
      for (int g = 0; g < cols; ++g) {
        const double x = src[(long long)g * post];
        re = fma(Mr[g].x, x, re);
        im = fma(Mr[g].y, x, im);
      }
    } else {
      const double2* src = reinterpret_cast<const double2*>(in) + pr * cols * post + po;
      for (int g = 0; g < cols; ++g) {
        const double2 x = src[(long long)g * post];
        re += Mr[g].x * x.x - Mr[g].y * x.y;
        im += Mr[g].x * x.y + Mr[g].y * x.x;
      }
    }
    out[o] = make_double2(re, im);
  }
}

// Poisson factors of Eq. 68 / 71 on the mode lattice c[m_0][m_1][m_2] (p_0 = m_0 >= 0, p_i = m_i - P_i for i > 0):
// Et[i][mode] = i k_i c / |k|^2 (E = -grad Phi, Phi_p = -c_p / k^2), zero at p = 0 (reading C5).
__global__ void __launch_bounds__(256) poisson_nd_kernel(const double2* __restrict__ c, int dx, int M0, int M1, int M2, int P1, int P2,
                                                          double k0, double k1, double k2, double2* __restrict__ Et) {
  const long long total = (long long)M0 * M1 * M2;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (long long)gridDim.x * blockDim.x) {
    const int m2 = (int)(o % M2), m1 = (int)((o / M2) % M1), m0 = (int)(o / ((long long)M2 * M1));
    const double kk[3] = {k0 * m0, dx >= 2 ? k1 * (m1 - P1) : 0.0, dx >= 3 ? k2 * (m2 - P2) : 0.0};
    const double q = kk[0] * kk[0] + kk[1] * kk[1] + kk[2] * kk[2];
    const double2 cv = c[o];
    for (int i = 0; i < dx; ++i) {
      const double fac = q > 0.0 ? kk[i] / q : 0.0;
      Et[(long long)i * total + o] = make_double2(-fac * cv.y, fac * cv.x);          // i * fac * (re + i im)
    }
  }
}

// E[g0][post] = Re B[0][post] + 2 Re sum_{p >= 1} B[p][post] e^{i k_p x_g0}: the last synthesis step of Eq. 71 (the kept
// half-space p_0 >= 0; the plane p_0 = 0 holds both signs of the other mode numbers and is real by itself).
// W0: [G0][M0] complex = e^{i k_p x_g}.
__global__ void __launch_bounds__(256) synth0_kernel(const double2* __restrict__ W0, const double2* __restrict__ B, int G0, int M0,
                                                      long long post, double* __restrict__ E) {
  const long long total = (long long)G0 * post;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (long long)gridDim.x * blockDim.x) {
    const long long po = o % post;
    const int g = (int)(o / post);
    const double2* w = W0 + (long long)g * M0;
    double acc = 0.0;
    for (int p = 1; p < M0; ++p) {
      const double2 b = B[(long long)p * post + po];
      acc += b.x * w[p].x - b.y * w[p].y;
    }
    E[o] = B[po].x + 2.0 * acc;
  }
}

}  // namespace dgn
