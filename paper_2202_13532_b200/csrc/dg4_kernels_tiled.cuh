// 2D2V tiled RHS + stage kernel for n = 4 LGL nodes in all four dimensions (sm_100a).
//
// Tile = one (x, y, u) element x KV v-elements = 4 x 4 x 4 x (4 KV) nodes: 64 rows of R = 4 KV contiguous doubles
// (KV = 8: 256-byte rows, 16 KB).  One CTA of 16 KV threads per tile; shared memory holds the f_s tile and a tile of partial
// sums (2 x 16 KB), so 7 CTAs are resident per SM and the loads of one overlap the arithmetic of the others.
//   fill    cp.async (16 bytes per request, L2 only) of the 64 rows, chunk-swizzled so that both phases below are
//           bank-conflict free; the upwind x / y face values of phase A are fetched into registers meanwhile.
//   phase A thread = (u node, v node of the tile) owns the 4 x 4 (x, y) nodes above it: x and y contractions + lifts in
//           registers (the speeds a_x = u, a_y = v are per-thread constants), partial sums to shared memory.
//   phase B thread = (x node, y node, v element) owns the 4 x 4 (u, v) nodes of that element: u and v contractions + lifts;
//           v-face neighbours inside the tile come from the adjacent lanes by warp shuffle, the two tile-edge faces and the
//           u faces from global memory (L2: the neighbouring tiles are a few CTAs away); stage combination, 128-bit stores;
//           LGL-weighted sum of the 16 outputs, reduced over the KV lanes -> one density partial per (g_x, g_y, tile).
// f is read once and written once per stage from HBM; every operator coefficient is a kernel-parameter constant.
#pragma once
#include "dg4_kernels.cuh"

namespace dg4 {

template <int KV>
__device__ __forceinline__ int swz(int row, int chunk) {      // 16-byte chunk position inside a row
  if (KV == 8) return chunk ^ ((chunk >> 3) & 1);
  if (KV == 4) return chunk ^ ((row >> 2) & 1);
  return chunk;
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}

// Tile rasterisation.  Row-major (v fastest, x slowest) puts a whole x-element slab (G_y G_u G_v n doubles) between a tile
// and its x neighbour -- more than the L2 holds on large grids, so every x-face value would come from HBM a second time.
// Blocked: x elements in groups of BX, inside a group (y, u, x, v-block) row-major -> the x neighbour is N_v/KV tiles away,
// the y neighbour N_u BX N_v/KV tiles.
__device__ __forceinline__ void decode_tile(const Params& p, int nvb, long long t, int& ex, int& ey, int& eu, int& evb) {
  if (p.order_mode <= 1) {
    evb = (int)(t % nvb); t /= nvb;
    eu = (int)(t % p.N[2]); t /= p.N[2];
    ey = (int)(t % p.N[1]); t /= p.N[1];
    ex = (int)t;
  } else {
    const int BX = p.order_mode;
    const long long per_group = (long long)p.N[1] * p.N[2] * BX * nvb;
    const int xb = (int)(t / per_group);
    t -= xb * per_group;
    const int bx = min(BX, p.N[0] - xb * BX);          // the last group may be narrower
    evb = (int)(t % nvb); t /= nvb;
    const int xi = (int)(t % bx); t /= bx;
    eu = (int)(t % p.N[2]); t /= p.N[2];
    ey = (int)t;
    ex = xb * BX + xi;
  }
}

template <int KV>
__global__ void __launch_bounds__(16 * KV) rhs4_tile_kernel(const Params p) {
  constexpr int R = 4 * KV, ROWS = 64, NT = 16 * KV, HC = R / 2;
  extern __shared__ double2 smem_raw[];
  double* tile = reinterpret_cast<double*>(smem_raw);
  double* accT = tile + ROWS * R;
  const int nvb = p.N[3] / KV;
  int ex, ey, eu, evb;
  decode_tile(p, nvb, blockIdx.x, ex, ey, eu, evb);
  const int gx0 = ex * 4, gy0 = ey * 4, gu0 = eu * 4, gv0 = evb * R;
  const long long s2 = p.G[3], s1 = s2 * p.G[2], s0 = s1 * p.G[1];
  const int tid = threadIdx.x;

  // ---- fill -------------------------------------------------------------------------------------------------------
#pragma unroll
  for (int t = tid; t < ROWS * HC; t += NT) {
    const int row = t / HC, ch = t % HC;
    const int jx = row >> 4, jy = (row >> 2) & 3, ju = row & 3;
    const double* src = p.f + (gx0 + jx) * s0 + (gy0 + jy) * s1 + (gu0 + ju) * s2 + gv0 + 2 * ch;
    cp_async16(tile + row * R + swz<KV>(row, ch) * 2, src);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");

  // ---- phase A: upwind x / y face values while the tile is in flight -----------------------------------------------
  const int ju_a = tid / R, rv = tid % R;
  const double ax = p.coord[2][gu0 + ju_a], ay = p.coord[3][gv0 + rv];
  double hX[4] = {0.0, 0.0, 0.0, 0.0}, hY[4] = {0.0, 0.0, 0.0, 0.0};
  {
    const long long uv = (long long)(gu0 + ju_a) * s2 + gv0 + rv;
    int hx = -1, hy = -1;
    if (ax > 0.0) hx = ex > 0 ? gx0 - 1 : (p.bc[0] == 0 ? p.G[0] - 1 : -1);
    else if (ax < 0.0) hx = ex < p.N[0] - 1 ? gx0 + 4 : (p.bc[0] == 0 ? 0 : -1);
    if (ay > 0.0) hy = ey > 0 ? gy0 - 1 : (p.bc[1] == 0 ? p.G[1] - 1 : -1);
    else if (ay < 0.0) hy = ey < p.N[1] - 1 ? gy0 + 4 : (p.bc[1] == 0 ? 0 : -1);
    if (hx >= 0) {
#pragma unroll
      for (int jy = 0; jy < 4; ++jy) hX[jy] = __ldg(p.f + hx * s0 + (gy0 + jy) * s1 + uv);
    }
    if (hy >= 0) {
#pragma unroll
      for (int jx = 0; jx < 4; ++jx) hY[jx] = __ldg(p.f + (gx0 + jx) * s0 + hy * s1 + uv);
    }
  }
  asm volatile("cp.async.wait_all;" ::: "memory");
  __syncthreads();

  {
    double fa[4][4], acc[4][4];
    const int col = rv;
#pragma unroll
    for (int jx = 0; jx < 4; ++jx)
#pragma unroll
      for (int jy = 0; jy < 4; ++jy) {
        const int row = (jx * 4 + jy) * 4 + ju_a;
        fa[jx][jy] = tile[row * R + swz<KV>(row, col >> 1) * 2 + (col & 1)];
      }
    const double sx = p.J[0] * ax, sy = p.J[1] * ay;
#pragma unroll
    for (int jy = 0; jy < 4; ++jy) {
      const double uL = ax > 0.0 ? hX[jy] : fa[0][jy], uR = ax > 0.0 ? fa[3][jy] : hX[jy];
#pragma unroll
      for (int jx = 0; jx < 4; ++jx) {
        double v = p.Xi[2 * jx] * uL;
        v = fma(-p.Xi[2 * jx + 1], uR, v);
#pragma unroll
        for (int k = 0; k < 4; ++k) v = fma(p.U[jx * 4 + k], fa[k][jy], v);
        acc[jx][jy] = sx * v;
      }
    }
#pragma unroll
    for (int jx = 0; jx < 4; ++jx) {
      const double uL = ay > 0.0 ? hY[jx] : fa[jx][0], uR = ay > 0.0 ? fa[jx][3] : hY[jx];
#pragma unroll
      for (int jy = 0; jy < 4; ++jy) {
        double v = p.Xi[2 * jy] * uL;
        v = fma(-p.Xi[2 * jy + 1], uR, v);
#pragma unroll
        for (int k = 0; k < 4; ++k) v = fma(p.U[jy * 4 + k], fa[jx][k], v);
        acc[jx][jy] = fma(sy, v, acc[jx][jy]);
      }
    }
#pragma unroll
    for (int jx = 0; jx < 4; ++jx)
#pragma unroll
      for (int jy = 0; jy < 4; ++jy) {
        const int row = (jx * 4 + jy) * 4 + ju_a;
        accT[row * R + swz<KV>(row, col >> 1) * 2 + (col & 1)] = acc[jx][jy];
      }
  }

  // ---- phase B ----------------------------------------------------------------------------------------------------
  const int ev = tid % KV, jy_b = (tid / KV) & 3, jx_b = tid / (4 * KV);
  const int gx = gx0 + jx_b, gy = gy0 + jy_b;
  const long long xy = gx * s0 + gy * s1;
  const long long gxy = (long long)gx * p.G[1] + gy;
  const double exf = p.Ex ? __ldg(p.Ex + gxy) : 0.0, eyf = p.Ey ? __ldg(p.Ey + gxy) : 0.0;
  const int gvb = gv0 + ev * 4;                                   // first v node of this thread's element
  double au[4], av[4];
  {
    const double2 v01 = *reinterpret_cast<const double2*>(p.coord[3] + gvb), v23 = *reinterpret_cast<const double2*>(p.coord[3] + gvb + 2);
    const double2 u01 = *reinterpret_cast<const double2*>(p.coord[2] + gu0), u23 = *reinterpret_cast<const double2*>(p.coord[2] + gu0 + 2);
    au[0] = -exf - p.omega_c * v01.x; au[1] = -exf - p.omega_c * v01.y; au[2] = -exf - p.omega_c * v23.x; au[3] = -exf - p.omega_c * v23.y;
    av[0] = -eyf + p.omega_c * u01.x; av[1] = -eyf + p.omega_c * u01.y; av[2] = -eyf + p.omega_c * u23.x; av[3] = -eyf + p.omega_c * u23.y;
  }
  // u faces: the row below / above the tile, the four v nodes of this element
  double hUlo[4] = {0.0, 0.0, 0.0, 0.0}, hUhi[4] = {0.0, 0.0, 0.0, 0.0};
  {
    const int lo = eu > 0 ? gu0 - 1 : (p.bc[2] == 0 ? p.G[2] - 1 : -1);
    const int hi = eu < p.N[2] - 1 ? gu0 + 4 : (p.bc[2] == 0 ? 0 : -1);
    const bool pos = au[0] > 0.0 || au[1] > 0.0 || au[2] > 0.0 || au[3] > 0.0;
    const bool neg = au[0] < 0.0 || au[1] < 0.0 || au[2] < 0.0 || au[3] < 0.0;
    if (lo >= 0 && pos) {
      const double2* q = reinterpret_cast<const double2*>(p.f + xy + lo * s2 + gvb);
      const double2 a = __ldg(q), b = __ldg(q + 1);
      hUlo[0] = a.x; hUlo[1] = a.y; hUlo[2] = b.x; hUlo[3] = b.y;
    }
    if (hi >= 0 && neg) {
      const double2* q = reinterpret_cast<const double2*>(p.f + xy + hi * s2 + gvb);
      const double2 a = __ldg(q), b = __ldg(q + 1);
      hUhi[0] = a.x; hUhi[1] = a.y; hUhi[2] = b.x; hUhi[3] = b.y;
    }
  }
  // v faces at the two tile edges (lanes ev = 0 and ev = KV-1 only)
  double eVlo[4] = {0.0, 0.0, 0.0, 0.0}, eVhi[4] = {0.0, 0.0, 0.0, 0.0};
  if (ev == 0) {
    const int lo = evb > 0 ? gv0 - 1 : (p.bc[3] == 0 ? p.G[3] - 1 : -1);
    if (lo >= 0) {
#pragma unroll
      for (int ju = 0; ju < 4; ++ju) if (av[ju] > 0.0) eVlo[ju] = __ldg(p.f + xy + (gu0 + ju) * s2 + lo);
    }
  }
  if (ev == KV - 1) {
    const int hi = evb < nvb - 1 ? gv0 + R : (p.bc[3] == 0 ? 0 : -1);
    if (hi >= 0) {
#pragma unroll
      for (int ju = 0; ju < 4; ++ju) if (av[ju] < 0.0) eVhi[ju] = __ldg(p.f + xy + (gu0 + ju) * s2 + hi);
    }
  }
  // step input of the stage combination
  double fnv[4][4];
  const bool use_fn = p.mode != 0 && p.fn != nullptr;
  if (use_fn) {
#pragma unroll
    for (int ju = 0; ju < 4; ++ju) {
      const double2* q = reinterpret_cast<const double2*>(p.fn + xy + (gu0 + ju) * s2 + gvb);
      const double2 a = __ldcs(q), b = __ldcs(q + 1);
      fnv[ju][0] = a.x; fnv[ju][1] = a.y; fnv[ju][2] = b.x; fnv[ju][3] = b.y;
    }
  }
  __syncthreads();

  double fb[4][4], res[4][4];
  const int rowb = (jx_b * 4 + jy_b) * 4;
#pragma unroll
  for (int ju = 0; ju < 4; ++ju) {
    const int row = rowb + ju;
    const double2 a = *reinterpret_cast<const double2*>(tile + row * R + swz<KV>(row, 2 * ev) * 2);
    const double2 b = *reinterpret_cast<const double2*>(tile + row * R + swz<KV>(row, 2 * ev + 1) * 2);
    fb[ju][0] = a.x; fb[ju][1] = a.y; fb[ju][2] = b.x; fb[ju][3] = b.y;
    const double2 c = *reinterpret_cast<const double2*>(accT + row * R + swz<KV>(row, 2 * ev) * 2);
    const double2 d = *reinterpret_cast<const double2*>(accT + row * R + swz<KV>(row, 2 * ev + 1) * 2);
    res[ju][0] = c.x; res[ju][1] = c.y; res[ju][2] = d.x; res[ju][3] = d.y;
  }
  // u lines (fixed jv)
#pragma unroll
  for (int jv = 0; jv < 4; ++jv) {
    const double uL = au[jv] > 0.0 ? hUlo[jv] : fb[0][jv], uR = au[jv] > 0.0 ? fb[3][jv] : hUhi[jv];
    const double su = p.J[2] * au[jv];
#pragma unroll
    for (int ju = 0; ju < 4; ++ju) {
      double v = p.Xi[2 * ju] * uL;
      v = fma(-p.Xi[2 * ju + 1], uR, v);
#pragma unroll
      for (int k = 0; k < 4; ++k) v = fma(p.U[ju * 4 + k], fb[k][jv], v);
      res[ju][jv] = fma(su, v, res[ju][jv]);
    }
  }
  // v lines (fixed ju): neighbours inside the tile from the adjacent lanes
#pragma unroll
  for (int ju = 0; ju < 4; ++ju) {
    const double from_lo = __shfl_up_sync(0xffffffffu, fb[ju][3], 1), from_hi = __shfl_down_sync(0xffffffffu, fb[ju][0], 1);
    const double nlo = ev > 0 ? from_lo : eVlo[ju], nhi = ev < KV - 1 ? from_hi : eVhi[ju];
    const double uL = av[ju] > 0.0 ? nlo : fb[ju][0], uR = av[ju] > 0.0 ? fb[ju][3] : nhi;
    const double sv = p.J[3] * av[ju];
#pragma unroll
    for (int jv = 0; jv < 4; ++jv) {
      double v = p.Xi[2 * jv] * uL;
      v = fma(-p.Xi[2 * jv + 1], uR, v);
#pragma unroll
      for (int k = 0; k < 4; ++k) v = fma(p.U[jv * 4 + k], fb[ju][k], v);
      res[ju][jv] = fma(sv, v, res[ju][jv]);
    }
  }
  // stage combination, stores, density partial
  double dens = 0.0;
#pragma unroll
  for (int ju = 0; ju < 4; ++ju) {
    double o[4];
#pragma unroll
    for (int jv = 0; jv < 4; ++jv) {
      if (p.mode == 0) o[jv] = res[ju][jv];
      else {
        const double v = fma(p.dt, res[ju][jv], fb[ju][jv]);
        o[jv] = use_fn ? fma(p.c1, v, p.c0 * fnv[ju][jv]) : p.c1 * v;
      }
    }
    double2* q = reinterpret_cast<double2*>(p.out + xy + (gu0 + ju) * s2 + gvb);
    __stcs(q, make_double2(o[0], o[1]));
    __stcs(q + 1, make_double2(o[2], o[3]));
    if (p.partials) {
      const double2 w01 = *reinterpret_cast<const double2*>(p.wqv + gvb), w23 = *reinterpret_cast<const double2*>(p.wqv + gvb + 2);
      const double rowsum = fma(w01.x, o[0], fma(w01.y, o[1], fma(w23.x, o[2], w23.y * o[3])));
      dens = fma(p.wqu[gu0 + ju], rowsum, dens);
    }
  }
  if (p.partials) {
#pragma unroll
    for (int off = KV / 2; off > 0; off >>= 1) dens += __shfl_xor_sync(0xffffffffu, dens, off);
    if (ev == 0) p.partials[gxy * p.chunks + eu * nvb + evb] = dens;
  }
}

}  // namespace dg4
