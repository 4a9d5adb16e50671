// 2D2V tiled RHS + stage kernel for n = 4 LGL nodes in all four dimensions (sm_100a).
//
// Tile = one (x, y, u) element x KV v-elements = 4 x 4 x 4 x (4 KV) nodes: 64 rows of R = 4 KV contiguous doubles
// (KV = 8: 256-byte rows, 16 KB).  One CTA of 16 KV threads per tile.
//   fill    every global read of the CTA is issued at the top of the kernel, all but four scalars as cp.async into shared
//           memory -- the f_s tile and the f_n tile (16 bytes per request, chunk-swizzled so that both phases below are
//           bank-conflict free), the upwind x / y face values of phase A and the upwind u face values of phase B (8 bytes per
//           request, only the side the sign of the speed selects) -- followed by ONE wait: a CTA pays the memory latency
//           once.  The running sums of phase A replace f_n in its tile (c0 f_n + c1 dt (x and y parts)), so a CTA holds 44 KB
//           and five CTAs (20 warps, 96 registers per thread) share an SM.
//   phase A thread = (u node, v node of the tile) owns the 4 x 4 (x, y) nodes above it: x and y contractions + lifts in
//           registers (the speeds a_x = u, a_y = v are per-thread constants), partial sums to shared memory.
//   phase B thread = (x node, y node, v element) owns the 4 x 4 (u, v) nodes of that element: u and v contractions + lifts;
//           v-face neighbours inside the tile come from the adjacent lanes by warp shuffle; stage combination, 128-bit
//           stores; LGL-weighted sum of the 16 outputs, reduced over the KV lanes -> one density partial per
//           (g_x, g_y, tile).
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

__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}

// 8-byte copy that reads `bytes` (8 or 0) from global memory and fills the rest with zeros: an absent neighbour (zero inflow,
// or a = 0: no flux) costs no branch
__device__ __forceinline__ void cp_async8_zfill(void* smem, const void* gmem, unsigned bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem), "r"(bytes) : "memory");
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}

// Shared memory (doubles): f_s tile 64 R | f_n tile, then the running sums, 64 R | x faces 4 NT | y faces 4 NT | u faces 4 NT
// (KV = 8: 44 KB, five CTAs per SM).
template <int KV>
constexpr int tile_smem_doubles(bool) { return 2 * 64 * 4 * KV + 12 * (16 * KV); }

template <int KV, int MINB>
__global__ void __launch_bounds__(16 * KV, MINB) rhs4_tile_kernel(const Params p) {
  constexpr int R = 4 * KV, ROWS = 64, NT = 16 * KV, HC = R / 2;
  extern __shared__ double2 smem_raw[];
  double* tile = reinterpret_cast<double*>(smem_raw);
  double* accT = tile + ROWS * R;
  double* hXs = accT + ROWS * R;          // [jy][tid]
  double* hYs = hXs + 4 * NT;             // [jx][tid]
  double* hUs = hYs + 4 * NT;             // [jv][tid]: the upwind u face of each of the thread's four u lines
  // grid = (N_v/KV * BX * N_u, N_y, N_x / BX), BX = 2^bx_log2 x-elements per group: consecutive CTAs walk v, then the x elements
  // of a group, then u -- the v, x and u neighbours of a tile are in flight with it and the y neighbour is N_u BX N_v/KV tiles
  // away (L2), where a row-major walk would put a whole x slab (G_y G_u G_v n doubles, more than the L2 on large grids)
  // between a tile and its x neighbour.
  const int nvb = p.N[3] / KV;
  const int bq = blockIdx.x / nvb, evb = blockIdx.x - bq * nvb;
  const int eu = bq >> p.bx_log2, ex = (blockIdx.z << p.bx_log2) + (bq & ((1 << p.bx_log2) - 1)), ey = blockIdx.y;
  const int gx0 = ex * 4, gy0 = ey * 4, gu0 = eu * 4, gv0 = evb * R;
  const long long s2 = p.G[3], s1 = s2 * p.G[2], s0 = s1 * p.G[1];
  const int tid = threadIdx.x;
  const bool use_fn = p.mode != 0 && p.fn != nullptr;
  // phase A / phase B coordinates of this thread
  const int ju_a = tid / R, rv = tid % R;
  const int ev = tid % KV, jy_b = (tid / KV) & 3, jx_b = tid / (4 * KV);
  const int gx = gx0 + jx_b, gy = gy0 + jy_b;
  const long long xy = gx * s0 + gy * s1;
  const long long gxy = (long long)gx * p.G[1] + gy;
  const int gvb = gv0 + ev * 4;                                   // first v node of this thread's element (phase B)
  const double ax = p.coord[2][gu0 + ju_a], ay = p.coord[3][gv0 + rv];

  // ---- all global reads, asynchronously ---------------------------------------------------------------------------
  // tile rows: pass i of the CTA covers rows r0 + 8 i (NT / HC = 8 rows per pass): jx = i / 2, jy = r0 / 4 + 2 (i % 2), ju = r0 % 4
  const long long tile_off = gx0 * s0 + gy0 * s1 + gu0 * s2 + gv0;
  const int r0 = tid / HC, ch = tid % HC;
  const long long fill_off = tile_off + (r0 >> 2) * s1 + (r0 & 3) * s2 + 2 * ch;
  const int fill_dst = r0 * R + swz<KV>(r0, ch) * 2;           // swz(r0 + 8 i, ch) = swz(r0, ch)
  {
    const double* src = p.f + fill_off;
#pragma unroll
    for (int jx = 0; jx < 4; ++jx) {
      cp_async16(tile + fill_dst + (16 * jx) * R, src);
      cp_async16(tile + fill_dst + (16 * jx + 8) * R, src + 2 * s1);
      src += s0;
    }
  }
  {
    // x and y faces of phase A: one value per (x or y) line of the thread, from the side the sign of the speed selects
    const long long uv = (long long)(gu0 + ju_a) * s2 + gv0 + rv;
    int hx = -1, hy = -1;
    if (ax > 0.0) hx = ex > 0 ? gx0 - 1 : (p.bc[0] == 0 ? p.G[0] - 1 : -1);
    else if (ax < 0.0) hx = ex < p.N[0] - 1 ? gx0 + 4 : (p.bc[0] == 0 ? 0 : -1);
    if (ay > 0.0) hy = ey > 0 ? gy0 - 1 : (p.bc[1] == 0 ? p.G[1] - 1 : -1);
    else if (ay < 0.0) hy = ey < p.N[1] - 1 ? gy0 + 4 : (p.bc[1] == 0 ? 0 : -1);
    const double* px = p.f + hx * s0 + gy0 * s1 + uv;
    if (p.bc[0] == 2) {        // x-slab: at the slab's two x faces the exterior planes come from the halo buffer
      if (ax > 0.0 && ex == 0) { hx = 0; px = p.xhalo + gy0 * s1 + uv; }
      else if (ax < 0.0 && ex == p.N[0] - 1) { hx = 0; px = p.xhalo + s0 + gy0 * s1 + uv; }
    }
    const double* py = p.f + gx0 * s0 + hy * s1 + uv;
    const unsigned nx = hx >= 0 ? 8u : 0u, ny = hy >= 0 ? 8u : 0u;
    if (hx < 0) px = p.f;          // nothing is read, the address only has to be valid
    if (hy < 0) py = p.f;
    const long long sx = hx >= 0 ? s1 : 0, sy = hy >= 0 ? s0 : 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      cp_async8_zfill(hXs + j * NT + tid, px, nx);
      cp_async8_zfill(hYs + j * NT + tid, py, ny);
      px += sx; py += sy;
    }
  }
  if (use_fn) {                                                   // f_n lands where the running sums will live
    const double* src = p.fn + fill_off;
#pragma unroll
    for (int jx = 0; jx < 4; ++jx) {
      cp_async16(accT + fill_dst + (16 * jx) * R, src);
      cp_async16(accT + fill_dst + (16 * jx + 8) * R, src + 2 * s1);
      src += s0;
    }
  }
  const double exf = p.Ex ? __ldg(p.Ex + gxy) : 0.0, eyf = p.Ey ? __ldg(p.Ey + gxy) : 0.0;
  double au[4], av[4];
  {
    const double2 v01 = *reinterpret_cast<const double2*>(p.coord[3] + gvb), v23 = *reinterpret_cast<const double2*>(p.coord[3] + gvb + 2);
    const double2 u01 = *reinterpret_cast<const double2*>(p.coord[2] + gu0), u23 = *reinterpret_cast<const double2*>(p.coord[2] + gu0 + 2);
    au[0] = -exf - p.omega_c * v01.x; au[1] = -exf - p.omega_c * v01.y; au[2] = -exf - p.omega_c * v23.x; au[3] = -exf - p.omega_c * v23.y;
    av[0] = -eyf + p.omega_c * u01.x; av[1] = -eyf + p.omega_c * u01.y; av[2] = -eyf + p.omega_c * u23.x; av[3] = -eyf + p.omega_c * u23.y;
  }
  {
    // u faces: one value per u line (fixed jv), from the row below or above the tile by the sign of a_u
    const int lo = eu > 0 ? gu0 - 1 : (p.bc[2] == 0 ? p.G[2] - 1 : -1);
    const int hi = eu < p.N[2] - 1 ? gu0 + 4 : (p.bc[2] == 0 ? 0 : -1);
    const double* blo = lo >= 0 ? p.f + xy + lo * s2 + gvb : p.f;
    const double* bhi = hi >= 0 ? p.f + xy + hi * s2 + gvb : p.f;
    const unsigned nlo = lo >= 0 ? 8u : 0u, nhi = hi >= 0 ? 8u : 0u;
#pragma unroll
    for (int jv = 0; jv < 4; ++jv) {
      const bool up = au[jv] > 0.0;
      const unsigned nb = up ? nlo : (au[jv] < 0.0 ? nhi : 0u);
      const double* src = up ? blo : bhi;
      cp_async8_zfill(hUs + jv * NT + tid, src + jv, nb);         // blo / bhi are valid addresses even when nothing is read
    }
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  // v faces at the two tile edges: lanes ev = 0 (a_v > 0) and ev = KV-1 (a_v < 0) only, one scalar per u row
  double eV[4] = {0.0, 0.0, 0.0, 0.0};
  {
    const int vlo = evb > 0 ? gv0 - 1 : (p.bc[3] == 0 ? p.G[3] - 1 : -1);
    const int vhi = evb < nvb - 1 ? gv0 + R : (p.bc[3] == 0 ? 0 : -1);
    // a lane sits on at most one tile edge (KV >= 2): its candidate neighbour column, and the sign of a_v that takes it
    const bool low = (ev == 0);
    const int gedge = low ? vlo : (ev == KV - 1 ? vhi : -1);
    const double* rowp = p.f + xy + gu0 * s2 + (gedge >= 0 ? gedge : 0);
#pragma unroll
    for (int ju = 0; ju < 4; ++ju) {
      const bool need = gedge >= 0 && (low ? av[ju] > 0.0 : av[ju] < 0.0);
      double v = 0.0;
      asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q ld.global.nc.f64 %0, [%1];\n}" : "+d"(v) : "l"(rowp + ju * s2), "r"((int)need) : "memory");
      eV[ju] = v;
    }
  }
  asm volatile("cp.async.wait_all;" ::: "memory");
  __syncthreads();

  // ---- phase A: x and y ---------------------------------------------------------------------------------------------
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
      const double h = hXs[jy * NT + tid];
      const double uL = ax > 0.0 ? h : fa[0][jy], uR = ax > 0.0 ? fa[3][jy] : h;
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
      const double h = hYs[jx * NT + tid];
      const double uL = ay > 0.0 ? h : fa[jx][0], uR = ay > 0.0 ? fa[jx][3] : h;
#pragma unroll
      for (int jy = 0; jy < 4; ++jy) {
        double v = p.Xi[2 * jy] * uL;
        v = fma(-p.Xi[2 * jy + 1], uR, v);
#pragma unroll
        for (int k = 0; k < 4; ++k) v = fma(p.U[jy * 4 + k], fa[jx][k], v);
        acc[jx][jy] = fma(sy, v, acc[jx][jy]);
      }
    }
    // running sum: the x and y parts of the stage result, c0 f_n + c1 dt (.) (mode 0: the plain sums), in place of f_n
    const double cs = p.mode == 0 ? 1.0 : p.c1 * p.dt;
#pragma unroll
    for (int jx = 0; jx < 4; ++jx)
#pragma unroll
      for (int jy = 0; jy < 4; ++jy) {
        const int row = (jx * 4 + jy) * 4 + ju_a;
        double* slot = accT + row * R + swz<KV>(row, col >> 1) * 2 + (col & 1);
        *slot = use_fn ? fma(cs, acc[jx][jy], p.c0 * *slot) : cs * acc[jx][jy];
      }
  }
  __syncthreads();

  // ---- phase B: u and v, stage combination --------------------------------------------------------------------------
  double fb[4][4], res[4][4];
  const int rowb = (jx_b * 4 + jy_b) * 4;
#pragma unroll
  for (int ju = 0; ju < 4; ++ju) {
    const int row = rowb + ju;
    const double2 a = *reinterpret_cast<const double2*>(tile + row * R + swz<KV>(row, 2 * ev) * 2);
    const double2 b = *reinterpret_cast<const double2*>(tile + row * R + swz<KV>(row, 2 * ev + 1) * 2);
    fb[ju][0] = a.x; fb[ju][1] = a.y; fb[ju][2] = b.x; fb[ju][3] = b.y;
  }
  {
#pragma unroll
    for (int jv = 0; jv < 4; ++jv) {                                  // u lines (fixed jv)
      const double h = hUs[jv * NT + tid];
      const double uL = au[jv] > 0.0 ? h : fb[0][jv], uR = au[jv] > 0.0 ? fb[3][jv] : h;
      const double su = p.J[2] * au[jv];
#pragma unroll
      for (int ju = 0; ju < 4; ++ju) {
        double v = p.Xi[2 * ju] * uL;
        v = fma(-p.Xi[2 * ju + 1], uR, v);
#pragma unroll
        for (int k = 0; k < 4; ++k) v = fma(p.U[ju * 4 + k], fb[k][jv], v);
        res[ju][jv] = su * v;
      }
    }
  }
#pragma unroll
  for (int ju = 0; ju < 4; ++ju) {                                    // v lines (fixed ju): neighbours from the adjacent lanes
    const double from_lo = __shfl_up_sync(0xffffffffu, fb[ju][3], 1), from_hi = __shfl_down_sync(0xffffffffu, fb[ju][0], 1);
    const double nlo = ev > 0 ? from_lo : eV[ju], nhi = ev < KV - 1 ? from_hi : eV[ju];
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
  double dens = 0.0;
  double2* q = reinterpret_cast<double2*>(p.out + xy + gu0 * s2 + gvb);
  const double2 w01 = *reinterpret_cast<const double2*>(p.wqv + gvb), w23 = *reinterpret_cast<const double2*>(p.wqv + gvb + 2);
#pragma unroll
  for (int ju = 0; ju < 4; ++ju) {
    // running sum of phase A (x and y parts, already scaled, + c0 f_n) + the u and v parts
    const int row = rowb + ju;
    const double2 sa = *reinterpret_cast<const double2*>(accT + row * R + swz<KV>(row, 2 * ev) * 2);
    const double2 sb = *reinterpret_cast<const double2*>(accT + row * R + swz<KV>(row, 2 * ev + 1) * 2);
    double o[4] = {sa.x, sa.y, sb.x, sb.y};
#pragma unroll
    for (int jv = 0; jv < 4; ++jv) o[jv] += p.mode == 0 ? res[ju][jv] : p.c1 * fma(p.dt, res[ju][jv], fb[ju][jv]);
    if (p.wide_st) {        // the element's four v nodes are one 32-byte sector: a single 256-bit streaming store
      asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(q), "d"(o[0]), "d"(o[1]), "d"(o[2]), "d"(o[3]) : "memory");
    } else {
      __stcs(q, make_double2(o[0], o[1]));
      __stcs(q + 1, make_double2(o[2], o[3]));
    }
    q += s2 / 2;
    if (p.partials) {
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
