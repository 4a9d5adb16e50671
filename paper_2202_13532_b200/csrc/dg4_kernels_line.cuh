// 2D2V line kernel for n = 8 LGL nodes in all four dimensions (the order the paper runs), sm_100a:
// fused RHS (x, y, v_x, v_y volume contractions + upwind face lift, Eq. 14/20/21/23 of PAPER.md) + SSP-RK3 stage combination
// + density partials of the output.  The 1D2V tiled kernel (dg_kernels_tiled.cuh) carried over to four dimensions.
//
// Tile = ONE element = 8^4 nodes = 512 rows (jx, jy, ju) of 8 contiguous doubles (the v line, 64 bytes).  One CTA of 256
// threads per tile.  TMA (cp.async.bulk.tensor.4d) brings the tile, the f_n tile and the upwind face halos (x, y, u faces:
// 64 rows each; v faces: 512 rows of 2 doubles) into shared memory on one mbarrier -- periodic wrap by coordinate, zero
// inflow by letting the box fall outside the tensor (TMA fills zeros) -- and the result leaves by one TMA store.  No thread
// touches global memory for f.
//
// Four line phases, two lines per thread and phase (the operator coefficients, kernel-parameter constants, are fetched once
// for both), the even-odd form of the centro-antisymmetric operator (apply_lines2).  The running sum lives in the f_n tile
// (c0 f_n + c1 dt (parts so far)), so a CTA holds two 32 KB tiles + 40 KB of halos and two CTAs share an SM.
//
// Shared-memory layout of a tile: rows in TMA order, the four 16-byte chunks of a row XORed with (row / 2) mod 4
// (CU_TENSOR_MAP_SWIZZLE_64B).  A phase whose threads read, for two lines at once, the 16-byte chunk (v pair) `cv` of the rows of
// a line is bank-conflict free when the 8 lanes of a quarter-warp are 4 chunks x 2 rows of different parity:
//   phase x  thread = (jy, ju, cv), line over jx: the two rows are ju, ju+1                      (adjacent rows)
//   phase y  thread = (jx, ju, cv), line over jy: ju, ju+1                                        (adjacent rows)
//   phase u  thread = (jx, jy, cv), line over ju: the rows of jy and jy+1 are 8 apart -- same parity.  The odd-jy threads walk
//            their line BACKWARDS (row 7 - i at step i): the mirrored line f'_i = f_{7-i} has e' = e, o' = -o, so the same
//            even-odd routine with the two face states swapped gives (Ups f - Xi_R uR + Xi_L uL)_{7-i} = -s'_i; with the
//            mirrored speed a' = -a the contribution a s_{7-i} = a' s'_i -- no data is permuted, only the row address
//            (i XOR 7) and a sign (the reflection symmetry of the reference element, Eq. 53/54).
//   phase v  thread = rows t and t + 256, line = the row itself: 8 consecutive rows at one chunk index hit 8 bank groups.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

#include "dg_kernels_tiled.cuh"

namespace dg4l {

using dgt::smem_u32;

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const void* tmap, uint32_t bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_store_4d(const void* tmap, uint32_t src, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
               ::"l"(reinterpret_cast<uint64_t>(tmap)), "r"(src), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

constexpr int NN = 8, H = 4, NT = 256, ROWS = 512;
constexpr int SZ_TILE = ROWS * NN * 8;          // 32 KB
constexpr int SZ_FACE = 64 * NN * 8;            // 4 KB: x, y, u faces (64 rows of 8)
constexpr int SZ_VFACE = ROWS * 2 * 8;          // 8 KB: v faces (512 rows of 2)
constexpr int OFF_F = 0, OFF_N = OFF_F + SZ_TILE;
constexpr int OFF_XL = OFF_N + SZ_TILE, OFF_XR = OFF_XL + SZ_FACE;
constexpr int OFF_YL = OFF_XR + SZ_FACE, OFF_YR = OFF_YL + SZ_FACE;
constexpr int OFF_UL = OFF_YR + SZ_FACE, OFF_UR = OFF_UL + SZ_FACE;
constexpr int OFF_VL = OFF_UR + SZ_FACE, OFF_VR = OFF_VL + SZ_VFACE;
constexpr int OFF_BAR = OFF_VR + SZ_VFACE;
constexpr int SMEM_BYTES = OFF_BAR + 128;       // 106 624 B: two CTAs per SM

struct alignas(64) LineParams {
  CUtensorMap m_main;    // stage input f_s, box (8, 8, 8, 8), SWIZZLE_64B
  CUtensorMap m_fn;      // f_n, same box
  CUtensorMap m_out;     // output, same box
  CUtensorMap m_xface;   // f_s, box (8, 8, 8, 1)
  CUtensorMap m_yface;   // f_s, box (8, 8, 1, 8)
  CUtensorMap m_uface;   // f_s, box (8, 1, 8, 8)
  CUtensorMap m_vface;   // f_s, box (2, 8, 8, 8)
  CUtensorMap m_xhalo;   // exterior x-face planes [2][G1][G2][G3] of an x-slab (bc[0] = 2), box (8, 8, 8, 1)
  double pe[NN * NN / 4], qo[NN * NN / 4], la[H], lb[H];   // even-odd operator, see dg_kernels_tiled.cuh
  double wref[NN];       // LGL weights on [-1, 1] (Eq. 45)
  const double* cu;      // node coordinates of u = v_x and v = v_y
  const double* cv;
  const double* Ex;      // [G0][G1] or nullptr
  const double* Ey;
  double* partials;      // [G0*G1][chunks] density partials of the output
  double Jx, Jy, Ju, Jv, omega_c;
  double wscale;         // 1 / (J_u J_v)
  double c0, c1, dt;     // out = c0 f_n + c1 (f + dt rhs)  (mode 1);  out = rhs  (mode 0)
  int N[4], G[4], bc[4];
  int mode, want_partials, chunks, bx_log2, strong;
};

// offset (doubles) of the 16-byte chunk `c` (nodes 2c, 2c+1) of row `r` inside a swizzled tile
__device__ __forceinline__ int chunk_off(int r, int c) { return r * NN + (((c ^ (r >> 1)) & 3) << 1); }

template <bool FN>
__global__ void __launch_bounds__(NT, 2) rhs4_line_kernel(const __grid_constant__ LineParams P) {
  extern __shared__ __align__(1024) unsigned char smem[];
  double* sF = reinterpret_cast<double*>(smem + OFF_F);
  double* sN = reinterpret_cast<double*>(smem + OFF_N);
  double* sXL = reinterpret_cast<double*>(smem + OFF_XL);
  double* sXR = reinterpret_cast<double*>(smem + OFF_XR);
  double* sYL = reinterpret_cast<double*>(smem + OFF_YL);
  double* sYR = reinterpret_cast<double*>(smem + OFF_YR);
  double* sUL = reinterpret_cast<double*>(smem + OFF_UL);
  double* sUR = reinterpret_cast<double*>(smem + OFF_UR);
  double* sVL = reinterpret_cast<double*>(smem + OFF_VL);
  double* sVR = reinterpret_cast<double*>(smem + OFF_VR);
  const uint32_t bar = smem_u32(smem + OFF_BAR);
  const int t = threadIdx.x;

  // Tile coordinates.  Consecutive CTAs walk v, then the x elements of a group of 2^bx_log2, then u; then y; then the x
  // groups: the v, x and u neighbours of a tile are in flight with it and its y neighbour is N_u BX N_v tiles away (L2).
  int bid = blockIdx.x;
  const int ev = bid % P.N[3]; bid /= P.N[3];
  const int bx = bid & ((1 << P.bx_log2) - 1); bid >>= P.bx_log2;
  const int eu = bid % P.N[2]; bid /= P.N[2];
  const int ey = bid % P.N[1];
  const int ex = ((bid / P.N[1]) << P.bx_log2) + bx;
  const int gx0 = ex * NN, gy0 = ey * NN, gu0 = eu * NN, gv0 = ev * NN;

  if (t == 0) {
    if (smem_u32(smem) & 511u) __trap();             // the 64-byte swizzle pattern repeats every 512 bytes
    dgt::mbar_init(bar, 1);
    dgt::fence_mbar_init();
    // the tile itself (and f_n) first: the loads are in flight while the threads fetch their speeds and work out which halos
    // the signs need
    dgt::mbar_expect_tx_noarrive(bar, (FN ? 2u : 1u) * SZ_TILE);
    tma_load_4d(smem_u32(sF), &P.m_main, bar, gv0, gu0, gy0, gx0);
    if (FN) tma_load_4d(smem_u32(sN), &P.m_fn, bar, gv0, gu0, gy0, gx0);
  }
  const double cf = (P.mode != 0) ? P.c1 : 0.0;
  const double cr = (P.mode != 0) ? P.c1 * P.dt : 1.0;
  // the speeds below carry the factor cr; the upwind side of Eq. 23 follows the sign of the speed itself (upwind_bits)
  const bool flip = cr < 0.0;
  // thread <-> line maps.  x / y / u phases: t = (hi, mid, cv); v phase: rows t and t + 256.
  const int cv = t & 3, mid = (t >> 2) & 7, hi = t >> 5;
  const int c2 = 2 * cv;
  // speeds (Eq. 28), scaled by cr J_d: all global reads of the thread in one batch
  const double ax = cr * P.Jx * P.cu[gu0 + mid];                                   // phase x: mid = ju
  const double2 vv = *reinterpret_cast<const double2*>(P.cv + gv0 + c2);
  const double ay0 = cr * P.Jy * vv.x, ay1 = cr * P.Jy * vv.y;                     // phase y: a_y = v
  const int urev = (mid & 1) ? 7 : 0;                                              // phase u: mid = jy; odd jy walks backwards
  double au0, au1;
  {
    const double exf = P.Ex ? P.Ex[(long long)(gx0 + hi) * P.G[1] + gy0 + mid] : 0.0;
    au0 = cr * P.Ju * (-exf - P.omega_c * vv.x);                                   // a_u = -E_x - omega_c v
    au1 = cr * P.Ju * (-exf - P.omega_c * vv.y);
  }
  double avl[2];
  {
    const int ju = t & 7, jy = (t >> 3) & 7, jx = t >> 6;
    const double wu = P.omega_c * P.cu[gu0 + ju];
#pragma unroll
    for (int l = 0; l < 2; ++l) {
      const double eyf = P.Ey ? P.Ey[(long long)(gx0 + jx + 4 * l) * P.G[1] + gy0 + jy] : 0.0;
      avl[l] = cr * P.Jv * (-eyf + wu);                                            // a_v = -E_y + omega_c u
    }
  }
  // upwind sides of this thread's lines (Eq. 23): bits 0-1 x, 2-3 / 4-5 y, 6-7 / 8-9 u, 10-11 / 12-13 v; bit 0 of a pair =
  // a > 0 (the state below the element enters), bit 1 = a < 0.  The threads' lines cover the tile in every phase, so the OR
  // over the CTA says exactly which face halos are read at all.
  const int um = dgt::upwind_bits(ax, flip) | (dgt::upwind_bits(ay0, flip) << 2) | (dgt::upwind_bits(ay1, flip) << 4) |
                 (dgt::upwind_bits(au0, flip) << 6) | (dgt::upwind_bits(au1, flip) << 8) |
                 (dgt::upwind_bits(avl[0], flip) << 10) | (dgt::upwind_bits(avl[1], flip) << 12);
  if (urev) { au0 = -au0; au1 = -au1; }                                            // mirrored line: a' = -a
  int* sAny = reinterpret_cast<int*>(smem + OFF_BAR + 64);                         // one word per warp
  {
    const int w_or = __reduce_or_sync(0xffffffffu, um);
    if ((t & 31) == 0) sAny[t >> 5] = w_or;
  }
  __syncthreads();           // also makes the barrier initialisation visible to all waiters
  if (t == 0) {
    int any = 0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) any |= sAny[w];
    const int ax_pos = any & 1, ax_neg = (any >> 1) & 1;
    const int ay_pos = ((any >> 2) | (any >> 4)) & 1, ay_neg = ((any >> 3) | (any >> 5)) & 1;
    const int au_pos = ((any >> 6) | (any >> 8)) & 1, au_neg = ((any >> 7) | (any >> 9)) & 1;
    const int av_pos = ((any >> 10) | (any >> 12)) & 1, av_neg = ((any >> 11) | (any >> 13)) & 1;
    const uint32_t bytes = (uint32_t)((ax_pos + ax_neg + ay_pos + ay_neg + au_pos + au_neg) * SZ_FACE + (av_pos + av_neg) * SZ_VFACE);
    dgt::mbar_expect_tx(bar, bytes);          // the one arrival of this phase, with the halo bytes
    // neighbour node index in dimension d below / above the element: periodic wrap (the paper's roll) by
    // coordinate; zero inflow: outside the tensor, where TMA fills zeros (exterior state 0, reading C2)
    auto below = [&](int d, int e, int g0) { return e > 0 ? g0 - 1 : (P.bc[d] == 0 ? P.G[d] - 1 : -1); };
    auto above = [&](int d, int e, int g0) { return e < P.N[d] - 1 ? g0 + NN : (P.bc[d] == 0 ? 0 : P.G[d]); };
    if (ax_pos) {
      if (P.bc[0] == 2 && ex == 0) tma_load_4d(smem_u32(sXL), &P.m_xhalo, bar, gv0, gu0, gy0, 0);
      else tma_load_4d(smem_u32(sXL), &P.m_xface, bar, gv0, gu0, gy0, below(0, ex, gx0));
    }
    if (ax_neg) {
      if (P.bc[0] == 2 && ex == P.N[0] - 1) tma_load_4d(smem_u32(sXR), &P.m_xhalo, bar, gv0, gu0, gy0, 1);
      else tma_load_4d(smem_u32(sXR), &P.m_xface, bar, gv0, gu0, gy0, above(0, ex, gx0));
    }
    if (ay_pos) tma_load_4d(smem_u32(sYL), &P.m_yface, bar, gv0, gu0, below(1, ey, gy0), gx0);
    if (ay_neg) tma_load_4d(smem_u32(sYR), &P.m_yface, bar, gv0, gu0, above(1, ey, gy0), gx0);
    if (au_pos) tma_load_4d(smem_u32(sUL), &P.m_uface, bar, gv0, below(2, eu, gu0), gy0, gx0);
    if (au_neg) tma_load_4d(smem_u32(sUR), &P.m_uface, bar, gv0, above(2, eu, gu0), gy0, gx0);
    // v faces: boxes of two nodes (16 bytes, the TMA minimum); the face node is the second of the lower box, the first of the upper
    if (av_pos) tma_load_4d(smem_u32(sVL), &P.m_vface, bar, ev > 0 ? gv0 - 2 : (P.bc[3] == 0 ? P.G[3] - 2 : -2), gu0, gy0, gx0);
    if (av_neg) tma_load_4d(smem_u32(sVR), &P.m_vface, bar, ev < P.N[3] - 1 ? gv0 + NN : (P.bc[3] == 0 ? 0 : P.G[3]), gu0, gy0, gx0);
  }
  dgt::mbar_wait(bar, 0);
  // upwind tests on the bits (the mirrored u lines swapped their speeds' signs above, and their faces below)
  auto pos = [um](int line) { return (um >> (2 * line)) & 1; };
  auto neg = [um](int line) { return (um >> (2 * line + 1)) & 1; };

  // ---------------- phase x: thread = (jy = hi, ju = mid, cv), lines over jx ----------------
  {
    double f[2][NN], s[2][NN], uL[2], uR[2];
    const int rbase = hi * NN + mid;
#pragma unroll
    for (int k = 0; k < NN; ++k) {
      const double2 v = *reinterpret_cast<const double2*>(&sF[chunk_off(k * 64 + rbase, cv)]);
      f[0][k] = v.x; f[1][k] = v.y;
    }
    if (pos(0)) { const double2 v = *reinterpret_cast<const double2*>(&sXL[rbase * NN + c2]); uL[0] = v.x; uL[1] = v.y; }
    else { uL[0] = f[0][0]; uL[1] = f[1][0]; }
    if (neg(0)) { const double2 v = *reinterpret_cast<const double2*>(&sXR[rbase * NN + c2]); uR[0] = v.x; uR[1] = v.y; }
    else { uR[0] = f[0][NN - 1]; uR[1] = f[1][NN - 1]; }
    dgt::apply_lines2<NN>(P, P.strong != 0, f, uL, uR, s);
#pragma unroll
    for (int j = 0; j < NN; ++j) {
      double2* q = reinterpret_cast<double2*>(&sN[chunk_off(j * 64 + rbase, cv)]);
      if (FN) { const double2 n2 = *q; *q = make_double2(fma(P.c0, n2.x, ax * s[0][j]), fma(P.c0, n2.y, ax * s[1][j])); }
      else *q = make_double2(ax * s[0][j], ax * s[1][j]);
    }
  }
  __syncthreads();
  // ---------------- phase y: thread = (jx = hi, ju = mid, cv), lines over jy ----------------
  {
    double f[2][NN], s[2][NN], uL[2], uR[2];
    const int rbase = hi * 64 + mid;
#pragma unroll
    for (int k = 0; k < NN; ++k) {
      const double2 v = *reinterpret_cast<const double2*>(&sF[chunk_off(rbase + k * NN, cv)]);
      f[0][k] = v.x; f[1][k] = v.y;
    }
    const double2 hl = *reinterpret_cast<const double2*>(&sYL[(hi * NN + mid) * NN + c2]);
    const double2 hr = *reinterpret_cast<const double2*>(&sYR[(hi * NN + mid) * NN + c2]);
    uL[0] = pos(1) ? hl.x : f[0][0];
    uL[1] = pos(2) ? hl.y : f[1][0];
    uR[0] = neg(1) ? hr.x : f[0][NN - 1];
    uR[1] = neg(2) ? hr.y : f[1][NN - 1];
    dgt::apply_lines2<NN>(P, P.strong != 0, f, uL, uR, s);
#pragma unroll
    for (int j = 0; j < NN; ++j) {
      double2* q = reinterpret_cast<double2*>(&sN[chunk_off(rbase + j * NN, cv)]);
      const double2 n2 = *q;
      *q = make_double2(fma(ay0, s[0][j], n2.x), fma(ay1, s[1][j], n2.y));
    }
  }
  __syncthreads();
  // ---------------- phase u: thread = (jx = hi, jy = mid, cv), lines over ju (odd jy: mirrored) ----------------
  {
    double f[2][NN], s[2][NN], uL[2], uR[2];
    const int rbase = (hi * NN + mid) * NN;
#pragma unroll
    for (int i = 0; i < NN; ++i) {
      const double2 v = *reinterpret_cast<const double2*>(&sF[chunk_off(rbase + (i ^ urev), cv)]);
      f[0][i] = v.x; f[1][i] = v.y;
    }
    // the mirrored threads see the element's upper face as their "left" one
    const double2 hl = *reinterpret_cast<const double2*>(&(urev ? sUR : sUL)[(hi * NN + mid) * NN + c2]);
    const double2 hr = *reinterpret_cast<const double2*>(&(urev ? sUL : sUR)[(hi * NN + mid) * NN + c2]);
    // (bits 3, 4 describe the true speeds; a mirrored line sees them with the opposite sign)
    uL[0] = (urev ? neg(3) : pos(3)) ? hl.x : f[0][0];
    uL[1] = (urev ? neg(4) : pos(4)) ? hl.y : f[1][0];
    uR[0] = (urev ? pos(3) : neg(3)) ? hr.x : f[0][NN - 1];
    uR[1] = (urev ? pos(4) : neg(4)) ? hr.y : f[1][NN - 1];
    dgt::apply_lines2<NN>(P, P.strong != 0, f, uL, uR, s);
#pragma unroll
    for (int i = 0; i < NN; ++i) {
      double2* q = reinterpret_cast<double2*>(&sN[chunk_off(rbase + (i ^ urev), cv)]);
      const double2 n2 = *q;
      *q = make_double2(fma(au0, s[0][i], n2.x), fma(au1, s[1][i], n2.y));
    }
  }
  __syncthreads();
  // ---------------- phase v: thread = rows t and t + 256, the line is the row ----------------
  {
    double f[2][NN], s[2][NN], acc[2][NN], uL[2], uR[2];
#pragma unroll
    for (int l = 0; l < 2; ++l) {
      const int row = t + 256 * l;
#pragma unroll
      for (int c = 0; c < H; ++c) {
        const double2 v2 = *reinterpret_cast<const double2*>(&sF[chunk_off(row, c)]);
        f[l][2 * c] = v2.x; f[l][2 * c + 1] = v2.y;
        const double2 a2 = *reinterpret_cast<const double2*>(&sN[chunk_off(row, c)]);
        acc[l][2 * c] = a2.x; acc[l][2 * c + 1] = a2.y;
      }
      uL[l] = f[l][0]; uR[l] = f[l][NN - 1];
      if (pos(5 + l)) uL[l] = sVL[row * 2 + 1];
      if (neg(5 + l)) uR[l] = sVR[row * 2];
    }
    dgt::apply_lines2<NN>(P, P.strong != 0, f, uL, uR, s);
    double psum[2] = {0.0, 0.0};
#pragma unroll
    for (int l = 0; l < 2; ++l) {
      const int row = t + 256 * l;
#pragma unroll
      for (int j = 0; j < NN; ++j) acc[l][j] = fma(cf, f[l][j], fma(avl[l], s[l][j], acc[l][j]));
#pragma unroll
      for (int c = 0; c < H; ++c)
        *reinterpret_cast<double2*>(&sN[chunk_off(row, c)]) = make_double2(acc[l][2 * c], acc[l][2 * c + 1]);
      if (P.want_partials) {
        // Eq. 27: LGL quadrature of the stage output over this row
        double p0 = 0.0;
#pragma unroll
        for (int k = 0; k < NN; ++k) p0 = fma(P.wref[k], acc[l][k], p0);
        psum[l] = P.wref[t & 7] * p0 * P.wscale;
      }
    }
    if (P.want_partials) {
      // the 8 rows (ju) of an (jx, jy) node are 8 consecutive lanes: fixed butterfly, deterministic
#pragma unroll
      for (int off = 4; off > 0; off >>= 1) {
        psum[0] += __shfl_xor_sync(0xffffffffu, psum[0], off);
        psum[1] += __shfl_xor_sync(0xffffffffu, psum[1], off);
      }
      if ((t & 7) == 0) {
        const int jy = (t >> 3) & 7, jx = t >> 6;
        const long long tile_chunk = (long long)eu * P.N[3] + ev;
        P.partials[((long long)(gx0 + jx) * P.G[1] + gy0 + jy) * P.chunks + tile_chunk] = psum[0];
        P.partials[((long long)(gx0 + jx + 4) * P.G[1] + gy0 + jy) * P.chunks + tile_chunk] = psum[1];
      }
    }
  }
  dgt::fence_proxy_async();       // generic-proxy writes to sN must be visible to the TMA store
  __syncthreads();
  if (t == 0) {
    tma_store_4d(&P.m_out, smem_u32(sN), gv0, gu0, gy0, gx0);
    dgt::tma_store_commit_and_wait_read();
  }
}

}  // namespace dg4l
