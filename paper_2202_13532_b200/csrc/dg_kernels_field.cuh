// Batched DG->Fourier projection / synthesis as one dense FP64 contraction (Eq. 63 and Eq. 71,
// PAPER.md:405-411, 459):  C[M][N] = A[M][K] * B[N][K]^T, all row-major with K contiguous
// (projection: A = rho[batch][G], B = T[2(pmax+1)][G];  synthesis: A = c[batch][Q], B = S[G][Q]).
// Register-tiled DFMA kernel: 128x128 CTA tile, 8x8 thread tile, BK = 8, register prefetch of the
// next k-tile.  FP64-pipe bound.
#pragma once
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <cstdint>

#include "../../include/dgvlasov.h"
#include "dg_context.hpp"

namespace dgf {

constexpr int BM = 128, BN = 128, BK = 8, PITCH = 130;   // PITCH: conflict-free transposed stores, 16-B aligned rows

inline bool gemm_worthwhile(int M, int N, int K) { return M >= 32 && (long long)N * K >= (1LL << 16); }

// Load 4 consecutive k-values of row `row` (or zeros outside the matrix).
__device__ __forceinline__ void load4(const double* __restrict__ P, int row, int rows, int k, int K, bool vec, double v[4]) {
  if (row < rows) {
    const double* src = P + (size_t)row * K + k;
    if (vec && k + 3 < K) {
      const double2 a = *reinterpret_cast<const double2*>(src);
      const double2 b = *reinterpret_cast<const double2*>(src + 2);
      v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i) v[i] = (k + i < K) ? src[i] : 0.0;
    }
  } else {
    v[0] = v[1] = v[2] = v[3] = 0.0;
  }
}

__global__ void __launch_bounds__(256) field_gemm_tn_kernel(const double* __restrict__ A, const double* __restrict__ B,
                                                            double* __restrict__ C, int M, int N, int K, int vec) {
  __shared__ __align__(16) double As[2][BK][PITCH];
  __shared__ __align__(16) double Bs[2][BK][PITCH];
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;
  // tiles ordered so that consecutive CTAs share the same B rows (T / S panel) through L2
  const int tiles_m = (M + BM - 1) / BM;
  const int bm = (blockIdx.x % tiles_m) * BM, bn = (blockIdx.x / tiles_m) * BN;
  const int lrow = tid >> 1, lk = (tid & 1) * 4;      // this thread stages row lrow, k-offset lk of both tiles

  double acc[8][8];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j] = 0.0;

  double ra[4], rb[4];
  load4(A, bm + lrow, M, lk, K, vec != 0, ra);
  load4(B, bn + lrow, N, lk, K, vec != 0, rb);
#pragma unroll
  for (int i = 0; i < 4; ++i) { As[0][lk + i][lrow] = ra[i]; Bs[0][lk + i][lrow] = rb[i]; }
  __syncthreads();

  const int ktiles = (K + BK - 1) / BK;
  for (int kt = 0; kt < ktiles; ++kt) {
    const int cur = kt & 1;
    if (kt + 1 < ktiles) {
      load4(A, bm + lrow, M, (kt + 1) * BK + lk, K, vec != 0, ra);
      load4(B, bn + lrow, N, (kt + 1) * BK + lk, K, vec != 0, rb);
    }
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      double a[8], b[8];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const double2 va = *reinterpret_cast<const double2*>(&As[cur][k][i * 32 + ty * 2]);
        const double2 vb = *reinterpret_cast<const double2*>(&Bs[cur][k][i * 32 + tx * 2]);
        a[2 * i] = va.x; a[2 * i + 1] = va.y;
        b[2 * i] = vb.x; b[2 * i + 1] = vb.y;
      }
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    if (kt + 1 < ktiles) {
#pragma unroll
      for (int i = 0; i < 4; ++i) { As[cur ^ 1][lk + i][lrow] = ra[i]; Bs[cur ^ 1][lk + i][lrow] = rb[i]; }
    }
    __syncthreads();
  }

  const bool cvec = (N % 2 == 0) && ((reinterpret_cast<uintptr_t>(C) & 15) == 0);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int m = bm + (i >> 1) * 32 + ty * 2 + (i & 1);
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int nn = bn + j * 32 + tx * 2;
      double* dst = C + (size_t)m * N + nn;
      if (cvec && nn + 1 < N) *reinterpret_cast<double2*>(dst) = make_double2(acc[i][2 * j], acc[i][2 * j + 1]);
      else {
        if (nn < N) dst[0] = acc[i][2 * j];
        if (nn + 1 < N) dst[1] = acc[i][2 * j + 1];
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Tensor-core form of the same contraction: DMMA (mma.sync m8n8k4 f64, SASS DMMA.8x8x4).  On B200 DMMA has the
// DFMA peak (37 TFLOP/s measured for both), but one warp instruction carries 256 multiply-adds instead of 32,
// so operand fetch and issue no longer compete with the arithmetic.  128x128 CTA tile, 8 warps of 64x32,
// BK = 16, three cp.async stages, rows padded to 20 doubles (fragment loads are bank-conflict free).
// Needs K even and 16-byte aligned A, B.  The accumulation order over k is fixed: deterministic.
// ------------------------------------------------------------------------------------------------
constexpr int TK = 16, TPITCH = 20, TSTAGES = 3;
constexpr int DMMA_SMEM_BYTES = TSTAGES * 2 * 128 * TPITCH * 8;

__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}

__global__ void __launch_bounds__(256, 1) field_gemm_dmma_kernel(const double* __restrict__ A, const double* __restrict__ B,
                                                                 double* __restrict__ C, int M, int N, int K) {
  extern __shared__ __align__(16) double gsm[];
  double* As = gsm;                                   // [TSTAGES][128][TPITCH]
  double* Bs = gsm + TSTAGES * 128 * TPITCH;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, tig = lane & 3;
  const int wm = (warp & 1) * 64, wn = (warp >> 1) * 32;
  const int tiles_m = (M + 127) / 128;
  const int bm = (blockIdx.x % tiles_m) * 128, bn = (blockIdx.x / tiles_m) * 128;
  const uint32_t as_u = (uint32_t)__cvta_generic_to_shared(As), bs_u = (uint32_t)__cvta_generic_to_shared(Bs);

  auto load_stage = [&](int stage, int k0) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int c = tid + i * 256, row = c >> 3, kc = (c & 7) * 2;
      const int k = k0 + kc;
      const int kb = (k < K) ? 16 : 0;                // K is even: a 16-byte chunk is inside or outside
      const int ra = bm + row, rb = bn + row;
      const double* sa = A + (size_t)min(ra, M - 1) * K + min(k, K - 2);
      const double* sb = B + (size_t)min(rb, N - 1) * K + min(k, K - 2);
      const uint32_t off = (uint32_t)((stage * 128 + row) * TPITCH + kc) * 8u;
      cp_async16_zfill(as_u + off, sa, ra < M ? kb : 0);
      cp_async16_zfill(bs_u + off, sb, rb < N ? kb : 0);
    }
  };

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const int ktiles = (K + TK - 1) / TK;
  load_stage(0, 0);
  asm volatile("cp.async.commit_group;" ::: "memory");
  if (ktiles > 1) load_stage(1, TK);
  asm volatile("cp.async.commit_group;" ::: "memory");

  for (int kt = 0; kt < ktiles; ++kt) {
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    __syncthreads();                                  // stage kt landed; everyone is done with stage kt-1
    if (kt + 2 < ktiles) load_stage((kt + 2) % TSTAGES, (kt + 2) * TK);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const double* as = As + (size_t)(kt % TSTAGES) * 128 * TPITCH;
    const double* bs = Bs + (size_t)(kt % TSTAGES) * 128 * TPITCH;
#pragma unroll
    for (int k4 = 0; k4 < TK; k4 += 4) {
      double a[8], b[4];
#pragma unroll
      for (int i = 0; i < 8; ++i) a[i] = as[(wm + i * 8 + g) * TPITCH + k4 + tig];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = bs[(wn + j * 8 + g) * TPITCH + k4 + tig];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                       : "+d"(acc[i][j][0]), "+d"(acc[i][j][1]) : "d"(a[i]), "d"(b[j]));
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");

  const bool cvec = (N % 2 == 0) && ((reinterpret_cast<uintptr_t>(C) & 15) == 0);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int m = bm + wm + i * 8 + g;
    if (m >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int nn = bn + wn + j * 8 + 2 * tig;
      double* dst = C + (size_t)m * N + nn;
      if (cvec && nn + 1 < N) *reinterpret_cast<double2*>(dst) = make_double2(acc[i][j][0], acc[i][j][1]);
      else {
        if (nn < N) dst[0] = acc[i][j][0];
        if (nn + 1 < N) dst[1] = acc[i][j][1];
      }
    }
  }
}

// variant: 0 auto (DMMA when the operands allow it), 1 DFMA register-tiled kernel, 2 DMMA (error if not allowed)
inline int launch_gemm_tn(const double* A, const double* B, double* C, int M, int N, int K, cudaStream_t st, int variant = 0) {
  const bool dmma_ok = (K % 2 == 0) && K >= 2 && ((reinterpret_cast<uintptr_t>(A) & 15) == 0) && ((reinterpret_cast<uintptr_t>(B) & 15) == 0);
  if (variant == 2 && !dmma_ok) return DG_ERR_UNSUPPORTED;
  if (variant != 1 && dmma_ok) {
    const long long tiles = (long long)((M + 127) / 128) * ((N + 127) / 128);
    if (tiles <= 0 || tiles > 0x7fffffffLL) return DG_ERR_INVALID_ARG;
    if (ensure_dyn_smem(reinterpret_cast<const void*>(field_gemm_dmma_kernel), DMMA_SMEM_BYTES) != cudaSuccess) return DG_ERR_CUDA;
    field_gemm_dmma_kernel<<<(unsigned)tiles, 256, DMMA_SMEM_BYTES, st>>>(A, B, C, M, N, K);
    return DG_OK;
  }

  const int tiles_m = (M + BM - 1) / BM, tiles_n = (N + BN - 1) / BN;
  const long long tiles = (long long)tiles_m * tiles_n;
  if (tiles <= 0 || tiles > 0x7fffffffLL) return DG_ERR_INVALID_ARG;
  const int vec = (K % 2 == 0) && ((reinterpret_cast<uintptr_t>(A) & 15) == 0) && ((reinterpret_cast<uintptr_t>(B) & 15) == 0);
  field_gemm_tn_kernel<<<(unsigned)tiles, 256, 0, st>>>(A, B, C, M, N, K, vec);
  return DG_OK;
}


// ------------------------------------------------------------------------------------------------
// One-launch field solve of a single density vector (the per-stage solve inside dg_ssprk3_*):
//   rho[gx] = sum_c partial[gx][c]                    (finish of Eq. 27)
//   c_q     = sum_gx T[q][gx] rho[gx]                 (Eq. 63)
//   E[gx]   = sum_q S[gx][q] c_q                      (Eq. 71; Poisson factor folded into S)
// CTA b owns the x nodes [b*rows, (b+1)*rows): it finishes their densities, forms its share of every
// c_q, and after a grid-wide rendezvous sums all shares in CTA order (deterministic) and synthesises
// E at its own nodes.  The grid never exceeds the SM count and each CTA needs few resources; the launch
// is cooperative, so the driver checks that all CTAs are co-resident and the rendezvous is the grid
// barrier of cooperative groups.
// ------------------------------------------------------------------------------------------------
struct FieldFusedParams {
  const double* partials;   // [G0][nchunks]
  const double* T;          // [Q][G0]
  const double* S;          // [G0][Q]
  double* rho;              // [G0]
  double* cpart;            // [Q][grid] scratch (q-major)
  double* c;                // [Q]
  double* E;                // [G0]
  int nchunks, G0, Q, rows;
};

__global__ void __launch_bounds__(256) field_fused_kernel(const FieldFusedParams P) {
  extern __shared__ double fsm[];
  double* rho_s = fsm;                  // [rows]
  double* c_s = fsm + P.rows;           // [Q]
  double* half_s = c_s + P.Q;           // [2*rows] half-row sums of phase A
  double* T_s = half_s + 2 * P.rows;    // [Q][rows]  this CTA's columns of T
  double* S_s = T_s + P.Q * P.rows;     // [rows][Q]  this CTA's rows of S
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g0 = blockIdx.x * P.rows;
  const int nrows = max(0, min(P.rows, P.G0 - g0));
  // T and S are constants of the context: fetch this CTA's slices before waiting for the previous kernel, so their
  // DRAM latency (the f arrays streamed through L2 since the last stage) overlaps its tail.
  for (int e = tid; e < P.Q * nrows; e += 256) {
    const int q = e / nrows, i = e - q * nrows;
    T_s[q * P.rows + i] = P.T[(size_t)q * P.G0 + g0 + i];
    const int i2 = e / P.Q, q2 = e - i2 * P.Q;
    S_s[i2 * P.Q + q2] = P.S[(size_t)(g0 + i2) * P.Q + q2];
  }
#if __CUDA_ARCH__ >= 900
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
  // A: densities of the own nodes.  One warp per half row of partials (fixed split, fixed lane stride, fixed
  // butterfly), sixteen loads in flight per lane; the two halves are added in order: deterministic.
  const int hsplit = ((P.nchunks + 1) / 2 + 31) / 32 * 32;
  for (int item = warp; item < 2 * nrows; item += 8) {
    const int i = item >> 1, h = item & 1;
    const double* pr = P.partials + (size_t)(g0 + i) * P.nchunks;
    const int c_lo = h ? hsplit : 0, c_hi = h ? P.nchunks : min(hsplit, P.nchunks);
    double acc = 0.0;
#pragma unroll 16
    for (int cidx = c_lo + lane; cidx < c_hi; cidx += 32) acc += __ldcg(pr + cidx);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane == 0) half_s[item] = acc;
  }
  __syncthreads();
  if (tid < nrows) {
    const double r = half_s[2 * tid] + half_s[2 * tid + 1];
    rho_s[tid] = r;
    P.rho[g0 + tid] = r;
  }
  __syncthreads();
  // B: this CTA's share of c_q, stored q-major so that phase D reads along the CTA index
  for (int q = tid; q < P.Q; q += 256) {
    const double* tr = T_s + q * P.rows;
    double acc = 0.0;
    for (int i = 0; i < nrows; ++i) acc = fma(tr[i], rho_s[i], acc);
    P.cpart[(size_t)q * gridDim.x + blockIdx.x] = acc;
  }
  // C: grid-wide rendezvous.  The launch is cooperative (launch_field_fused), so the grid barrier of cooperative groups
  // applies: it orders the cpart stores above before the loads of phase D in every CTA.
  cooperative_groups::this_grid().sync();
  // D: c_q = sum of the shares.  One warp per q (q = warp, warp + 8, ...), lanes along the CTA index (grid <= 128: at
  // most four loads per lane, added in order), then a fixed butterfly: the same association in every CTA and every
  // run.  Eight q per pass: 32 loads in flight per lane.
  const int nb = (int)gridDim.x;
  for (int qb = warp; qb < P.Q; qb += 64) {
    double v[8][4];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int q = qb + 8 * u;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int b = lane + 32 * j;
        v[u][j] = (q < P.Q && b < nb) ? __ldcg(P.cpart + (size_t)q * nb + b) : 0.0;
      }
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      double acc = ((v[u][0] + v[u][1]) + v[u][2]) + v[u][3];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
      const int q = qb + 8 * u;
      if (lane == 0 && q < P.Q) {
        c_s[q] = acc;
        if (blockIdx.x == 0) P.c[q] = acc;
      }
    }
  }
  __syncthreads();
  // E: synthesis at the own nodes, one warp per node
  for (int i = warp; i < nrows; i += 8) {
    const double* sr = S_s + i * P.Q;
    double acc = 0.0;
#pragma unroll 8
    for (int q = lane; q < P.Q; q += 32) acc = fma(sr[q], c_s[q], acc);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane == 0) P.E[g0 + i] = acc;
  }
}

constexpr int FIELD_FUSED_MAX_GRID = 128;

// rows per CTA and grid of the fused field kernel for G0 x nodes
inline void field_fused_shape(int G0, int* rows, int* grid) {
  const int r = (G0 + FIELD_FUSED_MAX_GRID - 1) / FIELD_FUSED_MAX_GRID;
  *rows = r; *grid = (G0 + r - 1) / r;
}
inline size_t field_fused_smem(int rows, int Q) { return sizeof(double) * ((size_t)3 * rows + Q + (size_t)2 * rows * Q); }
inline bool field_fused_supported(int G0, int Q) {
  int rows, grid; field_fused_shape(G0, &rows, &grid);
  return field_fused_smem(rows, Q) <= 160 * 1024;
}

inline int launch_field_fused(const FieldFusedParams& P, int grid, bool pdl, cudaStream_t st) {
  const size_t smem = field_fused_smem(P.rows, P.Q);
  if (ensure_dyn_smem(reinterpret_cast<const void*>(field_fused_kernel), smem) != cudaSuccess) return DG_ERR_CUDA;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  // The kernel's CTAs meet at a grid-wide rendezvous: a cooperative launch makes the driver check that all of them can be
  // resident together (grid <= the SM count by construction, one CTA per SM) instead of assuming it.
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeCooperative;
  at[0].val.cooperative = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, field_fused_kernel, P) == cudaSuccess ? DG_OK : DG_ERR_CUDA;
}

}  // namespace dgf
