// Batched DG->Fourier projection / synthesis as one dense FP64 contraction (Eq. 63 and Eq. 71,
// PAPER.md:405-411, 459):  C[M][N] = A[M][K] * B[N][K]^T, all row-major with K contiguous
// (projection: A = rho[batch][G], B = T[2(pmax+1)][G];  synthesis: A = c[batch][Q], B = S[G][Q]).
// Register-tiled DFMA kernel: 128x128 CTA tile, 8x8 thread tile, BK = 8, register prefetch of the
// next k-tile.  FP64-pipe bound.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/dgvlasov.h"

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

inline int launch_gemm_tn(const double* A, const double* B, double* C, int M, int N, int K, cudaStream_t st) {
  const int tiles_m = (M + BM - 1) / BM, tiles_n = (N + BN - 1) / BN;
  const long long tiles = (long long)tiles_m * tiles_n;
  if (tiles <= 0 || tiles > 0x7fffffffLL) return DG_ERR_INVALID_ARG;
  const int vec = (K % 2 == 0) && ((reinterpret_cast<uintptr_t>(A) & 15) == 0) && ((reinterpret_cast<uintptr_t>(B) & 15) == 0);
  field_gemm_tn_kernel<<<(unsigned)tiles, 256, 0, st>>>(A, B, C, M, N, K, vec);
  return DG_OK;
}

}  // namespace dgf
