// FFT-factorised DG -> Fourier projection and spectral Poisson solve for equal-width elements.
//
// The paper concedes that its dense transform "does not beat" the DFT and notes that for piecewise
// constants it *is* the DFT.  With N equal-width elements the element-centre phase of Eq. 63
// is e^{-i k_p xbar_m} = e^{-i(k_p lo + pi p/N)} e^{-2 pi i p m / N}, so
//
//   c_p    = sum_j A_p^j X_j[p mod N],      X_j[q] = sum_m rho_{mj} e^{-2 pi i q m / N}   (n DFTs of length N)
//   A_p^j  = (1/N) e^{-i(k_p lo + pi p/N)} w_j sum_s gamma_s^{-1} (-i)^s P_s(xi_j) j_s(k_p dx/2)
//
// and the synthesis of Eq. 71 at x_mj = xbar_m + xi_j dx/2 folds the kept modes onto N bins:
//
//   E_mj   = 2 Re sum_q Y_j[q] e^{2 pi i q m / N},   Y_j[q] = sum_{p = q (mod N), 1 <= p <= pmax} D_p^j c_p
//   D_p^j  = (i/k_p) e^{i(k_p lo + pi p/N)} e^{i k_p xi_j dx/2}            (Phi: one more factor i/k_p, Eq. 70)
//
// Same numbers as the dense contraction with T and S up to rounding order; (pmax+1) n N complex MACs become
// n N log N + (pmax+1) n, and the 2 x 2.15 GB operators of config 5 become a 2 MB table.
//
// One CTA holds one density vector in shared memory.  Two real node sequences (j = 2k, 2k+1: adjacent doubles of
// rho, i.e. one 128-bit load) ride one complex FFT: z_k[m] = rho_{m,2k} + i rho_{m,2k+1}.  Forward = in-place
// decimation in frequency (natural in, bit-reversed out), the mode combination works on bit-reversed bins in
// place, inverse = in-place decimation in time (bit-reversed in, natural out); Re/Im of the result are
// E_{m,2k}, E_{m,2k+1}: one 128-bit store.  Up to three radix-2 stages are fused in registers per pass.
#pragma once
#include "dg_context.hpp"
#include <cuda_runtime.h>
#include <cstdint>

namespace dgfft {

struct FftParams {
  const double* rho;    // [batch][N*n]
  double* c;            // [batch][P1][2]  (nullptr: not wanted)
  double* out;          // [batch][N*n]    E or Phi (nullptr: projection only)
  const double2* AD;    // [n+1][P1]       rows B_p^j (j < n/2), u_p^j/(k_p N) (j < n/2), a_p; p fastest (lanes walk p: coalesced)
  const double2* W;     // [N/2]           e^{-2 pi i k / N}
  int N, logN, P1, batch;
  int phi;              // 1: potential (Eq. 70) instead of field (Eq. 71)
  double kinv;          // L / (2 pi): 1/k_p = kinv / p
};

constexpr int FFT_THREADS = 512;

// Shared-memory slot of element i of array k.  A 16-byte element occupies one of 8 bank groups; the group is the XOR
// of all 3-bit digits of i (and of 2k), so any 8 lanes that differ in three index bits at distinct positions mod 3 --
// unit stride, the strides 2^lh of every radix pass, and the bit-reversed order of the mode combination -- hit 8
// different groups.  No padding.
__host__ __device__ __forceinline__ int phys(int i, int kx) {
  int x = i ^ (i >> 3);
  x ^= x >> 6;
  return (i & ~7) | ((x ^ kx) & 7);
}
__host__ __device__ inline int arr_stride(int N) { return N < 8 ? 8 : N; }
inline size_t fft_smem_bytes(int N, int NP) { return sizeof(double2) * ((size_t)NP * arr_stride(N) + (N / 2 < 8 ? 8 : N / 2)); }

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 cmulc(double2 a, double2 bconj) {   // a * conj(b)
  return make_double2(fma(a.x, bconj.x, a.y * bconj.y), fma(a.y, bconj.x, -a.x * bconj.y));
}

// XOR of the 3-bit digits of i (the bank-group part of phys): linear over GF(2), so for index parts with disjoint bits
// digits(a + b) = digits(a) ^ digits(b) -- the passes below fold the thread-invariant parts once.
__host__ __device__ __forceinline__ int digits(int i) {
  int x = i ^ (i >> 3);
  x ^= x >> 6;
  return x & 7;
}

// One pass of R fused radix-2 stages over all NP arrays.  lh = log2 of the smallest half-size of the pass.
// Element t of a work item sits at base + (t << lh) with base's bits disjoint from t's, so its slot is
// ((base + (t << lh)) & ~7) | (digits(base) ^ digits(t << lh) ^ kx): one digit fold per item, the t part per pass.
template <int R, bool INV>
__device__ __forceinline__ void fft_pass(double2* z, const double2* Ws, int N, int logN, int lh, int NP, int stride, int tid) {
  constexpr int M = 1 << R;
  const int lg = logN - R, h = 1 << lh;           // 2^lg work items per array
  int dt[M];                                     // digits(t << lh): the same for every thread
#pragma unroll
  for (int t = 0; t < M; ++t) dt[t] = digits(t << lh);
#pragma unroll 2
  for (int item = tid; item < (NP << lg); item += FFT_THREADS) {
    const int k = item >> lg, g = item & ((1 << lg) - 1);
    const int blk = g >> lh, i0 = g & (h - 1);
    const int base = (blk << (lh + R)) + i0;
    double2* za = z + (size_t)k * stride;
    const int db = digits(base) ^ ((2 * k) & 7);
    int slot[M];
#pragma unroll
    for (int t = 0; t < M; ++t) slot[t] = ((base + (t << lh)) & ~7) | (db ^ dt[t]);
    double2 e[M];
#pragma unroll
    for (int t = 0; t < M; ++t) e[t] = za[slot[t]];
#pragma unroll
    for (int s = 0; s < R; ++s) {
      const int lt = INV ? s : (R - 1 - s);          // log2 of the half-size of this stage in units of t
      const int half_t = 1 << lt;
      const int shift = logN - 1 - (lh + lt);        // twiddle stride N / (2 hs)
      const int wi0 = i0 << shift, dw0 = digits(wi0);
#pragma unroll
      for (int t = 0; t < M; ++t) {
        if (t & half_t) continue;
        // twiddle index (i0 + (tt << lh)) << shift, tt = t mod half_t: again two disjoint parts
        const int wt = (t & (half_t - 1)) << (lh + shift);
        const double2 w = Ws[((wi0 + wt) & ~7) | (dw0 ^ digits(wt))];
        const double2 a = e[t];
        if (!INV) {
          const double2 b = e[t + half_t];
          e[t] = make_double2(a.x + b.x, a.y + b.y);
          e[t + half_t] = cmul(make_double2(a.x - b.x, a.y - b.y), w);
        } else {
          const double2 b = cmulc(e[t + half_t], w);
          e[t] = make_double2(a.x + b.x, a.y + b.y);
          e[t + half_t] = make_double2(a.x - b.x, a.y - b.y);
        }
      }
    }
#pragma unroll
    for (int t = 0; t < M; ++t) za[slot[t]] = e[t];
  }
}

template <bool INV>
__device__ __forceinline__ void fft_all(double2* z, const double2* Ws, int N, int logN, int NP, int stride, int tid) {
  int rem = logN;
  int lh = INV ? 0 : logN;          // forward: passes walk down from the largest half N/2; inverse: up from 1
  while (rem > 0) {
    const int R = rem >= 3 ? 3 : rem;
    if (!INV) lh -= R;
    if (R == 3) fft_pass<3, INV>(z, Ws, N, logN, lh, NP, stride, tid);
    else if (R == 2) fft_pass<2, INV>(z, Ws, N, logN, lh, NP, stride, tid);
    else fft_pass<1, INV>(z, Ws, N, logN, lh, NP, stride, tid);
    if (INV) lh += R;
    rem -= R;
    __syncthreads();
  }
}

// Mode combination for bin q (and its mirror N-q unless q is its own mirror): reads the packed spectra at the
// bit-reversed slots, writes c_p for every kept p = q, N-q (mod N), and leaves the packed Hermitian input of the
// inverse transform in the same slots.
//
// The LGL nodes are symmetric (xi_{n-1-j} = -xi_j, w symmetric), so B_p^{n-1-j} = conj B_p^j and u_p^{n-1-j} =
// conj u_p^j with  A_p^j = a_p B_p^j,  D_p^j = (i/k_p) conj(N a_p) u_p^j,  a_p = e^{-i(k_p lo + pi p/N)} / N:
//   s_p = sum_{j<n/2} ( B_p^j X_j + conj(B_p^j) X_{n-1-j} ),   c_p = a_p s_p,
//   D_p^j c_p = i u_p^j s_p / (k_p N)            (|a_p| = 1/N: the centre phase cancels between T and S; the table
//                                                 row holds u_p^j / (k_p N), zero at p = 0)
// i.e. n/2 + n/2 table entries per mode (+ a_p only when c_p itself is wanted) and 4 FMAs per node pair each way.
template <int NP>
__device__ __forceinline__ void combine_bin(const FftParams& P, double2* z, int stride, int b, int q) {
  constexpr int n = 2 * NP;
  const int N = P.N;
  const int qm = (N - q) & (N - 1);
  const bool self = (qm == q);
  const int sq = (int)(__brev((unsigned)q) >> (32 - P.logN));
  const int sm = (int)(__brev((unsigned)qm) >> (32 - P.logN));
  // node pair (j, n-1-j), j < NP: sums and differences of X_j[q] and X_{n-1-j}[q]
  double Sx[NP], Dx[NP], Sy[NP], Dy[NP];
  {
    double2 X[n];
#pragma unroll
    for (int k = 0; k < NP; ++k) {
      const double2 a = z[(size_t)k * stride + phys(sq, 2 * k)], m = z[(size_t)k * stride + phys(sm, 2 * k)];
      X[2 * k] = make_double2(0.5 * (a.x + m.x), 0.5 * (a.y - m.y));          // (Z[q] + conj Z[N-q]) / 2
      X[2 * k + 1] = make_double2(0.5 * (a.y + m.y), -0.5 * (a.x - m.x));     // (Z[q] - conj Z[N-q]) / (2i)
    }
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      Sx[j] = X[j].x + X[n - 1 - j].x; Dx[j] = X[j].x - X[n - 1 - j].x;
      Sy[j] = X[j].y + X[n - 1 - j].y; Dy[j] = X[j].y - X[n - 1 - j].y;
    }
  }
  // H_j[q] +- H_{n-1-j}[q] accumulate as sums (HS) and differences (HD)
  double HSx[NP], HSy[NP], HDx[NP], HDy[NP];
#pragma unroll
  for (int j = 0; j < NP; ++j) { HSx[j] = 0.0; HSy[j] = 0.0; HDx[j] = 0.0; HDy[j] = 0.0; }
  double2* cb = P.c ? reinterpret_cast<double2*>(P.c) + (size_t)b * P.P1 : nullptr;
#pragma unroll 1
  for (int side = 0; side < 2; ++side) {
    if (side == 1 && self) break;
    const double sg = side ? -1.0 : 1.0;             // side 1: X_j[N-q] = conj X_j[q] (rho is real)
    for (int p = side ? qm : q; p < P.P1; p += N) {
      const double2* tb = P.AD + p;
      // all table rows of this mode in flight together (one L2 latency per mode, not one per use)
      double2 B[NP], U[NP];
#pragma unroll
      for (int j = 0; j < NP; ++j) B[j] = __ldg(tb + (size_t)j * P.P1);
      if (P.out) {
#pragma unroll
        for (int j = 0; j < NP; ++j) U[j] = __ldg(tb + (size_t)(NP + j) * P.P1);
      }
      double sx = 0.0, sy = 0.0;
#pragma unroll
      for (int j = 0; j < NP; ++j) {
        sx = fma(B[j].x, Sx[j], fma(-sg * B[j].y, Dy[j], sx));
        sy = fma(sg * B[j].x, Sy[j], fma(B[j].y, Dx[j], sy));
      }
      if (cb) {
        const double2 a = __ldg(tb + (size_t)n * P.P1);
        cb[p] = make_double2(fma(a.x, sx, -a.y * sy), fma(a.x, sy, a.y * sx));
      }
      if (P.out) {
        double cx = -sy, cy = sx;                    // i s_p; the real factor 1/(k_p N) rides in the u table
        if (P.phi) {                                 // Phi~_p = E~_p (i/k_p)  (Eq. 70 vs Eq. 71)
          const double g = P.kinv / (double)(p ? p : 1);
          const double t = cx; cx = -cy * g; cy = t * g;
        }
        cy *= sg;                                    // side 1 contributes conj(Y_j[N-q]) to bin q: u c -> conj(u) conj(c)
        const double us = sg;
#pragma unroll
        for (int j = 0; j < NP; ++j) {
          const double2 u = U[j];
          const double ui = us * u.y;
          // u c = (ur cx - ui cy) + i(ur cy + ui cx);  conj(u) c = (ur cx + ui cy) + i(ur cy - ui cx)
          HSx[j] = fma(u.x, cx, HSx[j]); HSy[j] = fma(u.x, cy, HSy[j]);
          HDx[j] = fma(-ui, cy, HDx[j]); HDy[j] = fma(ui, cx, HDy[j]);
        }
      }
    }
  }
  if (P.out) {
    double2 H[n];
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      H[j] = make_double2(HSx[j] + HDx[j], HSy[j] + HDy[j]);
      H[n - 1 - j] = make_double2(HSx[j] - HDx[j], HSy[j] - HDy[j]);
    }
#pragma unroll
    for (int k = 0; k < NP; ++k) {
      double2 h0 = H[2 * k], h1 = H[2 * k + 1];
      if (self) { h0 = make_double2(2.0 * h0.x, 0.0); h1 = make_double2(2.0 * h1.x, 0.0); }     // Y + conj Y
      z[(size_t)k * stride + phys(sq, 2 * k)] = make_double2(h0.x - h1.y, h0.y + h1.x);            // H_2k + i H_2k+1
      if (!self) z[(size_t)k * stride + phys(sm, 2 * k)] = make_double2(h0.x + h1.y, h1.x - h0.y); // conj H_2k + i conj H_2k+1
    }
  }
}

template <int NP>
__global__ void __launch_bounds__(FFT_THREADS, 1) field_fft_kernel(const FftParams P) {
  extern __shared__ double2 fft_sm[];
  const int N = P.N, stride = arr_stride(N), tid = threadIdx.x;
  double2* z = fft_sm;
  double2* Ws = fft_sm + (size_t)NP * stride;
  for (int i = tid; i < N / 2; i += FFT_THREADS) Ws[phys(i, 0)] = P.W[i];
  for (int b = blockIdx.x; b < P.batch; b += gridDim.x) {
    const double2* src = reinterpret_cast<const double2*>(P.rho + (size_t)b * N * 2 * NP);
    for (int e = tid; e < N * NP; e += FFT_THREADS) {
      const int m = e / NP, k = e - m * NP;
      z[(size_t)k * stride + phys(m, 2 * k)] = __ldcs(src + e);
    }
    __syncthreads();
    fft_all<false>(z, Ws, N, P.logN, NP, stride, tid);
    // bins q = 0 .. N/2 (q and N-q together); lanes walk q, so the table loads and the c_p stores coalesce
    for (int q = tid; q < N / 2; q += FFT_THREADS) {
      combine_bin<NP>(P, z, stride, b, q);
      if (q == 0) combine_bin<NP>(P, z, stride, b, N / 2);
    }
    __syncthreads();
    if (P.out) {
      fft_all<true>(z, Ws, N, P.logN, NP, stride, tid);
      double2* dst = reinterpret_cast<double2*>(P.out + (size_t)b * N * 2 * NP);
      for (int e = tid; e < N * NP; e += FFT_THREADS) {
        const int m = e / NP, k = e - m * NP;
        __stcs(dst + e, z[(size_t)k * stride + phys(m, 2 * k)]);
      }
      __syncthreads();
    }
  }
}

// N a power of two >= 2, even order n in {2,...,10}, one vector fits in shared memory
inline bool fft_supported(int N, int n) {
  if (N < 2 || (N & (N - 1)) != 0 || (n & 1) || n < 2 || n > 10) return false;
  return fft_smem_bytes(N, n / 2) <= 200 * 1024;
}

template <int NP>
inline int launch_fft_t(const FftParams& P, int sms, cudaStream_t st) {
  const size_t smem = fft_smem_bytes(P.N, NP);
  if (ensure_dyn_smem(reinterpret_cast<const void*>(field_fft_kernel<NP>), smem) != cudaSuccess) return -3;
  int per_sm = (int)((220 * 1024) / (smem + 1024));
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 4) per_sm = 4;
  int grid = sms * per_sm;
  if (grid > P.batch) grid = P.batch;
  field_fft_kernel<NP><<<grid, FFT_THREADS, smem, st>>>(P);
  return 0;
}

inline int launch_fft(const FftParams& P, int n, int sms, cudaStream_t st) {
  switch (n) {
    case 2: return launch_fft_t<1>(P, sms, st);
    case 4: return launch_fft_t<2>(P, sms, st);
    case 6: return launch_fft_t<3>(P, sms, st);
    case 8: return launch_fft_t<4>(P, sms, st);
    case 10: return launch_fft_t<5>(P, sms, st);
    default: return -2;
  }
}

}  // namespace dgfft
