// dg_density_static (include/dgvlasov_noalloc.h): the density moment of Eq. 27 for callers that may not
// allocate device memory -- no context, no workspace.  The partial sums that dg_density keeps in the caller's
// workspace sit in the file-scope device array below instead.  A translation unit of its own: the array is `static`,
// so the host code that asks for its device address has to be in this file.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>
#include <string>

#include "../../include/dgvlasov_noalloc.h"

int dg_internal_fail(int code, const char* msg);      // dg_api.cu: the per-thread message behind dg_last_error()

namespace dgs {

// The scratch: partial[g_x][chunk], at most DG_STATIC_MAX_CHUNKS chunks per x node.  2 MiB on every GPU that loads this
// module, for the life of the process.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a
// device pointer and must never be handed to a kernel as one (see scratch_address below).
static __device__ __align__(256) double g_density_partials[(size_t)DG_STATIC_MAX_GX * DG_STATIC_MAX_CHUNKS];

constexpr int kMaxDevices = 64;
static std::mutex g_mu;
static double* g_scratch_dev[kMaxDevices];            // device address of g_density_partials per ordinal, nullptr = not yet asked

// Device address of the scratch array on the CURRENT device; looked up once per device and cached.
static int scratch_address(int device, double** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_dev[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_density_partials);
    if (e != cudaSuccess || !p)
      return dg_internal_fail(DG_ERR_CUDA, (std::string("dg_density_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e)).c_str());
    g_scratch_dev[device] = static_cast<double*>(p);
  }
  *out = g_scratch_dev[device];
  return DG_OK;
}

// Makes `device` current for the duration of the call and puts the caller's device back; a failed switch is an error.
struct ScopedDevice {
  int prev = -1;
  bool switched = false;
  cudaError_t err = cudaSuccess;
  explicit ScopedDevice(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) { err = cudaSetDevice(dev); switched = (err == cudaSuccess); }
  }
  ~ScopedDevice() { if (switched) cudaSetDevice(prev); }
};

// partial[g_x][chunk] = sum over rows [r0, r1) of the velocity plane of wq_u[r] * (sum_c wq_v[c] f[g_x][r][c]).
// grid = (chunks, G_x), 256 threads = 8 warps; warp w takes rows r0 + w, r0 + w + 8, ...; the lanes stride over the
// columns (two at a time with 128-bit loads when VEC).  Fixed association throughout: the same inputs give the same bits.
template <bool VEC>
__global__ void __launch_bounds__(256) density_partial_static_kernel(const double* __restrict__ f, const double* __restrict__ wq_u,
                                                                     const double* __restrict__ wq_v, int G_u, int G_v,
                                                                     int rows_per_chunk, double* __restrict__ partial) {
  __shared__ double warp_sum[8];
  const int gx = blockIdx.y, chunk = blockIdx.x, nchunks = gridDim.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r0 = chunk * rows_per_chunk;
  const int r1 = min(G_u, r0 + rows_per_chunk);
  const double* plane = f + (size_t)gx * G_u * G_v;
  double acc = 0.0;
  for (int r = r0 + warp; r < r1; r += 8) {
    const double* row = plane + (size_t)r * G_v;
    double a0 = 0.0, a1 = 0.0;
    if (VEC) {
      const double2* row2 = reinterpret_cast<const double2*>(row);
      const double2* w2 = reinterpret_cast<const double2*>(wq_v);
      const int npair = G_v >> 1;
#pragma unroll 4
      for (int c = lane; c < npair; c += 32) {
        const double2 v = __ldcs(row2 + c);
        const double2 w = w2[c];
        a0 = fma(w.x, v.x, a0);
        a1 = fma(w.y, v.y, a1);
      }
    } else {
#pragma unroll 4
      for (int c = lane; c < G_v; c += 32) a0 = fma(wq_v ? wq_v[c] : 1.0, row[c], a0);
    }
    acc = fma(wq_u[r], a0 + a1, acc);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
  if (lane == 0) warp_sum[warp] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) tot += warp_sum[w];
    partial[(size_t)gx * nchunks + chunk] = tot;
  }
}

// rho[g_x] = partial[g_x][0] + partial[g_x][1] + ... in index order.  One thread per x node (at most 16 terms).
__global__ void __launch_bounds__(128) density_finish_static_kernel(const double* __restrict__ partial, int nchunks, int G_x,
                                                                    double* __restrict__ rho) {
  const int gx = blockIdx.x * 128 + threadIdx.x;
  if (gx >= G_x) return;
  double tot = 0.0;
  for (int c = 0; c < nchunks; ++c) tot += partial[(size_t)gx * nchunks + c];
  rho[gx] = tot;
}

}  // namespace dgs

extern "C" int dg_density_static(const double* f_dev, int32_t G_x, int32_t G_u, int32_t G_v, const double* wq_u_dev,
                                 const double* wq_v_dev, double* rho_dev, int32_t device, void* stream) {
  if (!f_dev || !wq_u_dev || !rho_dev) return dg_internal_fail(DG_ERR_INVALID_ARG, "dg_density_static: null f, wq_u or rho");
  if (G_x < 1 || G_u < 1 || G_v < 1) return dg_internal_fail(DG_ERR_INVALID_ARG, "dg_density_static: G_x, G_u, G_v must be >= 1");
  if (!wq_v_dev && G_v != 1) return dg_internal_fail(DG_ERR_INVALID_ARG, "dg_density_static: wq_v may be NULL only when G_v = 1");
  if (G_x > DG_STATIC_MAX_GX)
    return dg_internal_fail(DG_ERR_UNSUPPORTED, ("dg_density_static: G_x = " + std::to_string(G_x) + " exceeds DG_STATIC_MAX_GX = " +
                                                 std::to_string(DG_STATIC_MAX_GX) + " (the built-in scratch holds no more x nodes); "
                                                 "use dg_density with a workspace").c_str());
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess) return dg_internal_fail(DG_ERR_CUDA, (std::string("dg_density_static: cudaGetDeviceCount: ") + cudaGetErrorString(e)).c_str());
  if (device < 0 || device >= ndev || device >= dgs::kMaxDevices) return dg_internal_fail(DG_ERR_INVALID_ARG, "dg_density_static: no such device");
  dgs::ScopedDevice guard(device);
  if (guard.err != cudaSuccess) return dg_internal_fail(DG_ERR_CUDA, (std::string("dg_density_static: cudaSetDevice: ") + cudaGetErrorString(guard.err)).c_str());

  // set-up on the first call per device (with that device current): the device address of the static array
  double* partial = nullptr;
  if (int rc = dgs::scratch_address(device, &partial)) return rc;

  // chunks of u rows per x node: enough CTAs to fill 148 SMs several times over, never more than the scratch has room for
  int nchunks = (148 * 16 + G_x - 1) / G_x;
  if (nchunks > DG_STATIC_MAX_CHUNKS) nchunks = DG_STATIC_MAX_CHUNKS;
  if (nchunks > G_u) nchunks = G_u;
  const int rows = (G_u + nchunks - 1) / nchunks;
  nchunks = (G_u + rows - 1) / rows;

  cudaStream_t st = (cudaStream_t)stream;
  const dim3 grid((unsigned)nchunks, (unsigned)G_x);
  const bool vec = wq_v_dev && G_v % 2 == 0 && ((uintptr_t)f_dev & 15) == 0 && ((uintptr_t)wq_v_dev & 15) == 0;
  if (vec) dgs::density_partial_static_kernel<true><<<grid, 256, 0, st>>>(f_dev, wq_u_dev, wq_v_dev, G_u, G_v, rows, partial);
  else dgs::density_partial_static_kernel<false><<<grid, 256, 0, st>>>(f_dev, wq_u_dev, wq_v_dev, G_u, G_v, rows, partial);
  e = cudaGetLastError();
  if (e != cudaSuccess) return dg_internal_fail(DG_ERR_CUDA, (std::string("dg_density_static: partial kernel: ") + cudaGetErrorString(e)).c_str());
  dgs::density_finish_static_kernel<<<(unsigned)((G_x + 127) / 128), 128, 0, st>>>(partial, nchunks, G_x, rho_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return dg_internal_fail(DG_ERR_CUDA, (std::string("dg_density_static: finish kernel: ") + cudaGetErrorString(e)).c_str());
  return DG_OK;
}
