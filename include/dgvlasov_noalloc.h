/* dgvlasov_noalloc.h -- the one entry point of libdgvlasov that never allocates device memory.
 *
 * Who this is for.  Every other compute call of the library needs a dg_ctx, and dg_create / dg_set_workspace mean a
 * cudaMalloc somewhere (inside the library for the operator tables, in the caller for the workspace).  Some callers
 * cannot do that at the point where they want a density:
 *   - a diagnostics hook that runs inside somebody else's time loop, where the host application has already handed
 *     all of the HBM to its own pool and a further cudaMalloc would simply fail;
 *   - a callback on a latency-critical path: cudaMalloc and cudaFree synchronise the whole device, so one call stalls
 *     every stream the application has in flight;
 *   - code running under a fixed memory quota (an MPS client limit, a MIG slice) that was sized without this library.
 * Such a caller passes its inputs and its output and nothing else: no context, no workspace.
 *
 * How.  The per-chunk partial sums of the reduction -- the scratch that dg_density keeps in the caller's workspace --
 * live in a fixed array compiled into the library (a file-scope `static __device__` array in
 * csrc/dg_density_static.cu) of DG_STATIC_MAX_GX * DG_STATIC_MAX_CHUNKS doubles = 2 MiB.  Every GPU on which the
 * library's device code gets loaded carries those 2 MiB until the process exits; that is the price of the entry point.
 *
 * Rules that follow from the shared array
 *   - Sizes: G_x <= DG_STATIC_MAX_GX.  Anything larger is refused with DG_ERR_UNSUPPORTED and a message naming the
 *     limit; nothing is launched.  G_u and G_v are unlimited (they only lengthen the sums).
 *   - First call per device: the call looks up the device address of the array (cudaGetSymbolAddress, with that
 *     device current, return code checked) and remembers it.  Make this first call on each device early, during
 *     start-up and outside any stream capture; later calls only launch two kernels.
 *   - One array for everybody: all calls on a device, from every thread and every stream, use the same scratch.
 *     Two calls whose kernels can overlap on the GPU (different streams, no event between them) race on it and
 *     both results are garbage.  Calls on one stream, or ordered by events, are safe.
 *   - Nothing to clear: the array keeps whatever the previous call left, but each call first writes every slot it
 *     later reads (G_x * chunks partials) and reads no other, so stale contents are never seen.
 *   - The call itself uses no cudaMalloc, cudaFree, cudaMemset or library routine that allocates; it only enqueues on
 *     `stream` and does not synchronise.
 */
#ifndef DGVLASOV_NOALLOC_H
#define DGVLASOV_NOALLOC_H

#include "dgvlasov.h"

#ifdef __cplusplus
extern "C" {
#endif

#define DG_STATIC_MAX_GX      16384   /* largest number of x nodes N_x*n_x the static scratch serves */
#define DG_STATIC_MAX_CHUNKS  16      /* partial sums per x node: 16384 * 16 doubles = 2 MiB per GPU */

/* Zeroth moment Eq. 27 by LGL quadrature, exactly what dg_density computes:
 *   rho[g_x] = sum_{g_u, g_v} wq_u[g_u] * wq_v[g_v] * f[g_x][g_u][g_v]
 *   f_dev     [in]  device, [G_x][G_u][G_v] row-major FP64 (the layout of dgvlasov.h); 1D1V: G_v = 1
 *   wq_u_dev  [in]  device, [G_u]: quadrature weight of each flat u node, w_b * (Delta u / 2) for node b of its element
 *   wq_v_dev  [in]  device, [G_v], same for v; may be NULL when G_v = 1 (weight 1)
 *   rho_dev   [out] device, [G_x]
 *   device    CUDA ordinal the pointers live on        stream    cudaStream_t as void* (NULL = default stream)
 * All four arrays are the caller's; the library keeps no pointer after the call.  Deterministic (fixed summation
 * order, no atomics); agrees with dg_density to rounding (the chunking differs, so not bit for bit).
 * Errors: DG_ERR_INVALID_ARG (null pointer, size < 1, no such device), DG_ERR_UNSUPPORTED (G_x above
 * DG_STATIC_MAX_GX), DG_ERR_CUDA (address look-up or launch failed); message through dg_last_error(). */
int dg_density_static(const double* f_dev, int32_t G_x, int32_t G_u, int32_t G_v, const double* wq_u_dev,
                      const double* wq_v_dev, double* rho_dev, int32_t device, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DGVLASOV_NOALLOC_H */
