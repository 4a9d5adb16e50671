// Tiled sm_100a fast path for the fused RHS + stage kernel (placeholder until the first GPU run of
// the generic path is green).
#pragma once
#include <cuda_runtime.h>
#include "dg_context.hpp"

namespace dgt {
inline const char* last_error() { return "tiled kernel not built"; }
inline bool tiled_supported(const dg_ctx*) { return false; }
inline int launch_rhs_tiled(dg_ctx*, const double*, const double*, const double*, double*, int, double, double, double,
                            bool, int*, cudaStream_t) { return DG_ERR_UNSUPPORTED; }
}  // namespace dgt
