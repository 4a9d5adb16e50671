// The Shu-Osher SSP-RK3 step (reading C3), written once for every phase-space dimension:
//   u1 = u + dt L(u);   u2 = 3/4 u + 1/4 (u1 + dt L(u1));   u <- 1/3 u + 2/3 (u2 + dt L(u2))  (in place)
// with the field solved from each stage's INPUT when the run is self-consistent (reading C4).  dg_ssprk3_run (1D1V / 1D2V)
// and dg4_ssprk3_run (2D2V) pass their own field solve and fused RHS + stage launch; the stage table and the order of the
// stages live here and in dg_ssprk3_stage_coeffs only.
#pragma once
#include "../../include/dgvlasov.h"

// field(src)                         -> int   field of the stage input `src` (only called when self_consistent)
// stage(k, src, fn, dst, c0, c1)     -> int   dst = c0 fn + c1 (src + dt L(src)); fn == nullptr when c0 == 0; k = 0, 1, 2
template <class FieldFn, class StageFn>
int ssprk3_run_loop(double* f, double* u1, double* u2, int nsteps, bool self_consistent, FieldFn&& field, StageFn&& stage) {
  const double* src[3] = {f, u1, u2};
  const double* fn[3] = {nullptr, f, f};
  double* dst[3] = {u1, u2, f};             // stage 3 writes u in place: each node of u is read and written by one thread
  for (int s = 0; s < nsteps; ++s) {
    for (int k = 0; k < 3; ++k) {
      int rc;
      if (self_consistent) { rc = field(src[k]); if (rc) return rc; }
      double c0, c1;
      dg_ssprk3_stage_coeffs(k, &c0, &c1);
      rc = stage(k, src[k], fn[k], dst[k], c0, c1);
      if (rc) return rc;
    }
  }
  return DG_OK;
}
