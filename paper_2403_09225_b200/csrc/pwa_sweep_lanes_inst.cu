// pwa_sweep_lanes_inst.cu - instantiates the lanes sweep kernel for ONE helicity count (-DPWA_LANES_H=1..4), so that
// the four counts compile in parallel (build.py).  The (RHO, LOG_SW, NW) table must match kLanesCombos in pwa_internal.h.
#include "pwa_internal.h"
#include "pwa_batch.cuh"
#include "pwa_sweep_pair.cuh"

#ifndef PWA_LANES_H
#error "compile with -DPWA_LANES_H=<n_hel>"
#endif

namespace pwa {
namespace {
template <int RHO, int LOG_SW, int NW, int PROD = 0, int TILE = 32>
lanes_fn for_mode(int mode) {
  switch (mode) {
    case MODE_NLL: return lanes::k_sweep_lanes<PWA_LANES_H, RHO, LOG_SW, NW, MODE_NLL, PROD, TILE>;
    case MODE_GRAD: return lanes::k_sweep_lanes<PWA_LANES_H, RHO, LOG_SW, NW, MODE_GRAD, PROD, TILE>;
    case MODE_GRAD3: return lanes::k_sweep_lanes<PWA_LANES_H, RHO, LOG_SW, NW, MODE_GRAD3, PROD, TILE>;
    case MODE_HVPQ: return lanes::k_sweep_lanes<PWA_LANES_H, RHO, LOG_SW, NW, MODE_HVPQ, PROD, TILE>;
    default: return lanes::k_sweep_lanes<PWA_LANES_H, RHO, LOG_SW, NW, MODE_FULL, PROD, TILE>;
  }
}
}  // namespace

#define PWA_CAT2(a, b) a##b
#define PWA_CAT(a, b) PWA_CAT2(a, b)
lanes_fn PWA_CAT(lanes_kernel_h, PWA_LANES_H)(int combo, int mode) {
  switch (combo) {
    case 0: return for_mode<1, 2, 15>(mode);
    case 1: return for_mode<2, 3, 15>(mode);
    case 2: return for_mode<3, 2, 11>(mode);
    case 3: return for_mode<3, 2, 8, 2>(mode);
    case 4: return for_mode<4, 3, 8, 2>(mode);
    case 5: return for_mode<4, 3, 7>(mode);
    case 6: return for_mode<4, 4, 8, 2>(mode);
    case 7: return for_mode<4, 4, 7>(mode);
    case 8: return for_mode<4, 5, 8, 2>(mode);
    case 9: return for_mode<4, 5, 7>(mode);
    case 10: return for_mode<4, 4, 8, 2, 8>(mode);
    case 11: return for_mode<4, 5, 8, 2, 8>(mode);
    case 12: return for_mode<4, 3, 11, 3>(mode);
    case 13: return for_mode<5, 1, 8, 2>(mode);
    case 14: return for_mode<4, 4, 8, 4, 8>(mode);
    case 15: return for_mode<4, 5, 8, 4, 8>(mode);
    case 16: return for_mode<3, 1, 8, 2>(mode);
    case 17: return for_mode<4, 1, 8, 2>(mode);
    case 18: return for_mode<5, 2, 8, 2>(mode);
    case 19: return for_mode<3, 4, 8, 2>(mode);
    case 20: return for_mode<6, 0, 8, 2>(mode);
    case 21: return for_mode<3, 3, 8, 2>(mode);
    case 22: return for_mode<3, 4, 8, 2, 8>(mode);
    case 23: return for_mode<3, 4, 8, 4, 8>(mode);
    case 24: return for_mode<3, 5, 8, 2, 8>(mode);
    case 25: return for_mode<3, 5, 8, 4, 8>(mode);
  }
  return nullptr;
}

// two events per lane (pwa_sweep_pair.cuh): the fused sweep of the (4 x 8 slices) shape, H <= 2 (two events' G fit the registers)
pair_fn PWA_CAT(pair_kernel_h, PWA_LANES_H)(int mode) {
#if PWA_LANES_H <= 2
  switch (mode) {
    case MODE_FULLP: return lanes::k_sweep_pair<PWA_LANES_H, MODE_FULLP>;
    case MODE_GRAD3: return lanes::k_sweep_pair<PWA_LANES_H, MODE_GRAD3>;
    case MODE_HVPQ: return lanes::k_sweep_pair<PWA_LANES_H, MODE_HVPQ>;
    case MODE_GRAD: return lanes::k_sweep_pair<PWA_LANES_H, MODE_GRAD>;
    case MODE_NLL: return lanes::k_sweep_pair<PWA_LANES_H, MODE_NLL>;
  }
#endif
  (void)mode;
  return nullptr;
}

// batch kernels (pwa_batch.cuh): only the warpgroup shapes (8 compute warps, 32-event tiles); kb: sets / directions per pass
namespace {
template <int RHO, int LOG_SW>
batch_fn batch_for(int kind, int kb) {
  if (kind == BK_NLL) {
    if (kb == 2) return lanes::k_batch_lanes<PWA_LANES_H, RHO, LOG_SW, 8, BK_NLL, 2>;
    if (kb == 4) return lanes::k_batch_lanes<PWA_LANES_H, RHO, LOG_SW, 8, BK_NLL, 4>;
  } else {
    if (kb == 2) return lanes::k_batch_lanes<PWA_LANES_H, RHO, LOG_SW, 8, BK_HVPQ, 2>;
    if (kb == 3) return lanes::k_batch_lanes<PWA_LANES_H, RHO, LOG_SW, 8, BK_HVPQ, 3>;
  }
  return nullptr;
}
}  // namespace
batch_fn PWA_CAT(batch_kernel_h, PWA_LANES_H)(int rho, int log_sw, int kind, int kb) {
  if (rho == 5 && log_sw == 1) return batch_for<5, 1>(kind, kb);
  if (rho == 3 && log_sw == 1) return batch_for<3, 1>(kind, kb);
  if (rho == 4 && log_sw == 1) return batch_for<4, 1>(kind, kb);
  if (rho == 5 && log_sw == 2) return batch_for<5, 2>(kind, kb);
  if (rho == 3 && log_sw == 3) return batch_for<3, 3>(kind, kb);
  if (rho == 3 && log_sw == 2) return batch_for<3, 2>(kind, kb);
  if (rho == 4 && log_sw == 3) return batch_for<4, 3>(kind, kb);
  // 16 or 32 slices (R > 32) leave fewer passes per tile than warps: no fixed column; those shapes take single passes
  return nullptr;
}
}  // namespace pwa
