// pwa_sweep_lanes_inst.cu - instantiates the lanes sweep kernel for ONE helicity count (-DPWA_LANES_H=1..4), so that
// the four counts compile in parallel (build.py).  The (RHO, LOG_SW, NW) table must match kLanesCombos in pwa_internal.h.
#include "pwa_internal.h"

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
  }
  return nullptr;
}
}  // namespace pwa
