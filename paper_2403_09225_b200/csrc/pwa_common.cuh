// pwa_common.cuh - shared device-side definitions of the PWA likelihood kernels (sm_100a).
//
// Notation follows DESIGN.md / include/pwa.h:  theta[4r..4r+3] = (a, phi, M, Gamma);
//   c = a e^{i phi};  D = (M^2 - m^2) - i M Gamma;  B = 1/D;  z = c B;
//   A_h = sum_r z_r F_rh;  I = sum_h |A_h|^2                         (Eq. 1)
// and, along a direction v (Eq. 7):
//   zdot = alpha B + beta B^2,  alpha = e^{i phi} v_a + i c v_phi,  beta = c (-(2M - i Gamma) v_M + i M v_Gamma)
//   Adot_h = sum_r zdot_r F_rh;  Idot = 2 Re sum_h conj(A_h) Adot_h.
// Per event and resonance the kernels accumulate the five complex "compact" sums
//   P1 = sum w B S, P2 = sum w B^2 S, P3 = sum w B^3 S, Q1 = sum w B S', Q2 = sum w B^2 S'
//   S = sum_h conj(A_h) F_rh,  S' = sum_h conj(Adot_h - kappa A_h) F_rh,
//   (MC: w = 1, kappa = 0;  data: w = weight/I, kappa = Idot/I)
// from which the finalize step forms every theta- and v-dependent factor once.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pwa {

// per-resonance constants produced by the prologue kernel; KSTRIDE doubles per resonance
constexpr int KSTRIDE = 12;
enum { K_M2 = 0, K_Y2 = 1, K_Y = 2, K_CR = 4, K_CI = 5, K_AR = 6, K_AI = 7, K_BR = 8, K_BI = 9 };

// MODE_GRAD3 and MODE_HVPQ split the fused sweep for Newton-CG: at a fixed theta the compact sums
// P1, P2, P3 do not depend on the direction v, so the gradient evaluation of an outer iteration keeps them (GRAD3) and
// every CG iteration only accumulates Q1, Q2 (HVPQ): 49 instead of 69 FP64 instructions per (event, resonance).
// MODE_FULLP: the fused sweep with P3 folded into Q2 (pwa_sweep_pair.cuh): P1, P2, Q1, Q2' = Q2 + 2 lambda P3 per resonance
enum Mode { MODE_NLL = 0, MODE_GRAD = 1, MODE_FULL = 2, MODE_GRAD3 = 3, MODE_HVPQ = 4, MODE_FULLP = 5 };
__host__ __device__ constexpr bool mode_p(int m) { return m == MODE_GRAD || m == MODE_FULL || m == MODE_GRAD3 || m == MODE_FULLP; }   // P1, P2
__host__ __device__ constexpr bool mode_p3(int m) { return m == MODE_FULL || m == MODE_GRAD3; }                     // P3
__host__ __device__ constexpr bool mode_q(int m) { return m == MODE_FULL || m == MODE_HVPQ || m == MODE_FULLP; }  // Adot, Q1, Q2 (needs v)

// values per resonance that the backward pass produces, and resonances per 32-value batch
__host__ __device__ constexpr int vpr_of(int mode) { return mode == MODE_FULL ? 10 : (mode == MODE_FULLP ? 8 : (mode == MODE_GRAD3 ? 6 : 4)); }
__host__ __device__ constexpr int rpb_of(int mode) { return mode == MODE_FULL ? 3 : 8; }

struct SampleDev {
  const double* mass;    // [C][stride]
  const double2* amp;    // [R][H][stride]
  const double* weight;  // [n] or nullptr
  long long n, stride;
};

// Library-owned TILED event store (copy-mode handles whose shape needs 8-event tiles, e.g. R = 100, H = 4): tile t holds
// the events 8t .. 8t+7 in ONE contiguous block of tile_bytes, laid out exactly as a stage of the sweep's ring -
//   [resonance r][helicity h][8 events x (re, im)]  128-byte rows, the 16-byte chunk of event e at position e ^ phase(r),
//                                                   phase(r) = (r * phase_mul) & 7   (bank-conflict-free reads)
//   [channel c][8 events]                           masses, at off_mass
//   [8 events]                                      weights (zeros when the sample has none), at off_wgt
// so that one bulk copy (cp.async.bulk) of contiguous HBM fills a stage.  Events beyond n are zero.
struct TiledDev {
  const unsigned char* base;
  long long n;
  unsigned tile_bytes, off_mass, off_wgt;
  int H, phase_mul;
  bool weighted;
};
__host__ __device__ inline size_t tiled_amp_off(const TiledDev& t, int r, int h, long long i) {
  const unsigned e = (unsigned)(i & 7), ph = (unsigned)(r * t.phase_mul) & 7u;
  return (size_t)(i >> 3) * t.tile_bytes + ((size_t)r * t.H + h) * 128 + ((e ^ ph) << 4);
}
__host__ __device__ inline size_t tiled_mass_off(const TiledDev& t, int c, long long i) {
  return (size_t)(i >> 3) * t.tile_bytes + t.off_mass + (size_t)c * 64 + ((size_t)(i & 7) << 3);
}
__host__ __device__ inline size_t tiled_weight_off(const TiledDev& t, long long i) {
  return (size_t)(i >> 3) * t.tile_bytes + t.off_wgt + ((size_t)(i & 7) << 3);
}

struct SweepArgs {
  SampleDev s[2];        // 0 = MC, 1 = data
  const double* K;       // [R][KSTRIDE]
  const int* ch;         // [R]
  int R, C;
  int nb;                // number of 32-value batches = ceil(R / rpb)
  double* partial;       // [2][gridDim.x][nb*32 + 2]
};

struct cplx {
  double re, im;
};
__host__ __device__ inline cplx cmul(cplx a, cplx b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__host__ __device__ inline cplx cadd(cplx a, cplx b) { return {a.re + b.re, a.im + b.im}; }
__host__ __device__ inline cplx cscale(cplx a, double s) { return {a.re * s, a.im * s}; }
__host__ __device__ inline cplx cmuli(cplx a) { return {-a.im, a.re}; }  // i * a

}  // namespace pwa
