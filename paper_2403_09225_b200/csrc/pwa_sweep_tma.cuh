// pwa_sweep_tma.cuh - the tiled sweep kernel of the hot path (SURVEY §8(a) rows a-1 .. a-7) for sm_100a.
//
// One block = one "event group": S warps, warp s owns the resonance slice [s*RHO, s*RHO+RHO), lane = event.
// A tile is 32 consecutive events.  Tiles arrive in shared memory through a ring of TMA stages
// (cp.async.bulk.tensor.2d, one box for all R*H amplitude planes, one for the mass planes, one for the
// weights), completion tracked by one mbarrier per stage; out-of-range events of the ragged last tile are
// zero-filled by the TMA unit.  Every F element is read from HBM exactly once and is consumed by exactly
// one thread.
//
// Per tile the work is split in two halves which are software-pipelined across tiles so that ONE block
// barrier per tile suffices and the cross-slice exchange never leaves the FP64 pipe idle:
//   forward(t+1): B_r = 1/D_r (a-1), G_rh = B_r F_rh, partial A_h = sum c_r G_rh, Adot_h = sum (alpha_r +
//                 beta_r B_r) G_rh over the slice (a-2)                      -> shared memory
//   barrier; a few warps add the S partial sums in fixed order (a-7, first stage)
//   backward(t):  I, ln I, omega, kappa (a-3, a-4); B S_r = sum_h conj(omega A_h) G_rh and
//                 B S'_r = sum_h conj(omega (Adot_h - kappa A_h)) G_rh, and from them the five compact sums
//                 P1,P2,P3,Q1,Q2 of pwa_common.cuh (a-5, a-6) in per-thread registers.
// G, B of two consecutive tiles live in registers; the ten accumulators per resonance never leave the
// register file until the sample ends (then: fixed-order warp butterfly, one partial row per block).
#pragma once
#include <cuda.h>

#include "pwa_common.cuh"

namespace pwa {

struct alignas(64) TmaArgs {
  CUtensorMap amp[2], mass[2], wgt[2];  // 0 = MC, 1 = data
  long long n[2];
  const double* theta;
  const double* v;
  const int* ch;
  double* partial;  // [2][gridDim.x][R*VPR + 2]
  int R, C, S, stages, nbox, rows_box, weighted;
  unsigned stage_bytes, amp_bytes, mass_bytes;
  unsigned off_part, off_tot, off_K, off_ch, off_bar;
};

constexpr int TILE = 32;  // events per tile

// ---- PTX helpers ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// 1/d for normal-range positive d: hardware seed (MUFU.RCP64H, relative error 1e-6 measured on B200) and one
// cubic Newton step; measured maximum relative error against the IEEE division 2.2e-16 (kernels).
// Three DFMA and no slow-path branch.
__device__ __forceinline__ double fast_rcp(double d) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  const double e = fma(-d, y, 1.0);
  const double p = fma(e, e, e);
  return fma(y, p, y);
}

// per-resonance constants (same definitions as k_prologue) written to shared memory by the block itself
__device__ __forceinline__ void resonance_constants(const double* __restrict__ theta, const double* __restrict__ v,
                                                    int r, double* k) {
  const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
  double s, c;
  sincos(phi, &s, &c);
  const cplx e = {c, s};
  const cplx cc = {a * c, a * s};
  k[K_M2] = M * M;
  k[K_Y] = M * G;
  k[K_Y2] = (M * G) * (M * G);
  k[3] = 0.0;
  k[K_CR] = cc.re;
  k[K_CI] = cc.im;
  cplx al = {0.0, 0.0}, be = {0.0, 0.0};
  if (v) {
    const double va = v[4 * r], vp = v[4 * r + 1], vM = v[4 * r + 2], vG = v[4 * r + 3];
    al = cadd(cscale(e, va), cscale(cmuli(cc), vp));
    const cplx lam = {-2.0 * M * vM, G * vM + M * vG};
    be = cmul(cc, lam);
  }
  k[K_AR] = al.re;
  k[K_AI] = al.im;
  k[K_BR] = be.re;
  k[K_BI] = be.im;
  k[10] = 0.0;
  k[11] = 0.0;
}

__device__ __forceinline__ double warp_sum_x(double x) {
#pragma unroll
  for (int m = 16; m >= 1; m >>= 1) x += __shfl_xor_sync(0xffffffffu, x, m);
  return x;
}

template <int MODE>
__host__ __device__ constexpr int nacc_of() {
  return MODE == MODE_FULL ? 10 : (MODE == MODE_GRAD ? 4 : 0);
}

// ------------------------------------------------------------------------------------------------------
template <int H, int RHO, int MODE, int MAXW>
__global__ void __launch_bounds__(MAXW * 32, 1) k_sweep_tma(const __grid_constant__ TmaArgs a) {
  constexpr int NQ = (MODE == MODE_FULL) ? 2 * H : H;  // complex values exchanged per event and slice
  constexpr int NACC = nacc_of<MODE>();
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, s = threadIdx.x >> 5;
  const int S = a.S, R = a.R;
  double2* part = reinterpret_cast<double2*>(smem_raw + a.off_part);  // [2][S][NQ][32]
  double2* tot = reinterpret_cast<double2*>(smem_raw + a.off_tot);    // [2][NQ][32]
  double* Ks = reinterpret_cast<double*>(smem_raw + a.off_K);         // [R][KSTRIDE]
  int* chs = reinterpret_cast<int*>(smem_raw + a.off_ch);             // [R]
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + a.off_bar);  // [stages]
  const uint32_t full0 = smem_u32(full), stage0 = smem_u32(smem_raw);
  const int stages = a.stages;

  // ---- block setup: constants from theta (and v), channel map, barriers ------------------------------
  for (int r = threadIdx.x; r < R; r += blockDim.x) {
    resonance_constants(a.theta, MODE == MODE_FULL ? a.v : nullptr, r, Ks + r * KSTRIDE);
    chs[r] = a.ch[r];
  }
  if (threadIdx.x == 0) {
    for (int k = 0; k < stages; ++k) mbar_init(full0 + 8 * k, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    tma_prefetch_desc(&a.amp[0]);
    tma_prefetch_desc(&a.mass[0]);
    tma_prefetch_desc(&a.amp[1]);
    tma_prefetch_desc(&a.mass[1]);
  }
  __syncthreads();

  // ---- this block's tile list: MC tiles b, b+G, ... then data tiles b, b+G, ... ------------------------
  const long long tilesM = (a.n[0] + TILE - 1) / TILE, tilesD = (a.n[1] + TILE - 1) / TILE;
  const long long G = gridDim.x, b = blockIdx.x;
  const long long TmB = b < tilesM ? (tilesM - b + G - 1) / G : 0;
  const long long TdB = b < tilesD ? (tilesD - b + G - 1) / G : 0;
  const long long T = TmB + TdB;

  auto issue = [&](long long k) {  // producer: one thread
    const int smp = k >= TmB ? 1 : 0;
    const long long idx = b + (k - (smp ? TmB : 0)) * G;
    const int i0 = (int)(idx * TILE);
    const int st = (int)(k % stages);
    const uint32_t bar = full0 + 8 * st, dst = stage0 + st * a.stage_bytes;
    const bool w = smp == 1 && a.weighted;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(bar, a.amp_bytes + a.mass_bytes + (w ? TILE * 8u : 0u));
    for (int x = 0; x < a.nbox; ++x)
      tma_load_2d(dst + x * a.rows_box * (TILE * 16), &a.amp[smp], 2 * i0, x * a.rows_box, bar);
    tma_load_2d(dst + a.amp_bytes, &a.mass[smp], i0, 0, bar);
    if (w) tma_load_2d(dst + a.amp_bytes + a.mass_bytes, &a.wgt[smp], i0, 0, bar);
  };

  if (threadIdx.x == 0)
    for (long long k = 0; k < stages && k < T; ++k) issue(k);

  double acc[RHO][NACC > 0 ? NACC : 1];
  double s0 = 0.0, s1 = 0.0;
#pragma unroll
  for (int j = 0; j < RHO; ++j)
#pragma unroll
    for (int q = 0; q < (NACC > 0 ? NACC : 1); ++q) acc[j][q] = 0.0;
  double2 Gc[RHO][H], Gn[RHO][H], Bc[RHO], Bn[RHO];
  double wc = 1.0, wn = 1.0;  // data weight of this lane's event (current / next tile)

  // ---- forward half of tile k: propagators, G = B F, slice-partial A_h and Adot_h ------------------------
  auto forward = [&](long long k) {
    const int smp = k >= TmB ? 1 : 0;
    const long long idx = b + (k - (smp ? TmB : 0)) * G;
    const bool valid = idx * TILE + lane < a.n[smp];
    const int st = (int)(k % stages);
    mbar_wait(full0 + 8 * st, (uint32_t)((k / stages) & 1));
    const unsigned char* sp = smem_raw + (size_t)st * a.stage_bytes;
    const double2* Ft = reinterpret_cast<const double2*>(sp);
    const double* mt = reinterpret_cast<const double*>(sp + a.amp_bytes);
    wn = (smp == 1 && a.weighted) ? reinterpret_cast<const double*>(sp + a.amp_bytes + a.mass_bytes)[lane] : 1.0;
    double2 pA[H], pD[H];
#pragma unroll
    for (int h = 0; h < H; ++h) pA[h] = pD[h] = make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const int r = s * RHO + j;
      if (r < R) {  // warp-uniform
        const double* kk = Ks + r * KSTRIDE;
        const double m = mt[chs[r] * TILE + lane];
        const double x = fma(-m, m, kk[K_M2]);
        double den = fma(x, x, kk[K_Y2]);
        den = valid ? den : 1.0;  // zero-filled lanes of the ragged tile stay finite
        const double u = fast_rcp(den);
        const double br = x * u, bi = kk[K_Y] * u;  // B = conj(D)/|D|^2
        Bn[j] = make_double2(br, bi);
        const double cr = kk[K_CR], ci = kk[K_CI];
        if (MODE == MODE_NLL) {
          const double zr = cr * br - ci * bi, zi = cr * bi + ci * br;
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = Ft[(r * H + h) * TILE + lane];
            pA[h].x = fma(zr, F.x, fma(-zi, F.y, pA[h].x));
            pA[h].y = fma(zr, F.y, fma(zi, F.x, pA[h].y));
          }
        } else {
          double wr = 0.0, wi = 0.0;
          if (MODE == MODE_FULL) {  // zdot = (alpha + beta B) B
            wr = fma(kk[K_BR], br, fma(-kk[K_BI], bi, kk[K_AR]));
            wi = fma(kk[K_BR], bi, fma(kk[K_BI], br, kk[K_AI]));
          }
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = Ft[(r * H + h) * TILE + lane];
            const double gx = fma(br, F.x, -bi * F.y), gy = fma(br, F.y, bi * F.x);
            Gn[j][h] = make_double2(gx, gy);
            pA[h].x = fma(cr, gx, fma(-ci, gy, pA[h].x));
            pA[h].y = fma(cr, gy, fma(ci, gx, pA[h].y));
            if (MODE == MODE_FULL) {
              pD[h].x = fma(wr, gx, fma(-wi, gy, pD[h].x));
              pD[h].y = fma(wr, gy, fma(wi, gx, pD[h].y));
            }
          }
        }
      } else {
        Bn[j] = make_double2(0.0, 0.0);
#pragma unroll
        for (int h = 0; h < H; ++h) Gn[j][h] = make_double2(0.0, 0.0);
      }
    }
    double2* dst = part + ((size_t)((k & 1) * S + s) * NQ) * TILE + lane;
#pragma unroll
    for (int h = 0; h < H; ++h) {
      dst[h * TILE] = pA[h];
      if (MODE == MODE_FULL) dst[(H + h) * TILE] = pD[h];
    }
  };

  // ---- first stage of the reduction: fixed-order sum of the S slice partials -----------------------------
  auto reduce = [&](long long k) {
    const int buf = (int)(k & 1);
    for (int q = s; q < NQ; q += S) {
      const double2* src = part + ((size_t)(buf * S) * NQ + q) * TILE + lane;
      double2 t = src[0];
      for (int w = 1; w < S; ++w) {
        const double2 p = src[(size_t)w * NQ * TILE];
        t.x += p.x;
        t.y += p.y;
      }
      tot[(buf * NQ + q) * TILE + lane] = t;
    }
  };

  // ---- backward half of tile k ---------------------------------------------------------------------------
  auto backward = [&](long long k) {
    const int smp = k >= TmB ? 1 : 0;
    const long long idx = b + (k - (smp ? TmB : 0)) * G;
    const bool valid = idx * TILE + lane < a.n[smp];
    const double2* tp = tot + ((int)(k & 1) * NQ) * TILE + lane;
    double2 A[H], D[H];
    double I = 0.0;
#pragma unroll
    for (int h = 0; h < H; ++h) {
      A[h] = tp[h * TILE];
      I = fma(A[h].x, A[h].x, I);
      I = fma(A[h].y, A[h].y, I);
      if (MODE == MODE_FULL) D[h] = tp[(H + h) * TILE];
    }
    if (smp == 0) {
      if (s == 0) s0 += valid ? I : 0.0;
    } else {
      double w = wc;
      w = valid ? w : 0.0;
      const double Iv = valid ? I : 1.0;
      const double inv = 1.0 / Iv;
      const double om = w * inv;
      if (s == 0) {
        s0 = fma(w, log(Iv), s0);
        s1 += w;
      }
      double kap = 0.0;
      if (MODE == MODE_FULL) {
        double Idot = 0.0;
#pragma unroll
        for (int h = 0; h < H; ++h) {
          Idot = fma(A[h].x, D[h].x, Idot);
          Idot = fma(A[h].y, D[h].y, Idot);
        }
        kap = 2.0 * Idot * inv;
      }
#pragma unroll
      for (int h = 0; h < H; ++h) {
        if (MODE == MODE_FULL) {
          D[h].x = om * fma(-kap, A[h].x, D[h].x);
          D[h].y = om * fma(-kap, A[h].y, D[h].y);
        }
        A[h].x *= om;
        A[h].y *= om;
      }
    }
    if (MODE == MODE_NLL) return;
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const double br = Bc[j].x, bi = Bc[j].y;
      // t1 = B S = sum_h conj(A_h) G_h ;  u1 = B S' = sum_h conj(D_h) G_h
      double t1r = 0.0, t1i = 0.0, u1r = 0.0, u1i = 0.0;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        const double2 g = Gc[j][h];
        t1r = fma(A[h].x, g.x, fma(A[h].y, g.y, t1r));
        t1i = fma(A[h].x, g.y, fma(-A[h].y, g.x, t1i));
        if (MODE == MODE_FULL) {
          u1r = fma(D[h].x, g.x, fma(D[h].y, g.y, u1r));
          u1i = fma(D[h].x, g.y, fma(-D[h].y, g.x, u1i));
        }
      }
      acc[j][0] += t1r;  // P1
      acc[j][1] += t1i;
      if (MODE == MODE_GRAD) {
        acc[j][2] = fma(br, t1r, fma(-bi, t1i, acc[j][2]));  // P2
        acc[j][3] = fma(br, t1i, fma(bi, t1r, acc[j][3]));
      } else {
        const double t2r = fma(br, t1r, -bi * t1i), t2i = fma(br, t1i, bi * t1r);
        acc[j][2] += t2r;  // P2
        acc[j][3] += t2i;
        acc[j][4] = fma(br, t2r, fma(-bi, t2i, acc[j][4]));  // P3
        acc[j][5] = fma(br, t2i, fma(bi, t2r, acc[j][5]));
        acc[j][6] += u1r;  // Q1
        acc[j][7] += u1i;
        acc[j][8] = fma(br, u1r, fma(-bi, u1i, acc[j][8]));  // Q2
        acc[j][9] = fma(br, u1i, fma(bi, u1r, acc[j][9]));
      }
    }
  };

  // ---- end of a sample: fixed-order butterfly over the 32 event lanes, one partial row per block ---------
  auto flush = [&](int smp) {
    double* out = a.partial + ((size_t)smp * gridDim.x + blockIdx.x) * ((size_t)R * NACC + 2);
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const int r = s * RHO + j;
#pragma unroll
      for (int q = 0; q < NACC; ++q) {
        const double t = warp_sum_x(acc[j][q]);
        if (lane == 0 && r < R) out[r * NACC + q] = t;
        acc[j][q] = 0.0;
      }
    }
    const double t0 = warp_sum_x(s0), t1 = warp_sum_x(s1);
    if (s == 0 && lane == 0) {
      out[R * NACC] = t0;
      out[R * NACC + 1] = t1;
    }
    s0 = s1 = 0.0;
  };

  // ---- the pipelined tile loop ------------------------------------------------------------------------------
  if (T > 0) forward(0);
  __syncthreads();
  if (threadIdx.x == 0 && stages < T) issue(stages);
  if (T > 0) reduce(0);
#pragma unroll 1
  for (long long k = 0; k < T; ++k) {
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      Bc[j] = Bn[j];
      wc = wn;
#pragma unroll
      for (int h = 0; h < H; ++h) Gc[j][h] = Gn[j][h];
    }
    if (k + 1 < T) forward(k + 1);
    __syncthreads();
    if (threadIdx.x == 0 && k + 1 + stages < T) issue(k + 1 + stages);
    if (k + 1 < T) reduce(k + 1);
    if (k == TmB) flush(0);
    backward(k);
  }
  if (T == TmB) flush(0);
  flush(1);
}

}  // namespace pwa
