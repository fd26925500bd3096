// pwa_sweep_tma.cuh - the tiled sweep kernel of the hot path (SURVEY §8(a) rows a-1 .. a-7) for sm_100a.
//
// One block = one "event group": S compute warps + one producer warp.  Compute warp s owns the resonance
// slice [s*RHO, s*RHO+RHO), lane = event.  A tile is 32 consecutive events.  Tiles arrive in shared memory
// through a ring of TMA stages (cp.async.bulk.tensor.2d: one box for all R*H amplitude planes, one for the mass
// planes, one for the weights) issued by the producer warp; full[stage] / empty[stage] mbarriers track the
// ring; out-of-range events of the ragged last tile are zero-filled by the TMA unit.  Every F element is read
// from HBM exactly once and is consumed by exactly one thread.
//
// Per tile the work is split in two halves, software-pipelined across tiles so that every wait has one
// half-tile of slack and the cross-slice exchange never leaves the FP64 pipe idle:
//   forward(t+1): B_r = 1/D_r (a-1), G_rh = B_r F_rh, partial A_h = sum c_r G_rh, Adot_h = sum (alpha_r +
//                 beta_r B_r) G_rh over the slice (a-2)            -> shared memory, arrive pf[(t+1)&1]
//   backward(t):  wait tf[t&1]; I, ln I, omega, kappa (a-3, a-4); B S_r = sum_h conj(omega A_h) G_rh and
//                 B S'_r = sum_h conj(omega (Adot_h - kappa A_h)) G_rh, and from them the five compact sums
//                 P1,P2,P3,Q1,Q2 of pwa_common.cuh (a-5, a-6) in per-thread registers.
//   reduce(t+1):  (up to 2*NQ warps) wait pf, add the S slice partials in a fixed tree (a-7, first stage),
//                 arrive tf[(t+1)&1]
// G, B of two consecutive tiles live in registers (two register sets, loop unrolled by two); the ten
// accumulators per resonance never leave the register file until the sample ends (then: fixed-order warp
// butterfly, one partial row per block).
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
  unsigned off_part, off_tot, off_K, off_bar;
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
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
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

// per-resonance constants (same definitions as k_prologue), packed in pairs for 128-bit shared loads:
//   k[0..1] = M^2, (M Gamma)^2   k[2..3] = M Gamma, 0   k[4..5] = c   k[6..7] = alpha   k[8..9] = beta
constexpr int KS = 10;
__device__ __forceinline__ void resonance_constants(const double* __restrict__ theta, const double* __restrict__ v,
                                                    int r, double* k) {
  const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
  double s, c;
  sincos(phi, &s, &c);
  const cplx e = {c, s};
  const cplx cc = {a * c, a * s};
  k[0] = M * M;
  k[1] = (M * G) * (M * G);
  k[2] = M * G;
  k[3] = 0.0;
  k[4] = cc.re;
  k[5] = cc.im;
  cplx al = {0.0, 0.0}, be = {0.0, 0.0};
  if (v) {
    const double va = v[4 * r], vp = v[4 * r + 1], vM = v[4 * r + 2], vG = v[4 * r + 3];
    al = cadd(cscale(e, va), cscale(cmuli(cc), vp));
    const cplx lam = {-2.0 * M * vM, G * vM + M * vG};
    be = cmul(cc, lam);
  }
  k[6] = al.re;
  k[7] = al.im;
  k[8] = be.re;
  k[9] = be.im;
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
// MAXW = the most warps (compute + producer) a block of this instance may have; it fixes the register cap:
// each of the four SM sub-partitions owns 16384 registers and hosts ceil(MAXW / 4) of the block's warps.
constexpr int regs_for_warps(int maxw) {
  const int r = 16384 / (((maxw + 3) / 4) * 32) / 8 * 8;
  return r > 255 ? 255 : r;
}
template <int H, int RHO, int MODE, int MAXW>
__global__ void __maxnreg__(regs_for_warps(MAXW)) k_sweep_tma(const __grid_constant__ TmaArgs a) {
  constexpr int NQ = (MODE == MODE_FULL) ? 2 * H : H;  // complex values exchanged per event and slice
  constexpr int NACC = nacc_of<MODE>();
  constexpr int NA = NACC > 0 ? NACC : 1;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, s = threadIdx.x >> 5;
  const int S = a.S, R = a.R;
  double2* part = reinterpret_cast<double2*>(smem_raw + a.off_part);  // [2][S][NQ][32]
  double2* tot = reinterpret_cast<double2*>(smem_raw + a.off_tot);    // [2][NQ][32]
  double* Ks = reinterpret_cast<double*>(smem_raw + a.off_K);         // [R][KS]
  const int stages = a.stages;
  // mbarriers: full[stages] | empty[stages] | pf[2] | tf[2]
  const uint32_t full0 = smem_u32(smem_raw + a.off_bar), empty0 = full0 + 8 * stages;
  const uint32_t pf0 = empty0 + 8 * stages, tf0 = pf0 + 16;
  const uint32_t stage0 = smem_u32(smem_raw);
  const int n_red = S < 2 * NQ ? S : 2 * NQ;  // warps that take part in the slice reduction

  // ---- block setup: constants from theta (and v), barriers ---------------------------------------------
  for (int r = threadIdx.x; r < R; r += blockDim.x)
    resonance_constants(a.theta, MODE == MODE_FULL ? a.v : nullptr, r, Ks + r * KS);
  if (threadIdx.x == 0) {
    for (int k = 0; k < stages; ++k) {
      mbar_init(full0 + 8 * k, 1);
      mbar_init(empty0 + 8 * k, S);
    }
    for (int k = 0; k < 2; ++k) {
      mbar_init(pf0 + 8 * k, S);
      mbar_init(tf0 + 8 * k, n_red);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // ---- this block's tile list: MC tiles b, b+G, ... then data tiles b, b+G, ... ------------------------
  const int nM = (int)a.n[0], nD = (int)a.n[1];
  const int tilesM = (nM + TILE - 1) / TILE, tilesD = (nD + TILE - 1) / TILE;
  const int G = gridDim.x, b = blockIdx.x;
  const int TmB = b < tilesM ? (tilesM - b + G - 1) / G : 0;
  const int TdB = b < tilesD ? (tilesD - b + G - 1) / G : 0;
  const int T = TmB + TdB;

  // ======================================= producer warp ===================================================
  if (s == S) {
    if (lane == 0) {
      tma_prefetch_desc(&a.amp[0]);
      tma_prefetch_desc(&a.mass[0]);
      tma_prefetch_desc(&a.amp[1]);
      tma_prefetch_desc(&a.mass[1]);
      int st = 0, round = 0;
      for (int k = 0; k < T; ++k) {
        if (round > 0) mbar_wait(empty0 + 8 * st, (uint32_t)((round - 1) & 1));
        const int smp = k >= TmB ? 1 : 0;
        const int i0 = (b + (k - (smp ? TmB : 0)) * G) * TILE;
        const uint32_t bar = full0 + 8 * st, dst = stage0 + st * a.stage_bytes;
        const bool w = smp == 1 && a.weighted;
        mbar_expect_tx(bar, a.amp_bytes + a.mass_bytes + (w ? TILE * 8u : 0u));
        for (int x = 0; x < a.nbox; ++x)
          tma_load_2d(dst + x * a.rows_box * (TILE * 16), &a.amp[smp], 2 * i0, x * a.rows_box, bar);
        tma_load_2d(dst + a.amp_bytes, &a.mass[smp], i0, 0, bar);
        if (w) tma_load_2d(dst + a.amp_bytes + a.mass_bytes, &a.wgt[smp], i0, 0, bar);
        if (++st == stages) {
          st = 0;
          ++round;
        }
      }
    }
    return;
  }

  // ======================================= compute warps ===================================================
  double acc[RHO][NA];
  double s0 = 0.0, s1 = 0.0;
#pragma unroll
  for (int j = 0; j < RHO; ++j)
#pragma unroll
    for (int q = 0; q < NA; ++q) acc[j][q] = 0.0;
  int moff[RHO];  // offset of this lane's mass inside a stage's mass tile, per owned resonance
#pragma unroll
  for (int j = 0; j < RHO; ++j) {
    const int r = s * RHO + j;
    moff[j] = (r < R ? a.ch[r] : 0) * TILE + lane;
  }
  int st_f = 0, ph_f = 0;  // ring position of the next forward()

  // ---- forward half of tile k: propagators, G = B F, slice-partial A_h and Adot_h ------------------------
  auto forward = [&](int k, double2(&Gn)[RHO][H], double2(&Bn)[RHO], double& wn) {
    const int smp = k >= TmB ? 1 : 0;
    const int i0 = (b + (k - (smp ? TmB : 0)) * G) * TILE;
    const bool valid = i0 + lane < (smp ? nD : nM);
    mbar_wait(full0 + 8 * st_f, (uint32_t)ph_f);
    const unsigned char* sp = smem_raw + (size_t)st_f * a.stage_bytes;
    const double2* Ft = reinterpret_cast<const double2*>(sp) + lane;
    const double* mt = reinterpret_cast<const double*>(sp + a.amp_bytes);
    wn = (smp == 1 && a.weighted) ? reinterpret_cast<const double*>(sp + a.amp_bytes + a.mass_bytes)[lane] : 1.0;
    double2 pA[H], pD[H];
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const int r = s * RHO + j;
      if (j == 0 || r < R) {  // warp-uniform; slice s always owns resonance s*RHO
        const double2* kk = reinterpret_cast<const double2*>(Ks + r * KS);
        const double2 k01 = kk[0], k23 = kk[1], c = kk[2];
        const double m = mt[moff[j]];
        const double x = fma(-m, m, k01.x);
        double den = fma(x, x, k01.y);
        den = valid ? den : 1.0;  // zero-filled lanes of the ragged tile stay finite
        const double u = fast_rcp(den);
        const double br = x * u, bi = k23.x * u;  // B = conj(D)/|D|^2
        Bn[j] = make_double2(br, bi);
        if (MODE == MODE_NLL) {
          const double zr = fma(c.x, br, -(c.y * bi)), zi = fma(c.x, bi, c.y * br);
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = Ft[(r * H + h) * TILE];
            if (j == 0) {
              pA[h].x = fma(zr, F.x, -(zi * F.y));
              pA[h].y = fma(zr, F.y, zi * F.x);
            } else {
              pA[h].x = fma(zr, F.x, fma(-zi, F.y, pA[h].x));
              pA[h].y = fma(zr, F.y, fma(zi, F.x, pA[h].y));
            }
          }
        } else {
          double wr = 0.0, wi = 0.0;
          if (MODE == MODE_FULL) {  // zdot = (alpha + beta B) B
            const double2 al = kk[3], be = kk[4];
            wr = fma(be.x, br, fma(-be.y, bi, al.x));
            wi = fma(be.x, bi, fma(be.y, br, al.y));
          }
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = Ft[(r * H + h) * TILE];
            const double gx = fma(br, F.x, -(bi * F.y)), gy = fma(br, F.y, bi * F.x);
            Gn[j][h] = make_double2(gx, gy);
            if (j == 0) {
              pA[h].x = fma(c.x, gx, -(c.y * gy));
              pA[h].y = fma(c.x, gy, c.y * gx);
              if (MODE == MODE_FULL) {
                pD[h].x = fma(wr, gx, -(wi * gy));
                pD[h].y = fma(wr, gy, wi * gx);
              }
            } else {
              pA[h].x = fma(c.x, gx, fma(-c.y, gy, pA[h].x));
              pA[h].y = fma(c.x, gy, fma(c.y, gx, pA[h].y));
              if (MODE == MODE_FULL) {
                pD[h].x = fma(wr, gx, fma(-wi, gy, pD[h].x));
                pD[h].y = fma(wr, gy, fma(wi, gx, pD[h].y));
              }
            }
          }
        }
      } else {
        Bn[j] = make_double2(0.0, 0.0);
#pragma unroll
        for (int h = 0; h < H; ++h) Gn[j][h] = make_double2(0.0, 0.0);
      }
    }
    // the stage has been read: hand it back to the producer
    __syncwarp();
    if (lane == 0) mbar_arrive(empty0 + 8 * st_f);
    if (++st_f == stages) {
      st_f = 0;
      ph_f ^= 1;
    }
    double2* dst = part + ((size_t)((k & 1) * S + s) * NQ) * TILE + lane;
#pragma unroll
    for (int h = 0; h < H; ++h) {
      dst[h * TILE] = pA[h];
      if (MODE == MODE_FULL) dst[(H + h) * TILE] = pD[h];
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(pf0 + 8 * (k & 1));
  };

  // ---- first stage of the reduction: fixed-order sum of the S slice partials -----------------------------
  // item = (quantity q, component c); warp s takes items s, s+S, ...  Lanes read one double each.
  auto reduce = [&](int k) {
    const int buf = k & 1;
    if (s >= n_red) return;
    mbar_wait(pf0 + 8 * buf, (uint32_t)((k >> 1) & 1));
    for (int item = s; item < 2 * NQ; item += S) {
      const int q = item >> 1, c = item & 1;
      const double* src = reinterpret_cast<const double*>(part + ((size_t)(buf * S) * NQ + q) * TILE + lane) + c;
      double t0 = src[0], t1 = 0.0;
      int w = 1;
      for (; w + 1 < S; w += 2) {
        t1 += src[(size_t)w * NQ * TILE * 2];
        t0 += src[(size_t)(w + 1) * NQ * TILE * 2];
      }
      if (w < S) t1 += src[(size_t)w * NQ * TILE * 2];
      reinterpret_cast<double*>(tot + (buf * NQ + q) * TILE + lane)[c] = t0 + t1;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(tf0 + 8 * buf);
  };

  // ---- backward half of tile k ---------------------------------------------------------------------------
  auto backward = [&](int k, const double2(&Gc)[RHO][H], const double2(&Bc)[RHO], double wc) {
    const int smp = k >= TmB ? 1 : 0;
    const int i0 = (b + (k - (smp ? TmB : 0)) * G) * TILE;
    const bool valid = i0 + lane < (smp ? nD : nM);
    mbar_wait(tf0 + 8 * (k & 1), (uint32_t)((k >> 1) & 1));
    const double2* tp = tot + ((k & 1) * NQ) * TILE + lane;
    double2 A[H], D[H];
    double I = 0.0;
#pragma unroll
    for (int h = 0; h < H; ++h) {
      A[h] = tp[h * TILE];
      I = h == 0 ? fma(A[h].x, A[h].x, A[h].y * A[h].y) : fma(A[h].x, A[h].x, fma(A[h].y, A[h].y, I));
      if (MODE == MODE_FULL) D[h] = tp[(H + h) * TILE];
    }
    if (smp == 0) {
      if (s == 0) s0 += valid ? I : 0.0;
    } else {
      const double w = valid ? wc : 0.0;
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
        for (int h = 0; h < H; ++h) Idot = fma(A[h].x, D[h].x, fma(A[h].y, D[h].y, Idot));
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
      double t1r, t1i, u1r = 0.0, u1i = 0.0;
      {
        const double2 g = Gc[j][0];
        t1r = fma(A[0].x, g.x, A[0].y * g.y);
        t1i = fma(A[0].x, g.y, -(A[0].y * g.x));
        if (MODE == MODE_FULL) {
          u1r = fma(D[0].x, g.x, D[0].y * g.y);
          u1i = fma(D[0].x, g.y, -(D[0].y * g.x));
        }
      }
#pragma unroll
      for (int h = 1; h < H; ++h) {
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
        const double t2r = fma(br, t1r, -(bi * t1i)), t2i = fma(br, t1i, bi * t1r);
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
    if (s == 0) {
      const double t0 = warp_sum_x(s0), t1 = warp_sum_x(s1);
      if (lane == 0) {
        out[R * NACC] = t0;
        out[R * NACC + 1] = t1;
      }
    }
    s0 = s1 = 0.0;
  };

  // ---- the pipelined tile loop, unrolled by two so that the two register sets swap roles -------------------
  double2 G0[RHO][H], G1[RHO][H], B0[RHO], B1[RHO];
  double w0 = 1.0, w1 = 1.0;
  if (T > 0) {
    forward(0, G0, B0, w0);
    reduce(0);
  }
  int k = 0;
#pragma unroll 1
  while (k < T) {
    if (k + 1 < T) forward(k + 1, G1, B1, w1);
    if (k == TmB) flush(0);
    backward(k, G0, B0, w0);
    if (k + 1 < T) reduce(k + 1);
    if (++k >= T) break;
    if (k + 1 < T) forward(k + 1, G0, B0, w0);
    if (k == TmB) flush(0);
    backward(k, G1, B1, w1);
    if (k + 1 < T) reduce(k + 1);
    ++k;
  }
  if (T == TmB) flush(0);
  flush(1);
}

}  // namespace pwa
