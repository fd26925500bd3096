// pwa_sweep_pair.cuh - the fused sweep (NLL + gradient + HVP, SURVEY 8(a) rows a-1 .. a-7) with TWO events per lane.
//
// Same tiles, ring, producer warpgroup and lane = slice x event decomposition as k_sweep_lanes (pwa_sweep_lanes.cuh) for
// the shape RHO = 4 resonances per lane, 8 slices, 4 events per column, 8 compute warps; what changes:
//   * warp w takes the column PAIR w % 4 of the local tiles w / 4, w / 4 + 2, ...; a lane works on two events, one per
//     column - even slices take the columns in the order (2cp, 2cp + 1), odd slices in the order (2cp + 1, 2cp);
//   * two independent events per lane double the independent FP64 chains a warp can issue (ncu on the one-event kernel:
//     FP64 pipe 65 % active with 2 warps per scheduler, "wait" - the fixed latency of dependent DFMAs - the first stall);
//   * a quarter-warp (two slices x four events) reads 128 CONTIGUOUS bytes of a plane row: the 2-way bank conflict of
//     the one-event kernel's F reads is gone; the per-resonance constants are read once for two events;
//   * the first exchange level needs no selects: both lanes of a slice pair keep their first event and send the second.
// To fit two events' G = B F (64 registers) beside the accumulators, P3 is folded into Q2: with
//   lam2 = 2 lambda,  lambda = -(2M - i Gamma) v_M + i M v_Gamma      (beta = c lambda)
// the kernel accumulates Q2' = sum B (u1 + lam2 t2) = Q2 + lam2 P3 instead of Q2 and P3 separately - the unpacking of
// h_M and h_Gamma needs exactly this combination (k3 = -c D_M lam2, k3' = i M c lam2) - 8 accumulators per resonance
// instead of 10, the same FP64 count (34 backward instructions per (event, resonance) at H = 2).
// Partial row layout per resonance: P1, P2, Q1, Q2' (MODE_FULLP in pwa_common.cuh).
#pragma once
#include "pwa_sweep_lanes.cuh"

namespace pwa {

struct PairArgs {
  int stages;
  unsigned off_K, off_red, off_xch, off_bar;  // after the stages (stage geometry: LaneArgs)
};

namespace lanes {

constexpr int KSP = 14;  // doubles of constants per resonance: the KS of the one-event kernel, lam2, 2 of padding (112-byte
                         // stride: the 8 slices of a warp read 8 different 16-byte bank groups)

// MODE: MODE_FULLP (P1, P2, Q1, Q2'), MODE_GRAD3 (P1, P2, P3: the gradient call of the split evaluation) or MODE_HVPQ
// (Q1, Q2 at the kept theta: the cached HVP) - the three sweeps a Newton-CG fit and the timed fused call consist of.
template <int H, int MODE>
__global__ void __launch_bounds__(lanes_threads(8, 2), 1) k_sweep_pair(const __grid_constant__ LaneArgs a,
                                                                       const __grid_constant__ PairArgs pa) {
  static_assert(MODE == MODE_FULLP || MODE == MODE_GRAD3 || MODE == MODE_HVPQ || MODE == MODE_GRAD || MODE == MODE_NLL,
                "modes of the two-event kernel");
  constexpr int RHO = 4, LOG_SW = 3, NW = 8, TILE = 32;
  constexpr int SW = 1 << LOG_SW, EW = 32 / SW, NP = TILE / EW, NPP = NP / 2, RP = RHO * SW;
  constexpr bool WQ = MODE == MODE_FULLP || MODE == MODE_HVPQ;   // needs Adot, accumulates Q sums
  constexpr bool WP = MODE == MODE_FULLP || MODE == MODE_GRAD3 || MODE == MODE_GRAD;  // accumulates P sums
  constexpr bool BWD = MODE != MODE_NLL;
  constexpr int NV = (WQ ? 4 : 2) * H;   // A_h [, Adot_h] (re, im) per event
  constexpr int NACC = MODE == MODE_NLL ? 0 : vpr_of(MODE);  // FULLP: P1, P2, Q1, Q2'; GRAD3: P1, P2, P3; GRAD: P1, P2; HVPQ: Q1, Q2
  constexpr int NA = NACC > 0 ? NACC : 1;
  constexpr int QO = MODE == MODE_FULLP ? 4 : 0;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  if (a.skip != nullptr && *a.skip != 0.0) return;
  const int lane = threadIdx.x & 31, w = (int)(threadIdx.x >> 5) - 4;
  const int R = a.R, stages = pa.stages;
  double* Ks = reinterpret_cast<double*>(smem_raw + pa.off_K);    // [RP][KSP]
  double* red = reinterpret_cast<double*>(smem_raw + pa.off_red);  // [NW][R*NACC + 2]
  const uint32_t full0 = smem_u32(smem_raw + pa.off_bar), empty0 = full0 + 8 * stages;

  for (int r = threadIdx.x; r < RP; r += blockDim.x) {
    double* k = Ks + r * KSP;
    if (r < R) {
      resonance_constants(a.theta, WQ ? a.v : nullptr, r, (long long)a.off_mass + (long long)a.ch[r] * (TILE * 8), k);
      k[10] = k[11] = 0.0;
      if (MODE == MODE_FULLP) {
        const double M = a.theta[4 * r + 2], G = a.theta[4 * r + 3], vM = a.v[4 * r + 2], vG = a.v[4 * r + 3];
        k[10] = 2.0 * (-2.0 * M * vM);        // lam2 = 2 lambda
        k[11] = 2.0 * (G * vM + M * vG);
      }
    } else {
      k[0] = 0.0; k[1] = 1.0; k[2] = 0.0; k[3] = __longlong_as_double((long long)a.off_mass);
      k[4] = k[5] = k[6] = k[7] = k[8] = k[9] = k[10] = k[11] = 0.0;
    }
    k[12] = k[13] = 0.0;
  }
  if (threadIdx.x == 0) {
    for (int k = 0; k < stages; ++k) {
      mbar_init(full0 + 8 * k, 1);
      mbar_init(empty0 + 8 * k, NPP);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const long long nM = a.n[0], nD = a.n[1];
  const int tilesM = (int)((nM + TILE - 1) / TILE), tilesD = (int)((nD + TILE - 1) / TILE);
  const int G = gridDim.x, b = blockIdx.x;
  const int TmB = b < tilesM ? (tilesM - b + G - 1) / G : 0;
  const int TdB = b < tilesD ? (tilesD - b + G - 1) / G : 0;
  const int T = TmB + TdB;

  // ======================================= producer ========================================================
  if (w < 0) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
    // the warps of the producer warpgroup take the local tiles in turn (pwa_sweep_lanes.cuh: one issuing thread caps
    // the ring near one tile per 800 cycles)
    const int NPW = a.nprod, p0 = w + 4;
    if (lane == 0 && p0 < NPW) {
      tma_prefetch_desc(&a.tm_amp[0]);
      tma_prefetch_desc(&a.tm_mass[0]);
      tma_prefetch_desc(&a.tm_amp[1]);
      tma_prefetch_desc(&a.tm_mass[1]);
      int st = p0 % stages, wrap = p0 / stages;  // stage of tile k and how often the ring has wrapped before it
      for (int k = p0; k < T; k += NPW) {
        if (wrap > 0) mbar_wait(empty0 + 8 * st, (uint32_t)((wrap - 1) & 1));
        const int smp = k >= TmB ? 1 : 0;
        const int i0 = (b + (k - (smp ? TmB : 0)) * G) * TILE;
        const bool wg = smp == 1 && a.weighted;
        const uint32_t bar = full0 + 8 * st, dst = smem_u32(smem_raw) + st * a.stage_bytes;
        mbar_expect_tx(bar, a.amp_bytes + (unsigned)a.C * (TILE * 8) + (wg ? TILE * 8u : 0u));
        for (int x = 0; x < a.nbox; ++x)
          tma_load_2d(dst + x * a.rows_box * (TILE * 16), &a.tm_amp[smp], 2 * i0, x * a.rows_box, bar);
        tma_load_2d(dst + a.off_mass, &a.tm_mass[smp], i0, 0, bar);
        if (wg) tma_load_2d(dst + a.off_wgt, &a.tm_wgt[smp], i0, 0, bar);
        st += NPW;
        while (st >= stages) {
          st -= stages;
          ++wrap;
        }
      }
    }
    return;
  }

  // ======================================= compute warps ===================================================
  asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
  const int s = lane >> (5 - LOG_SW), e = lane & (EW - 1);
  double acc[RHO][NA];
  double s0 = 0.0, s1 = 0.0;
#pragma unroll
  for (int j = 0; j < RHO; ++j)
#pragma unroll
    for (int q = 0; q < NA; ++q) acc[j][q] = 0.0;
  const double* lane_k = Ks + s * KSP;
  unsigned moff[RHO];
#pragma unroll
  for (int j = 0; j < RHO; ++j) moff[j] = (unsigned)__double_as_longlong(lane_k[j * (SW * KSP) + 3]);

  const int cp = w % NPP;
  const int colA = 2 * cp + (s & 1), colB = 2 * cp + ((s & 1) ^ 1);
  const int evA = colA * EW + e, evB = colB * EW + e;
  const unsigned fA = (unsigned)s * (H * TILE * 16) + (unsigned)evA * 16u, fB = (unsigned)s * (H * TILE * 16) + (unsigned)evB * 16u;
  // exchange rows: [NW][2 EW events of the column pair][NV + 2]; row of event (column parity, e)
  double* xbase = reinterpret_cast<double*>(smem_raw + pa.off_xch) + (size_t)w * (2 * EW) * (NV + 2);
  double* rowA = xbase + ((s & 1) * EW + e) * (NV + 2);
  double* rowB = xbase + (((s & 1) ^ 1) * EW + e) * (NV + 2);
  int t = w / NPP;
  int st = t % stages, ph = (t / stages) & 1;  // advanced incrementally (an integer division per iteration showed up in ncu)

  for (int smp = 0; smp < 2; ++smp) {
    const int t_end = smp ? T : TmB;
    const int n = (int)(smp ? nD : nM);
    const bool weighted = smp == 1 && a.weighted;
#pragma unroll 1
    while (t < t_end) {
      const int i0 = (b + (t - (smp ? TmB : 0)) * G) * TILE;
      const bool validA = i0 + evA < n, validB = i0 + evB < n;
      mbar_wait(full0 + 8 * st, (uint32_t)ph);
      const unsigned char* sp = smem_raw + (size_t)st * a.stage_bytes;
      double wtA = 1.0, wtB = 1.0;
      if (weighted) {
        wtA = reinterpret_cast<const double*>(sp + a.off_wgt)[evA];
        wtB = reinterpret_cast<const double*>(sp + a.off_wgt)[evB];
      }

      // ---------------- forward, both events ----------------
      double2 Gr[2][BWD ? RHO : 1][H], Br[2][BWD ? RHO : 1];
      double x[2][NV];  // per event: slice partials A_h (re, im), then Adot_h (re, im)
#pragma unroll
      for (int j = 0; j < RHO; ++j) {
        const double2* kk = reinterpret_cast<const double2*>(lane_k + j * (SW * KSP));
        const double2 k01 = kk[0];
        const double mg = lane_k[j * (SW * KSP) + 2];
        const double2 c = kk[2], al = WQ ? kk[3] : make_double2(0.0, 0.0), be = WQ ? kk[4] : make_double2(0.0, 0.0);
#pragma unroll
        for (int sd = 0; sd < 2; ++sd) {
          const double m = *reinterpret_cast<const double*>(sp + moff[j] + (sd ? evB : evA) * 8);
          const double xx = fma(-m, m, k01.x);
          const double u = fast_rcp(fma(xx, xx, k01.y));
          const double br = xx * u, bi = mg * u;
          if (BWD) Br[sd][j] = make_double2(br, bi);
          double wr = 0.0, wi = 0.0;
          if (WQ) {  // zdot = (alpha + beta B) B
            wr = fma(be.x, br, fma(-be.y, bi, al.x));
            wi = fma(be.x, bi, fma(be.y, br, al.y));
          }
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = *reinterpret_cast<const double2*>(sp + (sd ? fB : fA) + (j * SW * H + h) * (TILE * 16));
            const double gx = fma(br, F.x, -(bi * F.y)), gy = fma(br, F.y, bi * F.x);
            if (BWD) Gr[sd][j][h] = make_double2(gx, gy);
            double* xs = x[sd];
            if (j == 0) {
              xs[2 * h] = fma(c.x, gx, -(c.y * gy));
              xs[2 * h + 1] = fma(c.x, gy, c.y * gx);
              if (WQ) {
                xs[2 * H + 2 * h] = fma(wr, gx, -(wi * gy));
                xs[2 * H + 2 * h + 1] = fma(wr, gy, wi * gx);
              }
            } else {
              xs[2 * h] = fma(c.x, gx, fma(-c.y, gy, xs[2 * h]));
              xs[2 * h + 1] = fma(c.x, gy, fma(c.y, gx, xs[2 * h + 1]));
              if (WQ) {
                xs[2 * H + 2 * h] = fma(wr, gx, fma(-wi, gy, xs[2 * H + 2 * h]));
                xs[2 * H + 2 * h + 1] = fma(wr, gy, fma(wi, gx, xs[2 * H + 2 * h + 1]));
              }
            }
          }
        }
      }
      __syncwarp();
      mbar_arrive_if_zero(empty0 + 8 * st, (uint32_t)lane);

      // ---------------- exchange over the slices ----------------
      // level 1 over the slice pair (keep the first event, send the second), then reduce-scatter over the other slice
      // bits; every lane stores its share of ITS first event's totals, then reads the rows of both its events
#pragma unroll
      for (int i = 0; i < NV; ++i) x[0][i] += shfl_x(x[1][i], EW);
      slice_reduce_store<NV, 2 * EW>(x[0], lane, rowA);
      __syncwarp();
#pragma unroll
      for (int i = 0; i < NV; i += 2) {
        const double2 p = *reinterpret_cast<const double2*>(rowA + i);
        const double2 q = *reinterpret_cast<const double2*>(rowB + i);
        x[0][i] = p.x; x[0][i + 1] = p.y;
        x[1][i] = q.x; x[1][i + 1] = q.y;
      }
      __syncwarp();  // the rows are rewritten by the next iteration

      // ---------------- event stage and backward, one event after the other ----------------
#pragma unroll
      for (int sd = 0; sd < 2; ++sd) {
        double* xs = x[sd];
        double I = 0.0;
#pragma unroll
        for (int h = 0; h < H; ++h) I = fma(xs[2 * h], xs[2 * h], fma(xs[2 * h + 1], xs[2 * h + 1], I));
        // every event of the column pair is held by the lanes of 8 slices: slice 0 counts the first event of its lanes,
        // slice 1 the first event of ITS lanes (the other column) - the scalars of an event are added exactly once
        const bool count = sd == 0 && s < 2;
        if (smp == 0) {
          if (count) s0 += I;  // lanes beyond the ragged end read zero-filled F: I = 0
        } else {
          const bool valid = sd ? validB : validA;
          const double wv = valid ? (sd ? wtB : wtA) : 0.0;
          const double Iv = valid ? I : 1.0;
          const double inv = 1.0 / Iv;
          const double om = wv * inv;
          if (count) {
            if (MODE != MODE_HVPQ) s0 = fma(wv, log(Iv), s0);  // HVPQ: the scalars come from the kept gradient evaluation
            s1 += wv;
          }
          if (WQ) {
            double Idot = 0.0;
#pragma unroll
            for (int h = 0; h < H; ++h)
              Idot = fma(xs[2 * h], xs[2 * H + 2 * h], fma(xs[2 * h + 1], xs[2 * H + 2 * h + 1], Idot));
            const double kap = 2.0 * Idot * inv;
#pragma unroll
            for (int h = 0; h < H; ++h) {
              xs[2 * H + 2 * h] = om * fma(-kap, xs[2 * h], xs[2 * H + 2 * h]);
              xs[2 * H + 2 * h + 1] = om * fma(-kap, xs[2 * h + 1], xs[2 * H + 2 * h + 1]);
            }
          }
#pragma unroll
          for (int h = 0; h < H; ++h) {
            xs[2 * h] *= om;
            xs[2 * h + 1] *= om;
          }
        }
#pragma unroll
        for (int j = 0; j < (BWD ? RHO : 0); ++j) {
          const double br = Br[sd][j].x, bi = Br[sd][j].y;
          double t1r = 0.0, t1i = 0.0, u1r = 0.0, u1i = 0.0;
          if (WP) {  // t1 = B S = sum_h conj(omega A_h) G_h
            const double2 g = Gr[sd][j][0];
            t1r = fma(xs[0], g.x, xs[1] * g.y);
            t1i = fma(xs[0], g.y, -(xs[1] * g.x));
#pragma unroll
            for (int h = 1; h < H; ++h) {
              const double2 gh = Gr[sd][j][h];
              t1r = fma(xs[2 * h], gh.x, fma(xs[2 * h + 1], gh.y, t1r));
              t1i = fma(xs[2 * h], gh.y, fma(-xs[2 * h + 1], gh.x, t1i));
            }
          }
          if (WQ) {  // u1 = B S' = sum_h conj(omega (Adot_h - kappa A_h)) G_h
            const double2 g = Gr[sd][j][0];
            u1r = fma(xs[2 * H], g.x, xs[2 * H + 1] * g.y);
            u1i = fma(xs[2 * H], g.y, -(xs[2 * H + 1] * g.x));
#pragma unroll
            for (int h = 1; h < H; ++h) {
              const double2 gh = Gr[sd][j][h];
              u1r = fma(xs[2 * H + 2 * h], gh.x, fma(xs[2 * H + 2 * h + 1], gh.y, u1r));
              u1i = fma(xs[2 * H + 2 * h], gh.y, fma(-xs[2 * H + 2 * h + 1], gh.x, u1i));
            }
          }
          if (MODE == MODE_GRAD) {
            acc[j][0] += t1r;  // P1
            acc[j][1] += t1i;
            acc[j][2] = fma(br, t1r, fma(-bi, t1i, acc[j][2]));  // P2
            acc[j][3] = fma(br, t1i, fma(bi, t1r, acc[j][3]));
          } else if (WP) {
            const double t2r = fma(br, t1r, -(bi * t1i)), t2i = fma(br, t1i, bi * t1r);  // B^2 S
            acc[j][0] += t1r;  // P1
            acc[j][1] += t1i;
            acc[j][2] += t2r;  // P2
            acc[j][3] += t2i;
            if (MODE == MODE_GRAD3) {
              acc[j][4] = fma(br, t2r, fma(-bi, t2i, acc[j][4]));  // P3
              acc[j][5] = fma(br, t2i, fma(bi, t2r, acc[j][5]));
            } else {  // FULLP: u1 <- u1 + lam2 t2, so that the Q2 accumulation below gives Q2' = Q2 + lam2 P3
              const double2 l2 = *reinterpret_cast<const double2*>(lane_k + j * (SW * KSP) + 10);
              const double vr = fma(l2.x, t2r, fma(-l2.y, t2i, u1r)), vi = fma(l2.x, t2i, fma(l2.y, t2r, u1i));
              acc[j][QO] += u1r;  // Q1 (before the fold)
              acc[j][QO + 1] += u1i;
              acc[j][QO + 2] = fma(br, vr, fma(-bi, vi, acc[j][QO + 2]));
              acc[j][QO + 3] = fma(br, vi, fma(bi, vr, acc[j][QO + 3]));
            }
          } else {  // HVPQ
            acc[j][0] += u1r;  // Q1
            acc[j][1] += u1i;
            acc[j][2] = fma(br, u1r, fma(-bi, u1i, acc[j][2]));  // Q2
            acc[j][3] = fma(br, u1i, fma(bi, u1r, acc[j][3]));
          }
        }
      }
      t += NW / NPP;
      st += NW / NPP;
      if (st >= stages) {
        st -= stages;
        ph ^= 1;
      }
    }

    // ---- end of a sample: every lane holds two events of its 4 resonances; sum over the event lanes (e) and over the
    //      slice pair members that share a resonance?  No: a resonance belongs to ONE slice; sum over e only ----------
    const int row_len = R * NACC + 2;
    double* out = a.partial + ((size_t)smp * gridDim.x + blockIdx.x) * (size_t)row_len;
    double* mine = red + (size_t)w * row_len;
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const int r = j * SW + s;
#pragma unroll
      for (int q = 0; q < NACC; ++q) {
        double tsum = acc[j][q];
#pragma unroll
        for (int m = 1; m < EW; m <<= 1) tsum += shfl_x(tsum, m);
        if (e == 0 && r < R) mine[r * NACC + q] = tsum;
        acc[j][q] = 0.0;
      }
    }
    {
      double t0 = s0, t1 = s1;  // counted by the lanes of slices 0 and 1 only: lanes 0 .. 2 EW - 1
#pragma unroll
      for (int m = 1; m < 2 * EW; m <<= 1) {
        t0 += shfl_x(t0, m);
        t1 += shfl_x(t1, m);
      }
      if (lane == 0) {
        mine[R * NACC] = t0;
        mine[R * NACC + 1] = t1;
      }
      s0 = s1 = 0.0;
    }
    asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
    for (int k = w * 32 + lane; k < row_len; k += NW * 32) {
      double tsum = red[k];
      for (int ww = 1; ww < NW; ++ww) tsum += red[(size_t)ww * row_len + k];
      out[k] = tsum;
    }
    asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
  }
}

}  // namespace lanes
}  // namespace pwa
