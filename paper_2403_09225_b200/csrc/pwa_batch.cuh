// pwa_batch.cuh - K evaluations in ONE pass over the event store ("multi-start batching";
// PAPER.md:121 300 fits on the same events, :133 11+ starts per analysis, :102-113 Table 1's parameter errors).
//
// Two kinds, both on the tile / ring / lane decomposition of pwa_sweep_lanes.cuh (32-event tiles through the TMA ring,
// producer warpgroup, lane = slice x event, shuffle reduce-scatter over the slices):
//   BK_NLL  : KB parameter sets theta_0 .. theta_{KB-1}: every F element is read from HBM and from shared memory once
//             and meets KB propagators / couplings; accumulates sum I_k (MC) and sum w ln I_k (data) per set.
//             The value-only sweep is bound by the feed (and, in long runs, by the power the feed draws), so KB
//             evaluations cost little more than one.
//   BK_HVPQ : KB directions v_0 .. v_{KB-1} at ONE theta (the theta kept by pwa_nll_grad_for_hvp): the propagators,
//             G = B F and A_h are shared by the directions; per direction only zdot, Adot_h and the sums Q1, Q2.
//             23 + 26 KB FP64 instructions per (event, resonance) at H = 2 instead of 49 KB.  This is the access pattern of
//             the Hessian (pwa_hessian: P unit directions at the fitted theta, the error matrix of Table 1).
// Everything theta- and v-dependent outside the event loop is done by k_reduce_batch (one block).
#pragma once
#include "pwa_kernels.cuh"
#include "pwa_sweep_lanes.cuh"

namespace pwa {

enum BatchKind { BK_NLL = 0, BK_HVPQ = 1 };

struct BatchArgs {
  const double* theta;  // BK_NLL: [KB][P]; BK_HVPQ: [P] (the kept theta)
  const double* v;      // BK_HVPQ: [KB][P]
  double* partial;      // [2][gridDim.x][row_len]
  int stages;
  unsigned off_K, off_red, off_xch, off_bar;  // after the stages (the stage geometry itself is LaneArgs')
};

namespace lanes {

__host__ __device__ constexpr int batch_row_len(int kind, int kb, int R) { return kind == BK_NLL ? kb + 1 : R * 4 * kb; }
__host__ __device__ constexpr int batch_nv(int kind, int kb, int H) { return kind == BK_NLL ? 2 * H * kb : 2 * H * (1 + kb); }
// constants: 16-byte slots per resonance, laid out [j][slot][slice] so that the 8 (or 4) slices of a warp read 128 (64)
// contiguous bytes: one shared-memory wavefront per load (a [resonance][slot] layout put the slices 192 bytes apart:
// 4-way bank conflicts, and the value batch of 4 ran at half speed).
//   BK_NLL : per set k: slot 3k = (M^2, (M Gamma)^2), 3k+1 = (M Gamma, -), 3k+2 = c
//   BK_HVPQ: slots 0..2 as above for theta, then per direction k: 3+2k = alpha_k, 4+2k = beta_k
__host__ __device__ constexpr int batch_slots(int kind, int kb) { return kind == BK_NLL ? 3 * kb : 3 + 2 * kb; }
__host__ __device__ constexpr int batch_ks(int kind, int kb) { return 2 * batch_slots(kind, kb); }  // doubles per resonance

template <int H, int RHO, int LOG_SW, int NW, int KIND, int KB>
__global__ void __launch_bounds__(lanes_threads(NW, 2), 1) k_batch_lanes(const __grid_constant__ LaneArgs a,
                                                                         const __grid_constant__ BatchArgs b) {
  constexpr int TILE = 32;
  constexpr int SW = 1 << LOG_SW, EW = 32 / SW, NP = TILE / EW, RP = RHO * SW;
  constexpr int NV = batch_nv(KIND, KB, H);
  constexpr int NSLOT = batch_slots(KIND, KB);
  constexpr int NACC = KIND == BK_NLL ? 0 : 4 * KB;  // per own resonance: Q1, Q2 of every direction
  constexpr int NA = NACC > 0 ? NACC : 1;
  constexpr int NS0 = KIND == BK_NLL ? KB : 1;
  // PAIR (value batch, 8 slices x 4 events): a warp takes TWO columns of every second tile and a lane two events, one per
  // column, odd slices in the opposite order - see the compute section
  constexpr bool PAIR = KIND == BK_NLL && LOG_SW == 3 && NW == NP;
  static_assert(NW % NP == 0, "a warp keeps its column");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, w = (int)(threadIdx.x >> 5) - 4;  // w: compute-warp index (warps 0..3: producer group)
  const int R = a.R, stages = b.stages, P = 4 * R;
  double2* Ks = reinterpret_cast<double2*>(smem_raw + b.off_K);   // [RHO][NSLOT][SW]
  double* red = reinterpret_cast<double*>(smem_raw + b.off_red);  // [NW][row_len]
  const uint32_t full0 = smem_u32(smem_raw + b.off_bar), empty0 = full0 + 8 * stages;
  const int row_len = batch_row_len(KIND, KB, R);

  // ---- block setup: constants, barriers -------------------------------------------------------------------
  for (int r = threadIdx.x; r < RP; r += blockDim.x) {
    double2* k = Ks + (size_t)(r / SW) * (NSLOT * SW) + (r % SW);  // slot q of resonance r: k[q * SW]
    double tmp[KS];
#pragma unroll
    for (int s = 0; s < KB; ++s) {
      if (r < R) {
        if (KIND == BK_NLL) resonance_constants(b.theta + (size_t)s * P, nullptr, r, 0, tmp);
        else resonance_constants(b.theta, b.v + (size_t)s * P, r, 0, tmp);
      } else {  // padding resonance: couples to nothing, propagator finite
        tmp[0] = 0.0; tmp[1] = 1.0; tmp[2] = 0.0;
        tmp[4] = tmp[5] = tmp[6] = tmp[7] = tmp[8] = tmp[9] = 0.0;
      }
      if (KIND == BK_NLL || s == 0) {
        const int q = KIND == BK_NLL ? 3 * s : 0;
        k[(q + 0) * SW] = make_double2(tmp[0], tmp[1]);
        k[(q + 1) * SW] = make_double2(tmp[2], 0.0);
        k[(q + 2) * SW] = make_double2(tmp[4], tmp[5]);
      }
      if (KIND == BK_HVPQ) {
        k[(3 + 2 * s) * SW] = make_double2(tmp[6], tmp[7]);
        k[(4 + 2 * s) * SW] = make_double2(tmp[8], tmp[9]);
      }
    }
  }
  if (threadIdx.x == 0) {
    for (int k = 0; k < stages; ++k) {
      mbar_init(full0 + 8 * k, 1);
      mbar_init(empty0 + 8 * k, PAIR ? NP / 2 : NP);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const long long nM = a.n[0], nD = a.n[1];
  const int tilesM = (int)((nM + TILE - 1) / TILE), tilesD = (int)((nD + TILE - 1) / TILE);
  const int G = gridDim.x, bk = blockIdx.x;
  const int TmB = bk < tilesM ? (tilesM - bk + G - 1) / G : 0;
  const int TdB = bk < tilesD ? (tilesD - bk + G - 1) / G : 0;
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
        const int i0 = (bk + (k - (smp ? TmB : 0)) * G) * TILE;
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
  double s0[NS0], s1 = 0.0;
#pragma unroll
  for (int j = 0; j < RHO; ++j)
#pragma unroll
    for (int q = 0; q < NA; ++q) acc[j][q] = 0.0;
#pragma unroll
  for (int k = 0; k < NS0; ++k) s0[k] = 0.0;
  const unsigned lane_f = (unsigned)s * (H * TILE * 16) + (unsigned)e * 16u;
  const double2* lane_k = Ks + s;  // slot q of own resonance j: lane_k[(j * NSLOT + q) * SW]
  unsigned moff[RHO];  // byte offset of each own resonance's mass row inside a stage
#pragma unroll
  for (int j = 0; j < RHO; ++j) {
    const int r = j * SW + s;
    moff[j] = a.off_mass + (unsigned)(r < R ? a.ch[r] : 0) * (TILE * 8);
  }
  // Constants in registers where the file has room (a shared load costs one wavefront per 4 bytes per lane, broadcast or
  // not: the value batch of 4 spends 160 of its 240 wavefronts per pass on constants, its shared-memory pipe is 82 % busy;
  // but 80 doubles of constants per lane cost more in lost instruction-level parallelism than they save).
  constexpr int NKR = KIND == BK_NLL ? KB : 1;
  constexpr bool KREG = KIND == BK_NLL && RHO * KB <= 8;  // measured: helps the batch of 2 (-5 %), hurts 4 sets and the direction batches
  double2 k01r[RHO][NKR], cr[RHO][NKR];
  double mgr[RHO][NKR];
#pragma unroll
  for (int j = 0; j < RHO; ++j)
#pragma unroll
    for (int k = 0; k < (KREG ? NKR : 0); ++k) {
      const double2* kj = lane_k + j * (NSLOT * SW);
      k01r[j][k] = kj[(3 * k) * SW];
      mgr[j][k] = kj[(3 * k + 1) * SW].x;
      cr[j][k] = kj[(3 * k + 2) * SW];
    }
  // rows padded by 16 bytes: the EW event rows a warp reads back together start in different banks
  double* xrow = reinterpret_cast<double*>(smem_raw + b.off_xch) + ((size_t)w * EW + e) * (NV + 2);

  if constexpr (PAIR) {
    // ---- value batch, two events per lane -----------------------------------------------------------------------
    // Warp w takes the column pair cp = w % 4 of the local tiles w / 4, w / 4 + 2, ...  A lane evaluates its RHO x KB
    // propagators for TWO events: even slices first column 2cp then 2cp + 1, odd slices the other way round.  Then
    //   - the constants of a (resonance, set) are read once for two events;
    //   - a quarter-warp (two slices x four events) reads 128 CONTIGUOUS bytes of a plane row: no bank conflict
    //     (with one column per warp the two slices hit the same banks);
    //   - the first exchange level needs no selects: both lanes of a slice pair keep their first event and send the second;
    //   - the event stage (I, ln I) runs once per event and slice pair instead of once per slice.
    constexpr int NPP = NP / 2;
    const int cp = w % NPP;
    const int colA = 2 * cp + (s & 1), colB = 2 * cp + ((s & 1) ^ 1);
    const int evA = colA * EW + e, evB = colB * EW + e;
    double* xrowp = reinterpret_cast<double*>(smem_raw + b.off_xch) + ((size_t)w * EW + e) * (NV + 2) +
                    (size_t)(s & 1) * ((size_t)NW * EW * (NV + 2));  // second half of the buffer: odd slices' events
    int t = w / NPP;
    int st = t % stages, ph = (t / stages) & 1;
    for (int smp = 0; smp < 2; ++smp) {
      const int t_end = smp ? T : TmB;
      const int n = (int)(smp ? nD : nM);
      const bool weighted = smp == 1 && a.weighted;
#pragma unroll 1
      while (t < t_end) {
        const int i0 = (bk + (t - (smp ? TmB : 0)) * G) * TILE;
        const bool valid = i0 + evA < n;
        mbar_wait(full0 + 8 * st, (uint32_t)ph);
        const unsigned char* sp = smem_raw + (size_t)st * a.stage_bytes;
        const unsigned char* fpA = sp + (unsigned)s * (H * TILE * 16) + evA * 16;
        const unsigned char* fpB = sp + (unsigned)s * (H * TILE * 16) + evB * 16;
        double wt = 1.0;
        if (weighted) wt = reinterpret_cast<const double*>(sp + a.off_wgt)[evA];
        double xa[NV], xb[NV];
#pragma unroll
        for (int j = 0; j < RHO; ++j) {
          const double2* kj = lane_k + j * (NSLOT * SW);
          const double mA = *reinterpret_cast<const double*>(sp + moff[j] + evA * 8);
          const double mB = *reinterpret_cast<const double*>(sp + moff[j] + evB * 8);
          double2 FA[H], FB[H];
#pragma unroll
          for (int h = 0; h < H; ++h) {
            FA[h] = *reinterpret_cast<const double2*>(fpA + (j * SW * H + h) * (TILE * 16));
            FB[h] = *reinterpret_cast<const double2*>(fpB + (j * SW * H + h) * (TILE * 16));
          }
#pragma unroll
          for (int k = 0; k < KB; ++k) {
            const double2 k01 = kj[(3 * k) * SW];
            const double mg = kj[(3 * k + 1) * SW].x;
            const double2 c = kj[(3 * k + 2) * SW];
#pragma unroll
            for (int side = 0; side < 2; ++side) {
              const double m = side ? mB : mA;
              const double xx = fma(-m, m, k01.x);
              const double u = fast_rcp(fma(xx, xx, k01.y));
              const double br = xx * u, bi = mg * u;
              const double zr = fma(c.x, br, -(c.y * bi)), zi = fma(c.x, bi, c.y * br);
#pragma unroll
              for (int h = 0; h < H; ++h) {
                const double2 F = side ? FB[h] : FA[h];
                double* xk = (side ? xb : xa) + 2 * H * k + 2 * h;
                if (j == 0) {
                  xk[0] = fma(zr, F.x, -(zi * F.y));
                  xk[1] = fma(zr, F.y, zi * F.x);
                } else {
                  xk[0] = fma(zr, F.x, fma(-zi, F.y, xk[0]));
                  xk[1] = fma(zr, F.y, fma(zi, F.x, xk[1]));
                }
              }
            }
          }
        }
        __syncwarp();
        mbar_arrive_if_zero(empty0 + 8 * st, (uint32_t)lane);
        // exchange: level 1 over the slice pair (keep the first event, send the second), then the usual reduce-scatter
        // over the remaining slice bits; every lane ends with its share of the totals of ITS first event
#pragma unroll
        for (int i = 0; i < NV; ++i) xa[i] += shfl_x(xb[i], EW);
        slice_reduce_store<NV, 2 * EW>(xa, lane, xrowp);
        __syncwarp();
#pragma unroll
        for (int i = 0; i < NV; i += 2) {
          const double2 pr = *reinterpret_cast<const double2*>(xrowp + i);
          xa[i] = pr.x;
          xa[i + 1] = pr.y;
        }
        __syncwarp();
        const double wv = valid ? wt : 0.0;
#pragma unroll
        for (int k = 0; k < KB; ++k) {
          double I = 0.0;
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double* xk = xa + 2 * H * k + 2 * h;
            I = fma(xk[0], xk[0], fma(xk[1], xk[1], I));
          }
          if (smp == 0) s0[k] += I;
          else s0[k] = fma(wv, log(valid ? I : 1.0), s0[k]);
        }
        if (smp == 1) s1 += wv;
        t += NW / NPP;
        st += NW / NPP;
        if (st >= stages) {
          st -= stages;
          ph ^= 1;
        }
      }
      // end of a sample: the lanes of slices 0 and 1 (lane < 2 EW) hold every event of the warp's columns once
      double* out = b.partial + ((size_t)smp * gridDim.x + blockIdx.x) * (size_t)row_len;
      double* mine = red + (size_t)w * row_len;
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        double t0 = s0[k];
#pragma unroll
        for (int m = 1; m < 2 * EW; m <<= 1) t0 += shfl_x(t0, m);
        if (lane == 0) mine[k] = t0;
        s0[k] = 0.0;
      }
      double t1 = s1;
#pragma unroll
      for (int m = 1; m < 2 * EW; m <<= 1) t1 += shfl_x(t1, m);
      if (lane == 0) mine[KB] = t1;
      s1 = 0.0;
      asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
      for (int k = w * 32 + lane; k < row_len; k += NW * 32) {
        double tsum = red[k];
        for (int ww = 1; ww < NW; ++ww) tsum += red[(size_t)ww * row_len + k];
        out[k] = tsum;
      }
      asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
    }
    return;
  }

  const int col = w % NP;
  int t = w / NP;
  int st = t % stages, ph = (t / stages) & 1;
  const int ev = col * EW + e;

  for (int smp = 0; smp < 2; ++smp) {
    const int t_end = smp ? T : TmB;
    const int n = (int)(smp ? nD : nM);
    const bool weighted = smp == 1 && a.weighted;
#pragma unroll 1
    while (t < t_end) {
      const int i0 = (bk + (t - (smp ? TmB : 0)) * G) * TILE;
      const bool valid = i0 + ev < n;
      mbar_wait(full0 + 8 * st, (uint32_t)ph);
      const unsigned char* sp = smem_raw + (size_t)st * a.stage_bytes;
      const unsigned char* fp = sp + lane_f + (col * EW) * 16;
      double wt = 1.0;
      if (weighted) wt = reinterpret_cast<const double*>(sp + a.off_wgt)[ev];

      // ---------------- forward ----------------
      double2 Gr[KIND == BK_HVPQ ? RHO : 1][H], Br[KIND == BK_HVPQ ? RHO : 1];
      double x[NV];
#pragma unroll
      for (int j = 0; j < RHO; ++j) {
        const double2* kj = lane_k + j * (NSLOT * SW);
        const double m = *reinterpret_cast<const double*>(sp + moff[j] + ev * 8);
        double2 F[H];
#pragma unroll
        for (int h = 0; h < H; ++h) F[h] = *reinterpret_cast<const double2*>(fp + (j * SW * H + h) * (TILE * 16));
        if (KIND == BK_NLL) {
#pragma unroll
          for (int k = 0; k < KB; ++k) {
            const double2 k01 = KREG ? k01r[j][k] : kj[(3 * k) * SW];
            const double mg = KREG ? mgr[j][k] : kj[(3 * k + 1) * SW].x;
            const double2 c = KREG ? cr[j][k] : kj[(3 * k + 2) * SW];
            const double xx = fma(-m, m, k01.x);
            const double u = fast_rcp(fma(xx, xx, k01.y));
            const double br = xx * u, bi = mg * u;
            const double zr = fma(c.x, br, -(c.y * bi)), zi = fma(c.x, bi, c.y * br);
#pragma unroll
            for (int h = 0; h < H; ++h) {
              double* xk = x + 2 * H * k + 2 * h;
              if (j == 0) {
                xk[0] = fma(zr, F[h].x, -(zi * F[h].y));
                xk[1] = fma(zr, F[h].y, zi * F[h].x);
              } else {
                xk[0] = fma(zr, F[h].x, fma(-zi, F[h].y, xk[0]));
                xk[1] = fma(zr, F[h].y, fma(zi, F[h].x, xk[1]));
              }
            }
          }
        } else {
          const double2 k01 = KREG ? k01r[j][0] : kj[0];
          const double mg = KREG ? mgr[j][0] : kj[SW].x;
          const double2 c = KREG ? cr[j][0] : kj[2 * SW];
          const double xx = fma(-m, m, k01.x);
          const double u = fast_rcp(fma(xx, xx, k01.y));
          const double br = xx * u, bi = mg * u;
          Br[j] = make_double2(br, bi);
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double gx = fma(br, F[h].x, -(bi * F[h].y)), gy = fma(br, F[h].y, bi * F[h].x);
            Gr[j][h] = make_double2(gx, gy);
            if (j == 0) {
              x[2 * h] = fma(c.x, gx, -(c.y * gy));
              x[2 * h + 1] = fma(c.x, gy, c.y * gx);
            } else {
              x[2 * h] = fma(c.x, gx, fma(-c.y, gy, x[2 * h]));
              x[2 * h + 1] = fma(c.x, gy, fma(c.y, gx, x[2 * h + 1]));
            }
          }
#pragma unroll
          for (int k = 0; k < KB; ++k) {  // zdot_k = (alpha_k + beta_k B) B
            const double2 al = kj[(3 + 2 * k) * SW];
            const double2 be = kj[(4 + 2 * k) * SW];
            const double wr = fma(be.x, br, fma(-be.y, bi, al.x));
            const double wi = fma(be.x, bi, fma(be.y, br, al.y));
#pragma unroll
            for (int h = 0; h < H; ++h) {
              double* xk = x + 2 * H * (1 + k) + 2 * h;
              const double gx = Gr[j][h].x, gy = Gr[j][h].y;
              if (j == 0) {
                xk[0] = fma(wr, gx, -(wi * gy));
                xk[1] = fma(wr, gy, wi * gx);
              } else {
                xk[0] = fma(wr, gx, fma(-wi, gy, xk[0]));
                xk[1] = fma(wr, gy, fma(wi, gx, xk[1]));
              }
            }
          }
        }
      }
      __syncwarp();
      mbar_arrive_if_zero(empty0 + 8 * st, (uint32_t)lane);

      // ---------------- exchange over the slices ----------------
      slice_reduce_store<NV, EW>(x, lane, xrow);
      __syncwarp();
#pragma unroll
      for (int i = 0; i < NV; i += 2) {
        const double2 p = *reinterpret_cast<const double2*>(xrow + i);
        x[i] = p.x;
        x[i + 1] = p.y;
      }
      __syncwarp();  // the row is rewritten by the next pass

      // ---------------- event ----------------
      if (KIND == BK_NLL) {
        const double wv = valid ? wt : 0.0;
#pragma unroll
        for (int k = 0; k < KB; ++k) {
          double I = 0.0;
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double* xk = x + 2 * H * k + 2 * h;
            I = fma(xk[0], xk[0], fma(xk[1], xk[1], I));
          }
          if (smp == 0) s0[k] += I;  // lanes beyond the ragged end read zero-filled F: I = 0
          else s0[k] = fma(wv, log(valid ? I : 1.0), s0[k]);
        }
        if (smp == 1) s1 += wv;
      } else {
        double I = 0.0;
#pragma unroll
        for (int h = 0; h < H; ++h) I = fma(x[2 * h], x[2 * h], fma(x[2 * h + 1], x[2 * h + 1], I));
        if (smp == 1) {
          const double wv = valid ? wt : 0.0;
          const double inv = 1.0 / (valid ? I : 1.0);
          const double om = wv * inv;
#pragma unroll
          for (int k = 0; k < KB; ++k) {
            double* xk = x + 2 * H * (1 + k);
            double Idot = 0.0;
#pragma unroll
            for (int h = 0; h < H; ++h) Idot = fma(x[2 * h], xk[2 * h], fma(x[2 * h + 1], xk[2 * h + 1], Idot));
            const double kap = 2.0 * Idot * inv;
#pragma unroll
            for (int h = 0; h < H; ++h) {
              xk[2 * h] = om * fma(-kap, x[2 * h], xk[2 * h]);
              xk[2 * h + 1] = om * fma(-kap, x[2 * h + 1], xk[2 * h + 1]);
            }
          }
        }
        // ---------------- backward: u1 = B S'_k = sum_h conj(x'_kh) G_h ; Q1_k += u1 ; Q2_k += B u1 ----------------
#pragma unroll
        for (int j = 0; j < RHO; ++j) {
          const double br = Br[j].x, bi = Br[j].y;
#pragma unroll
          for (int k = 0; k < KB; ++k) {
            const double* xk = x + 2 * H * (1 + k);
            double u1r, u1i;
            {
              const double2 g = Gr[j][0];
              u1r = fma(xk[0], g.x, xk[1] * g.y);
              u1i = fma(xk[0], g.y, -(xk[1] * g.x));
            }
#pragma unroll
            for (int h = 1; h < H; ++h) {
              const double2 g = Gr[j][h];
              u1r = fma(xk[2 * h], g.x, fma(xk[2 * h + 1], g.y, u1r));
              u1i = fma(xk[2 * h], g.y, fma(-xk[2 * h + 1], g.x, u1i));
            }
            acc[j][4 * k + 0] += u1r;
            acc[j][4 * k + 1] += u1i;
            acc[j][4 * k + 2] = fma(br, u1r, fma(-bi, u1i, acc[j][4 * k + 2]));
            acc[j][4 * k + 3] = fma(br, u1i, fma(bi, u1r, acc[j][4 * k + 3]));
          }
        }
      }

      // next pass of this warp (fixed column)
#pragma unroll
      for (int k = 0; k < NW / NP; ++k) {
        ++t;
        if (++st == stages) {
          st = 0;
          ph ^= 1;
        }
      }
    }

    // ---- end of a sample: butterfly over the event lanes, fixed-order sum over the warps, one partial row per block
    double* out = b.partial + ((size_t)smp * gridDim.x + blockIdx.x) * (size_t)row_len;
    double* mine = red + (size_t)w * row_len;
    if (KIND == BK_HVPQ) {
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
    } else {
      // every slice holds the same event totals: only slice 0's lanes count
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        double t0 = s0[k];
#pragma unroll
        for (int m = 1; m < EW; m <<= 1) t0 += shfl_x(t0, m);
        if (lane == 0) mine[k] = t0;
        s0[k] = 0.0;
      }
      double t1 = s1;
#pragma unroll
      for (int m = 1; m < EW; m <<= 1) t1 += shfl_x(t1, m);
      if (lane == 0) mine[KB] = t1;
      s1 = 0.0;
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

// ------------------------------------------------------------------------------------------------------
// Second stage for a batch sweep (one block of 1024 threads): fixed-order column sums over the per-block partial rows
// (one warp per column, as k_reduce_unpack), then
//   BK_NLL : nll[k] = -sum_data w ln I_k + W ln(G_k / N_mc)                         (Eq. 3 / 4)
//   BK_HVPQ: per direction k the compact sums (P1..P3 kept by pwa_nll_grad_for_hvp, Q1_k, Q2_k of this sweep) -> raw
//            sums -> Eq. 7 -> hv[k][P].  braw: scratch [4 + 4P] doubles.
// ------------------------------------------------------------------------------------------------------
template <int KIND, int KB>
__global__ void __launch_bounds__(1024) k_reduce_batch(const double* __restrict__ partial, int nblocks, int R,
                                                       const double* __restrict__ theta, const double* __restrict__ v,
                                                       double n_mc, double* sums, const double* pcache, double* braw,
                                                       double* __restrict__ out, unsigned* __restrict__ flags) {
  const int stride = lanes::batch_row_len(KIND, KB, R), P = 4 * R;
  const int lane = threadIdx.x & 31, warps = blockDim.x >> 5, wid = threadIdx.x >> 5;
  for (int k = wid; k < 2 * stride; k += warps) {
    const int sample = k / stride, idx = k - sample * stride;
    const double* p = partial + (size_t)sample * nblocks * stride + idx;
    double t = 0.0;
    for (int b = lane; b < nblocks; b += 32) t += p[(size_t)b * stride];
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) t += __shfl_xor_sync(0xffffffffu, t, m);
    if (lane == 0) sums[k] = t;
  }
  __syncthreads();
  if (KIND == BK_NLL) {
    __shared__ int bad;
    if (threadIdx.x == 0) bad = 0;
    __syncthreads();
    if (threadIdx.x < KB) {
      const double Ld = sums[stride + threadIdx.x], W = sums[stride + KB], G = sums[threadIdx.x];
      const double f = -Ld + W * log(G / n_mc);
      out[threadIdx.x] = f;
      if (!isfinite(f)) atomicOr(&bad, 1);
    }
    __syncthreads();
    if (threadIdx.x == 0) *flags = bad ? 1u : 0u;
    return;
  }
  const int cstride = 6 * R + 2;
  unsigned any_bad = 0;
  for (int k = 0; k < KB; ++k) {
    if (threadIdx.x == 0) {
      braw[0] = pcache[cstride + 6 * R];      // sum_data w ln I
      braw[1] = pcache[cstride + 6 * R + 1];  // W
      braw[2] = pcache[6 * R];                // G
      braw[3] = n_mc;
    }
    for (int r = threadIdx.x; r < R; r += blockDim.x) {
      const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
      for (int sample = 0; sample < 2; ++sample) {
        const double* pc = pcache + (size_t)sample * cstride + r * 6;
        const double* q = sums + (size_t)sample * stride + r * (4 * KB) + 4 * k;
        Sums5 s;
        s.P1 = {pc[0], pc[1]};
        s.P2 = {pc[2], pc[3]};
        s.P3 = {pc[4], pc[5]};
        s.Q1 = {q[0], q[1]};
        s.Q2 = {q[2], q[3]};
        double g4[4], h4[4] = {0.0, 0.0, 0.0, 0.0};
        unpack_res(s, a, phi, M, G, v + (size_t)k * P + 4 * r, g4, h4);
        double* gdst = braw + 4 + (sample == 1 ? 0 : P) + 4 * r;
        double* hdst = braw + 4 + 2 * P + (sample == 1 ? 0 : P) + 4 * r;
        for (int c = 0; c < 4; ++c) {
          gdst[c] = g4[c];
          hdst[c] = sample == 1 ? -h4[c] : h4[c];
        }
      }
    }
    __syncthreads();
    combine_block(braw, v + (size_t)k * P, P, nullptr, nullptr, out + (size_t)k * P, flags);
    __syncthreads();
    if (threadIdx.x == 0) any_bad |= *flags;
  }
  if (threadIdx.x == 0) *flags = any_bad;
}

}  // namespace pwa
