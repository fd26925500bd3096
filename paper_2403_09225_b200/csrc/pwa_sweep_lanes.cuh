// pwa_sweep_lanes.cuh - the warp-autonomous sweep kernel of the hot path (SURVEY §8(a) rows a-1 .. a-7), sm_100a.
//
// Work decomposition.  A tile is 32 consecutive events (8 for the large shapes, see k_sweep_lanes).  Tiles reach shared
// memory through a ring of stages filled by up to four producer threads (one per warp of the producer warpgroup, taking
// the tiles in turn) with TMA tensor copies (cp.async.bulk.tensor.2d): one box of 32 events x all R*H amplitude planes
// (512 contiguous bytes per plane; narrower boxes were measured to cap the feed near 4.1 TB/s), one box for the mass
// planes, one for the weights - or, from a library-owned tiled store, with ONE bulk copy per stage; full[stage] /
// empty[stage] mbarriers track the ring; events beyond the ragged end and the planes of padding resonances are
// zero-filled by the TMA unit.  Every F element is read from HBM exactly once and is consumed by exactly one thread.
//
// A compute warp works on one "pass" at a time: EW = 32 / SW consecutive events of a tile, the R resonances dealt
// over SW "slices" of RHO resonances each.  lane = s * EW + e (slice s, event e); lane (s, e) owns the resonances
// r = j * SW + s, j < RHO.  Per pass a lane
//   forward : B_r = 1/D_r (a-1), G_rh = B_r F_rh, slice-partial A_h = sum c_r G_rh, Adot_h = sum (alpha_r + beta_r B_r) G_rh
//             (a-2); F is now in registers, the stage is released
//   exchange: the 2H (4H with the HVP) real partials are summed over the SW slices INSIDE THE WARP: a shuffle
//             reduce-scatter over the slice bits of the lane id, then every lane stores the total it holds into the
//             warp's exchange row and reads all of them back (__syncwarp only; fixed order)
//   event   : I = sum |A_h|^2; data: ln I, omega = w / I, kappa = Idot / I  (a-3, a-4)
//   backward: B S_r = sum_h conj(omega A_h) G_rh, B S'_r = sum_h conj(omega (Adot_h - kappa A_h)) G_rh, and from them the
//             compact sums P1, P2, P3, Q1, Q2 of pwa_common.cuh (a-5, a-6; which of them: the MODE) in per-lane registers
// Warps never wait for one another: the only synchronisation inside the tile loop is the TMA ring.  At the end of
// each sample the accumulators are summed over the event lanes (butterfly), over the warps of the block (shared
// memory, fixed order) and written as one partial row per block (a-7, first stage).
#pragma once
#include <cuda.h>

#include "pwa_common.cuh"

namespace pwa {

struct alignas(64) LaneArgs {
  CUtensorMap tm_amp[2], tm_mass[2], tm_wgt[2];  // 0 = MC, 1 = data
  long long n[2];
  int weighted;  // data events carry weights
  const double* theta;
  const double* v;
  const double* skip;  // optional device scalar: a non-zero value turns this launch into a no-op (speculative CG
                       // iterations of the fit driver enqueued before the previous iteration's verdict is known)
  const int* ch;
  double* partial;  // [2][gridDim.x][R*NACC + 2]
  const unsigned char* tiled[2];  // PROD 4: the library-owned tiled stores (TiledDev, pwa_common.cuh), tile stride = stage_bytes
  int R, C, stages;
  int nprod;  // warps of the producer warpgroup that issue copies (1 .. 4; PWA_NPROD)
  int nbox, rows_box;                       // amplitude rows are loaded in nbox boxes of rows_box rows (<= 256)
  unsigned stage_bytes, amp_bytes, off_mass, off_wgt;  // inside a stage: amplitude planes [rows][32 events], mass, weights
  unsigned off_K, off_red, off_bar, off_xch;  // after the stages; xch: [NW][32/SW events][4H + 2] doubles
};

namespace lanes {

constexpr int TILE32 = 32;     // events per tile (a shape with 6.4 KB per event uses 8-event tiles, see k_sweep_lanes)
#ifdef PWA_DEBUG_NOLOAD           // timing experiments only: no TMA traffic, compute on whatever the stages hold
constexpr bool kNoLoad = true;
#else
constexpr bool kNoLoad = false;
#endif
constexpr int KS = 10;         // doubles of constants per resonance

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
// arrive by the lanes for which `who` is zero, as ONE predicated instruction (no divergent branch around it)
__device__ __forceinline__ void mbar_arrive_if_zero(uint32_t bar, uint32_t who) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.eq.u32 p, %1, 0;\n"
      "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n"
      "}\n" ::"r"(bar),
      "r"(who)
      : "memory");
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
// non-blocking probe of a phase (acquire): true once the phase with this parity has completed
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
// TMA tensor copy global -> shared, completion counted in bytes on an mbarrier (SASS: UTMALDG)
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}
// bulk copy of `bytes` contiguous bytes global -> shared (16-byte aligned, a multiple of 16), completion counted on an
// mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// 1/d for normal-range positive d: hardware seed (MUFU.RCP64H) and one cubic Newton step; measured maximum
// relative error against the IEEE division 2.2e-16 (kernels).  Three DFMA, no slow-path branch.
__device__ __forceinline__ double fast_rcp(double d) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  const double e = fma(-d, y, 1.0);
  const double p = fma(e, e, e);
  return fma(y, p, y);
}

__device__ __forceinline__ double shfl_x(double x, int m) { return __shfl_xor_sync(0xffffffffu, x, m); }

// Sum of v[0..N) over the lanes that differ in the bits MASK, 2 MASK, ..., 16 of the lane id; every lane ends
// with all N totals.  Even N: one reduce-scatter step (each half of the pair keeps half of the values), recurse,
// then the matching all-gather step.  Odd N: plain butterfly step.  The order of additions is fixed.
template <int N, int MASK>
__device__ __forceinline__ void slice_allreduce(double (&v)[N], int lane) {
  if constexpr (MASK <= 16) {
    if constexpr (N % 2 == 0) {
      constexpr int HF = N / 2;
      const bool up = (lane & MASK) != 0;
      double keep[HF];
#pragma unroll
      for (int i = 0; i < HF; ++i) {
        const double send = up ? v[i] : v[i + HF];
        const double mine = up ? v[i + HF] : v[i];
        keep[i] = mine + shfl_x(send, MASK);
      }
      slice_allreduce<HF, MASK * 2>(keep, lane);
#pragma unroll
      for (int i = 0; i < HF; ++i) {
        const double other = shfl_x(keep[i], MASK);
        v[i] = up ? other : keep[i];
        v[i + HF] = up ? keep[i] : other;
      }
    } else {
#pragma unroll
      for (int i = 0; i < N; ++i) v[i] += shfl_x(v[i], MASK);
      slice_allreduce<N, MASK * 2>(v, lane);
    }
  }
}

// First half of the exchange: reduce-scatter of v[0..N) over the slice bits MASK, 2 MASK, ..., 16 of the lane id
// (even N: each half of a lane pair keeps half of the values; odd N: butterfly), then every lane stores the totals
// it ends up with at their component index in dst (this event's row of the warp's exchange buffer).  The second
// half is a plain 128-bit read of the row after __syncwarp(): 1 STS + NV/2 LDS instead of NV - 1 shuffles with
// two selects each.  The order of additions is fixed.
template <int N, int MASK>
__device__ __forceinline__ void slice_reduce_store(double (&v)[N], int lane, double* dst) {
  if constexpr (MASK <= 16) {
    if constexpr (N % 2 == 0) {
      constexpr int HF = N / 2;
      const bool up = (lane & MASK) != 0;
      double keep[HF];
#pragma unroll
      for (int i = 0; i < HF; ++i) {
        const double send = up ? v[i] : v[i + HF];
        const double mine = up ? v[i + HF] : v[i];
        keep[i] = mine + shfl_x(send, MASK);
      }
      slice_reduce_store<HF, MASK * 2>(keep, lane, dst + (up ? HF : 0));
    } else {
#pragma unroll
      for (int i = 0; i < N; ++i) v[i] += shfl_x(v[i], MASK);
      slice_reduce_store<N, MASK * 2>(v, lane, dst);
    }
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) dst[i] = v[i];
  }
}

// per-resonance constants, packed in pairs for 128-bit shared loads:
//   k[0..1] = M^2, (M Gamma)^2   k[2] = M Gamma   k[3] = bits: byte offset of the resonance's mass row in a stage
//   k[4..5] = c   k[6..7] = alpha   k[8..9] = beta          (definitions: pwa_common.cuh)
__device__ __forceinline__ void resonance_constants(const double* __restrict__ theta, const double* __restrict__ v,
                                                    int r, long long mass_off, double* k) {
  const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
  double s, c;
  sincos(phi, &s, &c);
  const cplx e = {c, s};
  const cplx cc = {a * c, a * s};
  k[0] = M * M;
  k[1] = (M * G) * (M * G);
  // Events beyond the ragged end read zero-filled masses and amplitudes: |D|^2 = M^4 + (M Gamma)^2 there.  A resonance
  // with M = 0 exactly would give 1/0 * 0 = NaN on those lanes; a denominator floor far below any m^4 keeps them at 0.
  if (k[0] == 0.0 && k[1] == 0.0) k[1] = 1e-300;
  k[2] = M * G;
  k[3] = __longlong_as_double(mass_off);
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

template <int MODE>
__host__ __device__ constexpr int nacc_of() {
  return MODE == MODE_NLL ? 0 : vpr_of(MODE);
}
// NW compute warps + 1 producer warp per block; (NW + 1) / 4 warps share one SM sub-partition's 16 K registers,
// so NW = 7 / 11 / 15 allows 255 / 168 / 128 registers per thread.

// ------------------------------------------------------------------------------------------------------
// PROD selects who feeds the ring:
//   0  warp NW is a dedicated producer (NW + 1 warps; with NW = 7 one SM sub-partition has a single compute warp);
//      (a variant without any producer warp, the compute warp of column 0 issuing the copies, was measured slower:
//      the feed then waits for that warp's turn);
//   3  as 0, but without per-warp reduction rows in shared memory (the warps add into the block's partial row in
//      turn): the shape a handle uses for its gradient modes beside its main shape, whose scratch it shares;
//   2  producer warpgroup: warps 0..3 shrink to 24 registers (setmaxnreg.dec), warp 0 produces; the NW compute warps
//      4..NW+3 grow to 240 registers (setmaxnreg.inc), so every sub-partition carries NW / 4 compute warps.
//   4  as 2, fed from the library-owned TILED store (TiledDev, pwa_common.cuh) with ONE bulk copy of contiguous HBM per
//      stage instead of tensor copies of 128-byte rows (TILE = 8 only; copy-mode handles).
constexpr int lanes_threads(int nw, int prod) { return (nw + ((prod == 2 || prod == 4) ? 4 : 1)) * 32; }
//
// TILE = 32 (default): amplitude stage = [plane r*H + h][32 events], 512-byte rows, one or two 2-D boxes.
// TILE = 8 (shapes whose 32-event tile does not fit twice in shared memory, e.g. R = 100, H = 4: 6.4 KB per event):
//   amplitude stage = [h][resonance slot][8 events] written by ONE 3-D box with the 128-byte swizzle (16-byte chunk
//   index XOR (row & 7)); the 8 lanes of a quarter-warp own consecutive resonance slots, so their 128-bit reads hit
//   eight different chunks (conflict-free).  128-byte rows cap the TMA feed near 4.1 TB/s whatever the ring depth
//   (measured with this layout on config 3 in NLL mode: 0.62 of the HBM peak against 1.05 for 512-byte rows), so
//   this variant is only chosen when the 32-event tile does not fit; config 4 on a BORROWED store runs at that cap.
// TILE = 8, PROD = 4 (the same shapes on a library-owned copy of the events): the store itself is kept as 8-event tiles
//   in the layout of a stage (TiledDev: [resonance][h][8 events], chunk e ^ phase(r), then masses and weights), so one
//   bulk copy of ~50 contiguous KB fills a stage: no 128-byte-row cap, no padding rows in shared memory (the lanes of
//   padding resonances re-read the last real row and multiply it by zero constants), one stage more in the ring.
template <int H, int RHO, int LOG_SW, int NW, int MODE, int PROD, int TILE>
__global__ void __launch_bounds__(lanes_threads(NW, PROD), 1) k_sweep_lanes(const __grid_constant__ LaneArgs a) {
  constexpr int SW = 1 << LOG_SW;          // slices per warp
  constexpr int EW = 32 / SW;              // events per pass
  constexpr int NP = TILE / EW;            // passes per tile
  static_assert(TILE == 32 || (TILE == 8 && SW >= 8), "8-event tiles need at least 8 slices (swizzle phase = slice & 7)");
  constexpr bool WG = PROD == 2 || PROD == 4;  // producer warpgroup
  constexpr bool BULK = PROD == 4;             // stages filled by one bulk copy from the tiled store
  static_assert(!BULK || TILE == 8, "the tiled store holds 8-event tiles");
  constexpr bool WP = mode_p(MODE), WP3 = mode_p3(MODE), WQ = mode_q(MODE);
  constexpr int QO = MODE == MODE_FULL ? 6 : 0;  // first accumulator of Q1 (FULL: after P1..P3; HVPQ: the only ones)
  constexpr int NV = (WQ ? 4 : 2) * H;  // reals exchanged per event and slice
  constexpr int NACC = nacc_of<MODE>();
  constexpr int NA = NACC > 0 ? NACC : 1;
  constexpr int RP = RHO * SW;             // resonances incl. padding
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  if (a.skip != nullptr && *a.skip != 0.0) return;  // uniform over the grid
  const int lane = threadIdx.x & 31, w = (int)(threadIdx.x >> 5) - (WG ? 4 : 0);  // w: compute-warp index
  const int R = a.R, stages = a.stages;
  double* Ks = reinterpret_cast<double*>(smem_raw + a.off_K);    // [RP][KS]
  double* red = reinterpret_cast<double*>(smem_raw + a.off_red);  // [NW][R*NACC + 2]
  const uint32_t full0 = smem_u32(smem_raw + a.off_bar), empty0 = full0 + 8 * stages;

  // ---- block setup: constants from theta (and v), barriers -----------------------------------------------
  for (int r = threadIdx.x; r < RP; r += blockDim.x) {
    double* k = Ks + r * KS;
    if (r < R) {
      resonance_constants(a.theta, WQ ? a.v : nullptr, r, (long long)a.off_mass + (long long)a.ch[r] * (TILE * 8), k);
    } else {  // padding resonance: couples to nothing, propagator finite
      k[0] = 0.0; k[1] = 1.0; k[2] = 0.0; k[3] = __longlong_as_double((long long)a.off_mass);
      k[4] = k[5] = k[6] = k[7] = k[8] = k[9] = 0.0;
    }
  }
  if (threadIdx.x == 0) {
    for (int k = 0; k < stages; ++k) {
      mbar_init(full0 + 8 * k, 1);
      mbar_init(empty0 + 8 * k, NP);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // ---- this block's tile list: MC tiles b, b+G, ... then data tiles b, b+G, ... ------------------------
  const long long nM = a.n[0], nD = a.n[1];
  const int tilesM = (int)((nM + TILE - 1) / TILE), tilesD = (int)((nD + TILE - 1) / TILE);
  const int G = gridDim.x, b = blockIdx.x;
  const int TmB = b < tilesM ? (tilesM - b + G - 1) / G : 0;
  const int TdB = b < tilesD ? (tilesD - b + G - 1) / G : 0;
  const int T = TmB + TdB;

  // ======================================= producer ========================================================
  // copies of local tile k into its stage st; the caller has made sure the stage is free
  auto issue_tile = [&](int k, int st) {
    const int smp = k >= TmB ? 1 : 0;
    const int i0 = (b + (k - (smp ? TmB : 0)) * G) * TILE;
    const bool wg = smp == 1 && a.weighted;
    const uint32_t bar = full0 + 8 * st, dst = smem_u32(smem_raw) + st * a.stage_bytes;
    if (BULK) {  // the tile's image in the store is the stage's image
      mbar_expect_tx(bar, a.stage_bytes);
      bulk_load(dst, a.tiled[smp] + (size_t)(i0 / TILE) * a.stage_bytes, a.stage_bytes, bar);
      return;
    }
    mbar_expect_tx(bar, a.amp_bytes + (unsigned)a.C * (TILE * 8) + (wg ? TILE * 8u : 0u));
    if (TILE == 32) {
      for (int x = 0; x < a.nbox; ++x)
        tma_load_2d(dst + x * a.rows_box * (TILE * 16), &a.tm_amp[smp], 2 * i0, x * a.rows_box, bar);
    } else {
      tma_load_3d(dst, &a.tm_amp[smp], 2 * i0, 0, 0, bar);
    }
    tma_load_2d(dst + a.off_mass, &a.tm_mass[smp], i0, 0, bar);
    if (wg) tma_load_2d(dst + a.off_wgt, &a.tm_wgt[smp], i0, 0, bar);
  };
  if ((!WG && w == NW) || (WG && w < 0)) {
    if (WG) asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
    // The warps of a producer warpgroup take the local tiles in turn (warp p: tiles p, p + NPW, ...): one thread issuing
    // every tile's copies caps the ring near one tile per 800 cycles, which bounds the shapes with small tiles (a few
    // KB per 32 events) below the feed and below their arithmetic.  Tiles need no order among themselves: a stage's
    // empty barrier alone guards its reuse.
    const int NPW = WG ? a.nprod : 1, p0 = WG ? w + 4 : 0;
    if (lane == 0 && p0 < NPW && !kNoLoad) {
      if (!BULK) {
        tma_prefetch_desc(&a.tm_amp[0]);
        tma_prefetch_desc(&a.tm_mass[0]);
        tma_prefetch_desc(&a.tm_amp[1]);
        tma_prefetch_desc(&a.tm_mass[1]);
      }
      int st = p0 % stages, wrap = p0 / stages;  // stage of tile k and how often the ring has wrapped before it
      for (int k = p0; k < T; k += NPW) {
        if (wrap > 0) mbar_wait(empty0 + 8 * st, (uint32_t)((wrap - 1) & 1));
        issue_tile(k, st);
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
  if (WG) asm volatile("setmaxnreg.inc.sync.aligned.u32 240;");
  const int s = lane >> (5 - LOG_SW), e = lane & (EW - 1);
  double acc[RHO][NA];
  double s0 = 0.0, s1 = 0.0;
#pragma unroll
  for (int j = 0; j < RHO; ++j)
#pragma unroll
    for (int q = 0; q < NA; ++q) acc[j][q] = 0.0;
  // byte offset of (resonance 0 of this slice, helicity 0, this lane's event in column 0) inside a stage; resonance j,
  // helicity h and the column add compile-time / warp-uniform constants
  const unsigned lane_f = TILE == 32 ? (unsigned)s * (H * TILE * 16) + (unsigned)e * 16u : BULK ? 0u : (unsigned)s * 128u;
  // tiled store: byte offset of each own resonance's first row inside a stage; the lanes of padding resonances (slot >=
  // R: zero constants) read the last real row instead of rows the stage does not have
  unsigned rowoff[BULK ? RHO : 1];
  if (BULK) {
#pragma unroll
    for (int j = 0; j < RHO; ++j) rowoff[j] = (unsigned)min(j * SW + s, a.R - 1) * (H * 128u);
  }
  const double* lane_k = Ks + s * KS;
  unsigned moff[RHO];  // byte offset of each own resonance's mass row inside a stage (kept in registers: no dependent load)
#pragma unroll
  for (int j = 0; j < RHO; ++j) moff[j] = (unsigned)__double_as_longlong(lane_k[j * (SW * KS) + 3]);
  // with the producer warpgroup the compute warps own 240 registers: keep the constants every pass needs in
  // registers instead of re-reading them from shared memory (one wavefront per 4 bytes per lane, broadcast or not)
  constexpr bool KREG = WG && RHO * H <= 9;  // beyond that the amplitudes G_rh themselves fill the file
  // MODE_HVPQ holds 24 fewer accumulators per lane than the fused mode: alpha, beta live in registers there too
  // (in the fused mode the same change measured 4 % slower: no room)
  constexpr int KAB = (KREG && MODE == MODE_HVPQ) ? RHO : 0;
  double2 creg[RHO], k01reg[RHO], alreg[KAB > 0 ? KAB : 1], bereg[KAB > 0 ? KAB : 1];
  double mgreg[RHO];
#pragma unroll
  for (int j = 0; j < KAB; ++j) {
    const double2* kk = reinterpret_cast<const double2*>(lane_k + j * (SW * KS));
    alreg[j] = kk[3];
    bereg[j] = kk[4];
  }
  if (KREG) {
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const double2* kk = reinterpret_cast<const double2*>(lane_k + j * (SW * KS));
      k01reg[j] = kk[0];
      mgreg[j] = lane_k[j * (SW * KS) + 2];
      creg[j] = kk[2];
    }
  }
  // this event's exchange row; rows are 4H + 2 doubles apart so that the EW rows a warp reads back together start in
  // different banks (at 4H doubles the read-back of H = 2 had a 2-way conflict: 8 wavefronts per load instead of 4)
  double* xrow = reinterpret_cast<double*>(smem_raw + a.off_xch) + ((size_t)w * EW + e) * (4 * H + 2);

  // pass g = w + k NW  ->  local tile t = g / NP, column col = g % NP.  When NW is a multiple of NP a warp keeps
  // its column for the whole sweep (FIXCOL): the event index, the amplitude and mass offsets inside a stage are then
  // loop constants and a pass only adds the stage base.
  constexpr bool FIXCOL = NW % NP == 0;
  int t = w / NP, col = w % NP;
  int st = t % stages, ph = (t / stages) & 1;

  // Propagators of one pass (a-1): B_r = conj(D_r)/|D_r|^2 for this lane's RHO resonances and its event of column
  // col_ of the tile in stage st_.
  auto propagators = [&](int st_, int col_, double2 (&Bo)[RHO]) {
    const unsigned char* sp_ = smem_raw + (size_t)st_ * a.stage_bytes;
    const int ev_ = col_ * EW + e;
#pragma unroll
    for (int j = 0; j < RHO; ++j) {
      const double2* kk = reinterpret_cast<const double2*>(lane_k + j * (SW * KS));
      const double2 k01 = KREG ? k01reg[j] : kk[0];
      const double mg = KREG ? mgreg[j] : lane_k[j * (SW * KS) + 2];
      const double m = *reinterpret_cast<const double*>(sp_ + moff[j] + ev_ * 8);
      const double xx = fma(-m, m, k01.x);
      const double den = fma(xx, xx, k01.y);  // > 0 also on the zero-filled lanes beyond the ragged end
      const double u = fast_rcp(den);
      Bo[j] = make_double2(xx * u, mg * u);  // B = conj(D)/|D|^2
    }
  };
  for (int smp = 0; smp < 2; ++smp) {
    const int t_end = smp ? T : TmB;
    const int n = (int)(smp ? nD : nM);
    const bool weighted = smp == 1 && a.weighted;
#pragma unroll 1
    while (t < t_end) {
      const int i0 = (b + (t - (smp ? TmB : 0)) * G) * TILE;  // < 2^30 (lanes_configure)
      const int ev = col * EW + e;
      const bool valid = i0 + ev < n;
      if (!kNoLoad) mbar_wait(full0 + 8 * st, (uint32_t)ph);
      const unsigned char* sp = smem_raw + (size_t)st * a.stage_bytes;
      // TILE 32: row (j SW + s) H + h, column chunk col EW + e;  TILE 8: row h RP + j SW + s, chunk (col EW + e) ^ (s & 7);
      // tiled store: row (j SW + s) H + h, chunk (col EW + e) ^ ((s EW) & 7)
      const unsigned char* fp = sp + lane_f + (TILE == 32 ? (col * EW) * 16 : (((col * EW + e) ^ ((BULK ? s * EW : s) & 7)) * 16));
      auto f_at = [&](int j, int h) {
        if (BULK) return *reinterpret_cast<const double2*>(fp + rowoff[j] + h * 128);
        return *reinterpret_cast<const double2*>(fp + (TILE == 32 ? (j * SW * H + h) * (TILE * 16) : (h * RP + j * SW) * 128));
      };
      double wt = 1.0;
      if (weighted) wt = reinterpret_cast<const double*>(sp + a.off_wgt)[ev];

      // ---------------- forward ----------------
      double2 Gr[RHO][H], Br[RHO];
      double x[NV];  // slice partials: A_h (re, im) [then Adot_h (re, im)]
      propagators(st, col, Br);
#pragma unroll
      for (int j = 0; j < RHO; ++j) {
        const double2* kk = reinterpret_cast<const double2*>(lane_k + j * (SW * KS));
        const double2 c = KREG ? creg[j] : kk[2];
        const double br = Br[j].x, bi = Br[j].y;
        if (MODE == MODE_NLL) {
          const double zr = fma(c.x, br, -(c.y * bi)), zi = fma(c.x, bi, c.y * br);
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = f_at(j, h);
            if (j == 0) {
              x[2 * h] = fma(zr, F.x, -(zi * F.y));
              x[2 * h + 1] = fma(zr, F.y, zi * F.x);
            } else {
              x[2 * h] = fma(zr, F.x, fma(-zi, F.y, x[2 * h]));
              x[2 * h + 1] = fma(zr, F.y, fma(zi, F.x, x[2 * h + 1]));
            }
          }
        } else {
          double wr = 0.0, wi = 0.0;
          if (WQ) {  // zdot = (alpha + beta B) B
            const double2 al = j < KAB ? alreg[j < KAB ? j : 0] : kk[3], be = j < KAB ? bereg[j < KAB ? j : 0] : kk[4];
            wr = fma(be.x, br, fma(-be.y, bi, al.x));
            wi = fma(be.x, bi, fma(be.y, br, al.y));
          }
#pragma unroll
          for (int h = 0; h < H; ++h) {
            const double2 F = f_at(j, h);
            const double gx = fma(br, F.x, -(bi * F.y)), gy = fma(br, F.y, bi * F.x);
            Gr[j][h] = make_double2(gx, gy);
            if (j == 0) {
              x[2 * h] = fma(c.x, gx, -(c.y * gy));
              x[2 * h + 1] = fma(c.x, gy, c.y * gx);
              if (WQ) {
                x[2 * H + 2 * h] = fma(wr, gx, -(wi * gy));
                x[2 * H + 2 * h + 1] = fma(wr, gy, wi * gx);
              }
            } else {
              x[2 * h] = fma(c.x, gx, fma(-c.y, gy, x[2 * h]));
              x[2 * h + 1] = fma(c.x, gy, fma(c.y, gx, x[2 * h + 1]));
              if (WQ) {
                x[2 * H + 2 * h] = fma(wr, gx, fma(-wi, gy, x[2 * H + 2 * h]));
                x[2 * H + 2 * h + 1] = fma(wr, gy, fma(wi, gx, x[2 * H + 2 * h + 1]));
              }
            }
          }
        }
      }
      // everything this pass needs from the stage is in registers: hand the column back to the producer
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

      // ---------------- event: I, and for data ln I, omega, kappa ----------------
      double I = 0.0;
#pragma unroll
      for (int h = 0; h < H; ++h)
        I = h == 0 ? fma(x[0], x[0], x[1] * x[1]) : fma(x[2 * h], x[2 * h], fma(x[2 * h + 1], x[2 * h + 1], I));
      if (smp == 0) {
        s0 += I;  // lanes beyond the ragged end read zero-filled F: I = 0 and no contribution below
      } else {
        const double wv = valid ? wt : 0.0;
        const double Iv = valid ? I : 1.0;
        const double inv = 1.0 / Iv;
        const double om = wv * inv;
        if (MODE != MODE_HVPQ) s0 = fma(wv, log(Iv), s0);  // HVPQ: the scalars come from the cached gradient evaluation
        s1 += wv;
        double kap = 0.0;
        if (WQ) {
          double Idot = 0.0;
#pragma unroll
          for (int h = 0; h < H; ++h)
            Idot = fma(x[2 * h], x[2 * H + 2 * h], fma(x[2 * h + 1], x[2 * H + 2 * h + 1], Idot));
          kap = 2.0 * Idot * inv;
        }
#pragma unroll
        for (int h = 0; h < H; ++h) {
          if (WQ) {
            x[2 * H + 2 * h] = om * fma(-kap, x[2 * h], x[2 * H + 2 * h]);
            x[2 * H + 2 * h + 1] = om * fma(-kap, x[2 * h + 1], x[2 * H + 2 * h + 1]);
          }
          x[2 * h] *= om;
          x[2 * h + 1] *= om;
        }
      }

      // ---------------- backward ----------------
      if (MODE != MODE_NLL) {
#pragma unroll
        for (int j = 0; j < RHO; ++j) {
          const double br = Br[j].x, bi = Br[j].y;
          if (WP) {  // t1 = B S = sum_h conj(A_h) G_h
            double t1r, t1i;
            {
              const double2 g = Gr[j][0];
              t1r = fma(x[0], g.x, x[1] * g.y);
              t1i = fma(x[0], g.y, -(x[1] * g.x));
            }
#pragma unroll
            for (int h = 1; h < H; ++h) {
              const double2 g = Gr[j][h];
              t1r = fma(x[2 * h], g.x, fma(x[2 * h + 1], g.y, t1r));
              t1i = fma(x[2 * h], g.y, fma(-x[2 * h + 1], g.x, t1i));
            }
            acc[j][0] += t1r;  // P1
            acc[j][1] += t1i;
            if (!WP3) {
              acc[j][2] = fma(br, t1r, fma(-bi, t1i, acc[j][2]));  // P2
              acc[j][3] = fma(br, t1i, fma(bi, t1r, acc[j][3]));
            } else {
              const double t2r = fma(br, t1r, -(bi * t1i)), t2i = fma(br, t1i, bi * t1r);
              acc[j][2] += t2r;  // P2
              acc[j][3] += t2i;
              acc[j][4] = fma(br, t2r, fma(-bi, t2i, acc[j][4]));  // P3
              acc[j][5] = fma(br, t2i, fma(bi, t2r, acc[j][5]));
            }
          }
          if (WQ) {  // u1 = B S' = sum_h conj(omega (Adot_h - kappa A_h)) G_h
            double u1r, u1i;
            {
              const double2 g = Gr[j][0];
              u1r = fma(x[2 * H], g.x, x[2 * H + 1] * g.y);
              u1i = fma(x[2 * H], g.y, -(x[2 * H + 1] * g.x));
            }
#pragma unroll
            for (int h = 1; h < H; ++h) {
              const double2 g = Gr[j][h];
              u1r = fma(x[2 * H + 2 * h], g.x, fma(x[2 * H + 2 * h + 1], g.y, u1r));
              u1i = fma(x[2 * H + 2 * h], g.y, fma(-x[2 * H + 2 * h + 1], g.x, u1i));
            }
            acc[j][QO] += u1r;  // Q1
            acc[j][QO + 1] += u1i;
            acc[j][QO + 2] = fma(br, u1r, fma(-bi, u1i, acc[j][QO + 2]));  // Q2
            acc[j][QO + 3] = fma(br, u1i, fma(bi, u1r, acc[j][QO + 3]));
          }
        }
      }

      // ---------------- next pass of this warp ----------------
      if (FIXCOL) {
#pragma unroll
        for (int k = 0; k < NW / NP; ++k) {
          ++t;
          if (++st == stages) {
            st = 0;
            ph ^= 1;
          }
        }
      } else {
        col += NW;
        while (col >= NP) {
          col -= NP;
          ++t;
          if (++st == stages) {
            st = 0;
            ph ^= 1;
          }
        }
      }
    }

    // ---- end of a sample: fixed-order butterfly over the event lanes, fixed-order sum over the warps, one
    //      partial row per block --------------------------------------------------------------------------------
    const int row_len = R * NACC + 2;
    double* out = a.partial + ((size_t)smp * gridDim.x + blockIdx.x) * (size_t)row_len;
    if (TILE == 32 && PROD != 3) {
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
        double t0 = s0, t1 = s1;
#pragma unroll
        for (int m = 1; m < EW; m <<= 1) {
          t0 += shfl_x(t0, m);
          t1 += shfl_x(t1, m);
        }
        if (lane == 0) {  // slice 0, event lane 0
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
    } else {
      // no per-warp rows in shared memory (large shapes, or a shape with more warps than the handle's main one):
      // ONE row in shared memory: warp 0 writes it, warp 1 adds, ... (fixed order, one named barrier per turn)
#pragma unroll 1
      for (int turn = 0; turn < NW; ++turn) {
        if (w == turn) {
#pragma unroll
          for (int j = 0; j < RHO; ++j) {
            const int r = j * SW + s;
#pragma unroll
            for (int q = 0; q < NACC; ++q) {
              double tsum = acc[j][q];
#pragma unroll
              for (int m = 1; m < EW; m <<= 1) tsum += shfl_x(tsum, m);
              if (e == 0 && r < R) red[r * NACC + q] = turn == 0 ? tsum : red[r * NACC + q] + tsum;
              acc[j][q] = 0.0;
            }
          }
          double t0 = s0, t1 = s1;
#pragma unroll
          for (int m = 1; m < EW; m <<= 1) {
            t0 += shfl_x(t0, m);
            t1 += shfl_x(t1, m);
          }
          if (lane == 0) {
            red[R * NACC] = turn == 0 ? t0 : red[R * NACC] + t0;
            red[R * NACC + 1] = turn == 0 ? t1 : red[R * NACC + 1] + t1;
          }
          s0 = s1 = 0.0;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
      }
      for (int k = w * 32 + lane; k < row_len; k += NW * 32) out[k] = red[k];
      asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
    }
  }
}

}  // namespace lanes
}  // namespace pwa
