// pwa_kernels.cuh - prologue, generic streaming sweep, reduction/unpack and combine kernels.
#pragma once
#include "pwa_common.cuh"

namespace pwa {

// ------------------------------------------------------------------------------------------------
// Prologue: per-resonance constants from theta (and v).  One thread per resonance.
// PAPER.md:60 (couplings Lambda, here a e^{i phi}); BASELINE.json configs[0] (BW form).
// ------------------------------------------------------------------------------------------------
static __global__ void k_prologue(const double* __restrict__ theta, const double* __restrict__ v, int R,
                           double* __restrict__ K) {
  int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= R) return;
  const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
  double s, c;
  sincos(phi, &s, &c);
  const cplx e = {c, s};
  const cplx cc = {a * c, a * s};
  double* k = K + (size_t)r * KSTRIDE;
  k[K_M2] = M * M;
  k[K_Y] = M * G;
  k[K_Y2] = (M * G) * (M * G);
  k[3] = 0.0;
  k[K_CR] = cc.re;
  k[K_CI] = cc.im;
  cplx al = {0.0, 0.0}, be = {0.0, 0.0};
  if (v) {
    const double va = v[4 * r], vp = v[4 * r + 1], vM = v[4 * r + 2], vG = v[4 * r + 3];
    // alpha = e v_a + i c v_phi ;  beta = c * lambda,  lambda = -(2M - iG) v_M + i M v_G
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

// ------------------------------------------------------------------------------------------------
// 32 values per lane -> lane l ends with the sum over the 32 lanes of value l (transposing butterfly).
// Fixed exchange pattern: the result does not depend on anything but the inputs (deterministic).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double bfly32(double (&v)[32], int lane) {
#pragma unroll
  for (int half = 16; half >= 1; half >>= 1) {
    const bool up = (lane & half) != 0;
#pragma unroll
    for (int j = 0; j < half; ++j) {
      const double keep = up ? v[j + half] : v[j];
      const double send = up ? v[j] : v[j + half];
      v[j] = keep + __shfl_xor_sync(0xffffffffu, send, half);
    }
  }
  return v[0];
}

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
  for (int m = 16; m >= 1; m >>= 1) x += __shfl_xor_sync(0xffffffffu, x, m);
  return x;
}

// ------------------------------------------------------------------------------------------------
// Generic sweep (any R, C; H templated).  lane = event; each warp walks rows of 32 events.
// Forward pass over all resonances gives A_h, Adot_h; the backward pass revisits the resonances in
// batches, forms the per-event compact terms and reduces each batch across the warp at once, adding
// the result to a per-warp accumulator array in shared memory (one double per lane and batch).
// SURVEY/DESIGN §8(a) rows a-1 .. a-7.
// ------------------------------------------------------------------------------------------------
template <int H, int MODE>
__global__ void __launch_bounds__(256) k_sweep_generic(const SweepArgs a) {
  constexpr int VPR = vpr_of(MODE), RPB = rpb_of(MODE);
  extern __shared__ double smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const int nacc = a.nb * 32;
  double* acc = smem + (size_t)warp * nacc;
  double* scal = smem + (size_t)nwarp * nacc;  // [nwarp][2]
  const int R = a.R;
  const double* __restrict__ K = a.K;
  const int* __restrict__ ch = a.ch;

  for (int sample = 0; sample < 2; ++sample) {
    const SampleDev s = a.s[sample];
    const bool is_data = sample == 1;
    for (int k = lane; k < nacc; k += 32) acc[k] = 0.0;
    double s0 = 0.0, s1 = 0.0;
    const long long rows = (s.n + 31) / 32;
    for (long long row = (long long)blockIdx.x * nwarp + warp; row < rows; row += (long long)gridDim.x * nwarp) {
      const long long i = row * 32 + lane;
      const bool valid = i < s.n;
      const long long ic = valid ? i : s.n - 1;
      const double2* __restrict__ amp = s.amp + ic;
      const double* __restrict__ mass = s.mass + ic;

      // ---- forward: A_h, Adot_h ------------------------------------------------------------
      double Ar[H], Ai[H], Dr[H], Di[H];
#pragma unroll
      for (int h = 0; h < H; ++h) Ar[h] = Ai[h] = Dr[h] = Di[h] = 0.0;
#pragma unroll 2
      for (int r = 0; r < R; ++r) {
        const double* k = K + (size_t)r * KSTRIDE;
        const double m = __ldg(mass + (size_t)__ldg(ch + r) * s.stride);
        const double x = k[K_M2] - m * m;
        const double u = 1.0 / fma(x, x, k[K_Y2]);
        const double br = x * u, bi = k[K_Y] * u;  // B = conj(D)/|D|^2
        const double zr = k[K_CR] * br - k[K_CI] * bi, zi = k[K_CR] * bi + k[K_CI] * br;
        double dr = 0.0, di = 0.0;
        if (MODE == MODE_FULL) {
          const double wr = k[K_AR] + k[K_BR] * br - k[K_BI] * bi;
          const double wi = k[K_AI] + k[K_BR] * bi + k[K_BI] * br;
          dr = br * wr - bi * wi;  // zdot = B (alpha + beta B)
          di = br * wi + bi * wr;
        }
#pragma unroll
        for (int h = 0; h < H; ++h) {
          const double2 F = __ldg(amp + ((size_t)r * H + h) * s.stride);
          Ar[h] = fma(zr, F.x, Ar[h]);
          Ar[h] = fma(-zi, F.y, Ar[h]);
          Ai[h] = fma(zr, F.y, Ai[h]);
          Ai[h] = fma(zi, F.x, Ai[h]);
          if (MODE == MODE_FULL) {
            Dr[h] = fma(dr, F.x, Dr[h]);
            Dr[h] = fma(-di, F.y, Dr[h]);
            Di[h] = fma(dr, F.y, Di[h]);
            Di[h] = fma(di, F.x, Di[h]);
          }
        }
      }
      double I = 0.0, Idot = 0.0;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        I = fma(Ar[h], Ar[h], I);
        I = fma(Ai[h], Ai[h], I);
        Idot = fma(Ar[h], Dr[h], Idot);
        Idot = fma(Ai[h], Di[h], Idot);
      }
      Idot *= 2.0;

      // ---- per-event scalars: MC  s0 += I ; data  s0 += w ln I, s1 += w --------------------------
      double om, kap = 0.0;  // omega, kappa
      if (is_data) {
        const double w = valid ? (s.weight ? __ldg(s.weight + ic) : 1.0) : 0.0;
        const double inv = 1.0 / I;
        om = w * inv;
        kap = Idot * inv;
        s0 += valid ? w * log(I) : 0.0;
        s1 += w;
      } else {
        om = valid ? 1.0 : 0.0;
        s0 += valid ? I : 0.0;
      }
      if (MODE == MODE_NLL) continue;

      // ---- backward: conj(omega A_h), conj(omega (Adot_h - kappa A_h)) ---------------------------
#pragma unroll
      for (int h = 0; h < H; ++h) {
        if (MODE == MODE_FULL) {
          Dr[h] = om * (Dr[h] - kap * Ar[h]);
          Di[h] = -om * (Di[h] - kap * Ai[h]);
        }
        Ar[h] = om * Ar[h];
        Ai[h] = -om * Ai[h];
      }
      for (int b = 0; b < a.nb; ++b) {
        double val[32];
#pragma unroll
        for (int j = 0; j < RPB; ++j) {
          const int r = b * RPB + j;
          if (r < R) {
            const double* k = K + (size_t)r * KSTRIDE;
            const double m = __ldg(mass + (size_t)__ldg(ch + r) * s.stride);
            const double x = k[K_M2] - m * m;
            const double u = 1.0 / fma(x, x, k[K_Y2]);
            const double br = x * u, bi = k[K_Y] * u;
            double Sr = 0.0, Si = 0.0, Tr = 0.0, Ti = 0.0;
#pragma unroll
            for (int h = 0; h < H; ++h) {
              const double2 F = __ldg(amp + ((size_t)r * H + h) * s.stride);
              Sr = fma(Ar[h], F.x, Sr);
              Sr = fma(-Ai[h], F.y, Sr);
              Si = fma(Ar[h], F.y, Si);
              Si = fma(Ai[h], F.x, Si);
              if (MODE == MODE_FULL) {
                Tr = fma(Dr[h], F.x, Tr);
                Tr = fma(-Di[h], F.y, Tr);
                Ti = fma(Dr[h], F.y, Ti);
                Ti = fma(Di[h], F.x, Ti);
              }
            }
            // Horner: B S, B^2 S, B^3 S ; B S', B^2 S'
            const double t1r = br * Sr - bi * Si, t1i = br * Si + bi * Sr;
            const double t2r = br * t1r - bi * t1i, t2i = br * t1i + bi * t1r;
            val[j * VPR + 0] = t1r;
            val[j * VPR + 1] = t1i;
            val[j * VPR + 2] = t2r;
            val[j * VPR + 3] = t2i;
            if (MODE == MODE_FULL) {
              val[j * VPR + 4] = br * t2r - bi * t2i;
              val[j * VPR + 5] = br * t2i + bi * t2r;
              const double v1r = br * Tr - bi * Ti, v1i = br * Ti + bi * Tr;
              val[j * VPR + 6] = v1r;
              val[j * VPR + 7] = v1i;
              val[j * VPR + 8] = br * v1r - bi * v1i;
              val[j * VPR + 9] = br * v1i + bi * v1r;
            }
          } else {
#pragma unroll
            for (int q = 0; q < VPR; ++q) val[j * VPR + q] = 0.0;
          }
        }
#pragma unroll
        for (int q = RPB * VPR; q < 32; ++q) val[q] = 0.0;
        acc[b * 32 + lane] += bfly32(val, lane);
      }
    }

    // ---- block epilogue: fixed-order sum over the warps of this block ------------------------------
    s0 = warp_sum(s0);
    s1 = warp_sum(s1);
    if (lane == 0) {
      scal[warp * 2] = s0;
      scal[warp * 2 + 1] = s1;
    }
    __syncthreads();
    double* out = a.partial + ((size_t)sample * gridDim.x + blockIdx.x) * (nacc + 2);
    for (int k = threadIdx.x; k < nacc + 2; k += blockDim.x) {
      double t = 0.0;
      if (k < nacc) {
        for (int w = 0; w < nwarp; ++w) t += smem[(size_t)w * nacc + k];
      } else {
        for (int w = 0; w < nwarp; ++w) t += scal[w * 2 + (k - nacc)];
      }
      out[k] = t;
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// Stage 2 of the reduction + unpack: fixed-order sum of the per-block partials, then the theta- and
// v-dependent factors are applied ONCE per resonance to give the public raw vector of pwa_raw_sums
// (include/pwa.h; F_m, G_m, their first derivatives and HVPs).
// One block.  sums: scratch [2][nacc+2].
// ------------------------------------------------------------------------------------------------
struct Sums5 {
  cplx P1, P2, P3, Q1, Q2;
};

__device__ inline void unpack_res(const Sums5& s, double a, double phi, double M, double G, const double* v4,
                                  double* g4, double* h4) {
  double sn, cs;
  sincos(phi, &sn, &cs);
  const cplx e = {cs, sn}, c = {a * cs, a * sn};
  const cplx DM = {2.0 * M, -G};
  const cplx cDM = cmul(c, DM);
  // g_k = 2 Re( dz/dtheta_k-coefficient * P )
  g4[0] = 2.0 * cmul(e, s.P1).re;
  g4[1] = 2.0 * cmuli(cmul(c, s.P1)).re;
  g4[2] = -2.0 * cmul(cDM, s.P2).re;
  g4[3] = 2.0 * M * cmuli(cmul(c, s.P2)).re;
  if (!v4) return;
  const double va = v4[0], vp = v4[1], vM = v4[2], vG = v4[3];
  const cplx lam = {-2.0 * M * vM, G * vM + M * vG};
  const cplx al = cadd(cscale(e, va), cscale(cmuli(c), vp));
  const cplx be = cmul(c, lam);
  // h_a = 2Re( e Q1 + i e v_phi P1 + e lam P2 )
  cplx t = cadd(cmul(e, s.Q1), cadd(cscale(cmuli(cmul(e, s.P1)), vp), cmul(cmul(e, lam), s.P2)));
  h4[0] = 2.0 * t.re;
  // h_phi = 2Re( i c Q1 + i alpha P1 + i beta P2 )
  t = cmuli(cadd(cmul(c, s.Q1), cadd(cmul(al, s.P1), cmul(be, s.P2))));
  h4[1] = 2.0 * t.re;
  // h_M = 2Re( -c DM Q2 + k2 P2 + k3 P3 ),  k2 = -e DM v_a - i c DM v_phi - 2 c v_M + i c v_G,
  //                                          k3 = 2 c DM^2 v_M - 2 i M c DM v_G
  cplx k2 = cadd(cadd(cscale(cmul(e, DM), -va), cscale(cmuli(cDM), -vp)), cadd(cscale(c, -2.0 * vM), cscale(cmuli(c), vG)));
  cplx k3 = cadd(cscale(cmul(cDM, DM), 2.0 * vM), cscale(cmuli(cDM), -2.0 * M * vG));
  t = cadd(cscale(cmul(cDM, s.Q2), -1.0), cadd(cmul(k2, s.P2), cmul(k3, s.P3)));
  h4[2] = 2.0 * t.re;
  // h_G = 2Re( i M c Q2 + k2' P2 + k3' P3 ),  k2' = i M e v_a - M c v_phi + i c v_M,
  //                                            k3' = -2 i M c DM v_M - 2 M^2 c v_G
  k2 = cadd(cadd(cscale(cmuli(e), M * va), cscale(c, -M * vp)), cscale(cmuli(c), vM));
  k3 = cadd(cscale(cmuli(cDM), -2.0 * M * vM), cscale(c, -2.0 * M * M * vG));
  t = cadd(cscale(cmuli(cmul(c, s.Q2)), M), cadd(cmul(k2, s.P2), cmul(k3, s.P3)));
  h4[3] = 2.0 * t.re;
}

// ------------------------------------------------------------------------------------------------
// Combine: Eqs. 4, 6, 7 with NLL = -lnL and N_Data := W (S2, S3, S9).
// One block of 1024 threads; any of nll / grad / hv may be null.  Sets bit0 of *flags when a result is not finite.
// raw may have been written by this very block (fused path): plain loads, no read-only cache.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void combine_block(const double* raw, const double* __restrict__ v, int P, double* __restrict__ nll,
                                              double* __restrict__ grad, double* __restrict__ hv,
                                              unsigned* __restrict__ flags) {
  __shared__ double red[1024];
  __shared__ int bad;
  const double Ld = raw[0], W = raw[1], G = raw[2], n_mc = raw[3];
  const double* gd = raw + 4;
  const double* gG = raw + 4 + P;
  const double* hd = raw + 4 + 2 * P;
  const double* hG = raw + 4 + 3 * P;
  if (threadIdx.x == 0) bad = 0;
  double dot = 0.0;
  if (hv) {
    // fixed-order dot product gG . v : strided partials, then a tree in shared memory
    double t = 0.0;
    for (int k = threadIdx.x; k < P; k += blockDim.x) t = fma(gG[k], v[k], t);
    red[threadIdx.x] = t;
    __syncthreads();
    for (int s = blockDim.x / 2; s > 0; s >>= 1) {
      if ((int)threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
      __syncthreads();
    }
    dot = red[0];
  } else {
    __syncthreads();
  }
  int mybad = 0;
  const double invG = 1.0 / G;
  if (threadIdx.x == 0 && nll) {
    const double f = -Ld + W * log(G / n_mc);
    *nll = f;
    mybad |= !isfinite(f);
  }
  for (int k = threadIdx.x; k < P; k += blockDim.x) {
    if (grad) {
      const double g = -gd[k] + W * gG[k] * invG;
      grad[k] = g;
      mybad |= !isfinite(g);
    }
    if (hv) {
      const double h = hd[k] + W * (hG[k] * invG - gG[k] * dot * invG * invG);
      hv[k] = h;
      mybad |= !isfinite(h);
    }
  }
  if (mybad) atomicOr(&bad, 1);
  __syncthreads();
  if (threadIdx.x == 0) *flags = bad ? 1u : 0u;
}

static __global__ void __launch_bounds__(1024) k_combine(const double* raw, const double* __restrict__ v, int P,
                                                  double* __restrict__ nll, double* __restrict__ grad,
                                                  double* __restrict__ hv, unsigned* __restrict__ flags) {
  combine_block(raw, v, P, nll, grad, hv, flags);
}

// One truncated-CG iteration of the fit driver (pwa_fit.cu, step 3 of DESIGN.md S15'), run by the block that has just
// written q = H d (the tail of k_reduce_unpack<MODE_HVPQ>): one launch, one launch gap and one status copy less per CG
// iteration than a kernel of its own.  sc: the driver's scalar block (rr at [2], eps at [5], status at [6]); status
// 0 continue, 1 non-positive curvature, 2 residual small; on status != 0 the step p is written.  host_status: mapped
// pinned memory the host reads after its event (nullptr: none).  g == nullptr: no CG work in this launch.
struct CgTail {
  const double* g;
  const double* mask;
  double *z, *r, *d, *p, *sc;
  double* host_status;
  int P, j;
};

__device__ __forceinline__ double block_sum_1024(double x, double* red) {
  red[threadIdx.x] = x;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  const double r = red[0];
  __syncthreads();
  return r;
}

__device__ inline void cg_iter_block(const CgTail& c, const double* q) {
  __shared__ double red[1024];
  const int P = c.P, nt = blockDim.x;
  double dq = 0.0, dd = 0.0;
  for (int k = threadIdx.x; k < P; k += nt) {
    dq = fma(c.d[k], q[k] * c.mask[k], dq);
    dd = fma(c.d[k], c.d[k], dd);
  }
  dq = block_sum_1024(dq, red);
  dd = block_sum_1024(dd, red);
  const double rr = c.sc[2], eps = c.sc[5];
  double status = 0.0;
  if (!(dq > 1e-14 * dd)) {  // also catches NaN
    for (int k = threadIdx.x; k < P; k += nt) c.p[k] = (c.j == 0) ? -c.g[k] * c.mask[k] : c.z[k];
    status = 1.0;
  } else {
    const double alpha = rr / dq;
    double rn = 0.0;
    for (int k = threadIdx.x; k < P; k += nt) {
      c.z[k] = fma(alpha, c.d[k], c.z[k]);
      const double rk = fma(alpha, q[k] * c.mask[k], c.r[k]);
      c.r[k] = rk;
      rn = fma(rk, rk, rn);
    }
    rn = block_sum_1024(rn, red);
    if (sqrt(rn) <= eps) {
      for (int k = threadIdx.x; k < P; k += nt) c.p[k] = c.z[k];
      status = 2.0;
    } else {
      const double beta = rn / rr;
      for (int k = threadIdx.x; k < P; k += nt) c.d[k] = fma(beta, c.d[k], -c.r[k]);
      if (threadIdx.x == 0) c.sc[2] = rn;
    }
  }
  if (threadIdx.x == 0) {
    c.sc[6] = status;
    if (c.host_status) {
      *c.host_status = status;
      __threadfence_system();
    }
  }
}

// Second reduction stage (a-7): fixed-order sum of the per-block partial rows, compact sums -> raw sums
// (SURVEY appendix), and - when `combine` is set - Eqs. 4, 6, 7 in the same launch (the evaluation calls; the
// shard interface pwa_raw_sums stops at the raw vector).
// packed = 1: partial rows are [R][VPR] + 2 scalars (lanes sweep); packed = 0: [nb][32] + 2 (generic sweep)
template <int MODE>
__global__ void __launch_bounds__(1024) k_reduce_unpack(const double* __restrict__ partial, int nblocks, int nb, int R,
                                                        int packed, const double* __restrict__ theta,
                                                        const double* __restrict__ v, double n_mc, double* sums, double* raw,
                                                        int combine, double* __restrict__ nll, double* __restrict__ grad,
                                                        double* __restrict__ hv, unsigned* __restrict__ flags,
                                                        unsigned* ticket, double* pcache, const double* skip,
                                                        const CgTail cg) {
  if (skip != nullptr && *skip != 0.0) return;  // see LaneArgs::skip
  constexpr int VPR = vpr_of(MODE), RPB = rpb_of(MODE);
  const int nacc = packed ? (MODE == MODE_NLL ? 0 : R * VPR) : nb * 32, stride = nacc + 2, P = 4 * R;
  // Phase 1 over all blocks of this launch: one WARP per column (warp W of the launch takes columns W, W + #warps, ...):
  // lane l adds the rows l, l + 32, ... of the per-block partials in order, then a fixed butterfly over the lanes.  A
  // thread per column would walk the 148 rows one L2 latency after the other; this way a column costs about five
  // loads in flight and five shuffles.  The value of a column does not depend on the block that computes it.
  {
    const int lane = threadIdx.x & 31;
    const int warps = (gridDim.x * blockDim.x) >> 5, wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    for (int k = wid; k < 2 * stride; k += warps) {
      const int sample = k / stride, idx = k - sample * stride;
      const double* p = partial + (size_t)sample * nblocks * stride + idx;
      double t = 0.0;
      for (int b = lane; b < nblocks; b += 32) t += p[(size_t)b * stride];
#pragma unroll
      for (int m = 16; m > 0; m >>= 1) t += __shfl_xor_sync(0xffffffffu, t, m);
      if (lane == 0) sums[k] = t;
    }
  }
  // The block that finishes last (whichever it is: the sums do not depend on it) unpacks and combines.
  if (gridDim.x > 1) {
    __shared__ unsigned last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
      const unsigned done = atomicAdd(ticket, 1u);
      last = done == gridDim.x - 1 ? 1u : 0u;
      if (last) *ticket = 0u;  // ready for the next launch on this stream
    }
    __syncthreads();
    if (!last) return;
    __threadfence();  // what the other blocks wrote is read below with L2-only loads (__ldcg)
  } else {
    __syncthreads();
  }
  // MODE_GRAD3 leaves its block-summed compact sums (P1, P2, P3 and the scalars) in pcache: [2][6 R + 2];
  // MODE_HVPQ takes P1..P3 and the scalars from there and only Q1, Q2 from this sweep.
  const int cstride = 6 * R + 2;
  if (MODE == MODE_GRAD3)
    for (int k = threadIdx.x; k < 2 * stride; k += blockDim.x) pcache[k] = __ldcg(sums + k);
  const double* sc = MODE == MODE_HVPQ ? pcache : sums;   // where the scalars and the P sums live
  const int sstride = MODE == MODE_HVPQ ? cstride : stride, snacc = MODE == MODE_HVPQ ? 6 * R : nacc;
  if (threadIdx.x == 0) {
    raw[0] = __ldcg(sc + sstride + snacc);      // sum_data w ln I
    raw[1] = __ldcg(sc + sstride + snacc + 1);  // W
    raw[2] = __ldcg(sc + snacc);                // G
    raw[3] = n_mc;
  }
  if (MODE == MODE_NLL) {
    for (int k = threadIdx.x; k < 4 * P; k += blockDim.x) raw[4 + k] = 0.0;
  } else {
    // one thread per (resonance, sample): the two samples' unpacking (a sincos and ~150 dependent FP64 instructions each)
    // run side by side instead of one after the other
    for (int rs = threadIdx.x; rs < 2 * R; rs += blockDim.x) {
      const int r = rs >> 1, sample = rs & 1;
      const int b = r / RPB, j = r - b * RPB;
      const int qoff = packed ? r * VPR : b * 32 + j * VPR;
      const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
      {
        const double* q = sums + (size_t)sample * stride + qoff;
        Sums5 s;
        s.P3 = s.Q1 = s.Q2 = {0.0, 0.0};
        if (MODE == MODE_HVPQ) {
          const double* pc = pcache + (size_t)sample * cstride + r * 6;
          s.P1 = {__ldcg(pc), __ldcg(pc + 1)};
          s.P2 = {__ldcg(pc + 2), __ldcg(pc + 3)};
          s.P3 = {__ldcg(pc + 4), __ldcg(pc + 5)};
          s.Q1 = {__ldcg(q), __ldcg(q + 1)};
          s.Q2 = {__ldcg(q + 2), __ldcg(q + 3)};
        } else {
          s.P1 = {__ldcg(q), __ldcg(q + 1)};
          s.P2 = {__ldcg(q + 2), __ldcg(q + 3)};
          if (MODE == MODE_FULL || MODE == MODE_GRAD3) s.P3 = {__ldcg(q + 4), __ldcg(q + 5)};
          if (MODE == MODE_FULL) {
            s.Q1 = {__ldcg(q + 6), __ldcg(q + 7)};
            s.Q2 = {__ldcg(q + 8), __ldcg(q + 9)};
          }
          if (MODE == MODE_FULLP) {  // Q2 holds Q2 + 2 lambda P3: with P3 = 0 the unpacking below is unchanged
            s.Q1 = {__ldcg(q + 4), __ldcg(q + 5)};
            s.Q2 = {__ldcg(q + 6), __ldcg(q + 7)};
          }
        }
        double g4[4], h4[4] = {0.0, 0.0, 0.0, 0.0};
        unpack_res(s, a, phi, M, G, (mode_q(MODE) && v) ? v + 4 * r : nullptr, g4, h4);
        // raw layout: gd | gG | hd | hG ; data (sample 1) carries hd = -h
        double* gdst = raw + 4 + (sample == 1 ? 0 : P) + 4 * r;
        double* hdst = raw + 4 + 2 * P + (sample == 1 ? 0 : P) + 4 * r;
        for (int k = 0; k < 4; ++k) {
          gdst[k] = g4[k];
          hdst[k] = sample == 1 ? -h4[k] : h4[k];
        }
      }
    }
  }
  if (combine) {
    __syncthreads();  // the raw vector of this block's own writes is visible to the whole block
    combine_block(raw, mode_q(MODE) ? v : nullptr, P, nll, grad, mode_q(MODE) ? hv : nullptr, flags);
    if (MODE == MODE_HVPQ && cg.g != nullptr) {
      __syncthreads();  // hv = q = H d of this block's own writes
      cg_iter_block(cg, hv);
    }
  }
}

}  // namespace pwa
