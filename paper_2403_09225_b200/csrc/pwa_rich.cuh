// pwa_rich.cuh - the general-lineshape sweep (readings S21, S22): models in which a
// resonance has a mass-dependent width or a Flatte denominator.  Every lineshape kind is written as
//     D_l(i) = M^2 - m_i^2 - i Gamma chi_l(M) psi_l(m_i)
// with psi parameter-free (computed per event from the invariant mass) and chi a function of M alone (computed once per
// evaluation, with its first two derivatives, by k_prologue_rich):
//     kind 0 constant width        chi = M,               psi = 1
//     kind 1 mass-dependent width  chi = M^2 / q(M)^n,    psi = q(m)^n / m,   n = 2L + 1, q = two-body break-up momentum
//     kind 2 Flatte                chi = 1,               psi = rho_1(m) + Rg rho_2(m)  (complex below a threshold)
// dD/dM and dD/dGamma then depend on the event, so the compact sums of pwa_sweep_lanes.cuh (which pull every
// parameter-dependent factor out of the event loop) do not apply: this kernel accumulates the per-parameter sums
// themselves - per wave the eight reals (dI/da, dI/dphi, dI/dM, dI/dGamma) and the same four of H_i v, already weighted
// as Eqs. 6 and 7 need them - with the generic kernel's event -> thread map (lane = event, per-warp
// rows in shared memory, transposing butterfly over batches of four waves).  It runs at the generic kernel's speed
// (one read of F in the forward pass, one in the backward pass); models whose resonances are all constant-width
// never come here (shared resonances alone are served by the fast kernels through expansion, pwa_api.cu).
#pragma once
#include "pwa_kernels.cuh"

namespace pwa {

constexpr int RK = 16;  // doubles of constants per wave
enum { RK_X0 = 0, RK_Y = 1, RK_CR = 2, RK_CI = 3, RK_ER = 4, RK_EI = 5, RK_M = 6, RK_G = 7, RK_CHI = 8, RK_CHI1 = 9,
       RK_CHI2 = 10, RK_VA = 11, RK_VP = 12, RK_VM = 13, RK_VG = 14 };
constexpr int RICH_SP = 6;  // shape parameters per resonance (include/pwa.h)

struct RichArgs {
  SampleDev s[2];
  const double* K;      // [W][RK]
  const int* wres;      // [W] resonance of each wave
  const int* lch;       // [L] mass channel of each resonance
  const int* lkind;     // [L]
  const double* lshape; // [L][RICH_SP]
  int W;
  int nb;               // batches of 4 waves
  double* partial;      // [2][gridDim.x][nb*32 + 2]
};

typedef void (*sweep_rich_fn)(const RichArgs);

__device__ __forceinline__ double q2_two_body(double s, double m1, double m2) {
  return (s - (m1 + m2) * (m1 + m2)) * (s - (m1 - m2) * (m1 - m2)) / (4.0 * s);
}

// theta_full / v_full: the expanded vectors [W][4] = (a, phi, M, Gamma) per wave (pwa_api.cu: k_expand)
static __global__ void k_prologue_rich(const double* __restrict__ theta, const double* __restrict__ v, int W,
                                       const int* __restrict__ wres, const int* __restrict__ lkind,
                                       const double* __restrict__ lshape, double* __restrict__ K) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= W) return;
  const double a = theta[4 * m], phi = theta[4 * m + 1], M = theta[4 * m + 2], G = theta[4 * m + 3];
  const int l = wres[m], kind = lkind[l];
  const double* sp = lshape + (size_t)l * RICH_SP;
  double sn, cs;
  sincos(phi, &sn, &cs);
  double chi = M, chi1 = 1.0, chi2 = 0.0;
  if (kind == 1) {
    const double n = 2.0 * sp[2] + 1.0, u = M * M;
    const double sp_ = (sp[0] + sp[1]) * (sp[0] + sp[1]), sm_ = (sp[0] - sp[1]) * (sp[0] - sp[1]);
    const double p = q2_two_body(u, sp[0], sp[1]);
    const double p1 = 0.25 - sp_ * sm_ / (4.0 * u * u), p2 = sp_ * sm_ / (2.0 * u * u * u);
    const double pn = pow(p, -0.5 * n);
    const double f1 = pn - 0.5 * n * u * pn / p * p1;
    const double f2 = -n * pn / p * p1 + 0.5 * n * (0.5 * n + 1.0) * u * pn / (p * p) * p1 * p1 - 0.5 * n * u * pn / p * p2;
    chi = u * pn;
    chi1 = 2.0 * M * f1;
    chi2 = 2.0 * f1 + 4.0 * u * f2;
  } else if (kind == 2) {
    chi = 1.0;
    chi1 = 0.0;
  }
  double* k = K + (size_t)m * RK;
  k[RK_X0] = M * M;
  k[RK_Y] = G * chi;
  k[RK_CR] = a * cs;
  k[RK_CI] = a * sn;
  k[RK_ER] = cs;
  k[RK_EI] = sn;
  k[RK_M] = M;
  k[RK_G] = G;
  k[RK_CHI] = chi;
  k[RK_CHI1] = chi1;
  k[RK_CHI2] = chi2;
  k[RK_VA] = v ? v[4 * m] : 0.0;
  k[RK_VP] = v ? v[4 * m + 1] : 0.0;
  k[RK_VM] = v ? v[4 * m + 2] : 0.0;
  k[RK_VG] = v ? v[4 * m + 3] : 0.0;
  k[15] = 0.0;
}

// psi_l(m): parameter-free part of the width term (real for kinds 0, 1)
__device__ __forceinline__ cplx psi_of(int kind, const double* __restrict__ sp, double m) {
  if (kind == 0) return {1.0, 0.0};
  if (kind == 1) {
    const double q = sqrt(q2_two_body(m * m, sp[0], sp[1]));
    return {pow(q, 2.0 * sp[2] + 1.0) / m, 0.0};
  }
  const double s = m * m;
  const double qa = q2_two_body(s, sp[0], sp[1]), qb = q2_two_body(s, sp[2], sp[3]), Rg = sp[4];
  cplx r = {0.0, 0.0};
  const double ra = 2.0 * sqrt(fabs(qa)) / m, rb = Rg * 2.0 * sqrt(fabs(qb)) / m;
  if (qa >= 0.0) r.re += ra; else r.im += ra;
  if (qb >= 0.0) r.re += rb; else r.im += rb;
  return r;
}

// B = 1/D, D = X0 - m^2 - i Y psi
__device__ __forceinline__ cplx prop_of(const double* __restrict__ k, double m, cplx psi) {
  const cplx D = {k[RK_X0] - m * m + k[RK_Y] * psi.im, -k[RK_Y] * psi.re};
  const double u = 1.0 / (D.re * D.re + D.im * D.im);
  return {D.re * u, -D.im * u};
}

// MODE_NLL: scalars only; MODE_GRAD: + the four gradient sums per wave; MODE_FULL: + the four HVP sums per wave
template <int H, int MODE>
__global__ void __launch_bounds__(256) k_sweep_rich(const RichArgs a) {
  constexpr int VPR = 8, RPB = 4;
  extern __shared__ double smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const int nacc = MODE == MODE_NLL ? 0 : a.nb * 32;
  double* acc = smem + (size_t)warp * nacc;
  double* scal = smem + (size_t)nwarp * nacc;
  const int W = a.W;

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

      // ---- forward: A_h = sum_m z_m F_mh, Adot_h = sum_m zdot_m F_mh ----------------------------------------
      double Ar[H], Ai[H], Dr[H], Di[H];
#pragma unroll
      for (int h = 0; h < H; ++h) Ar[h] = Ai[h] = Dr[h] = Di[h] = 0.0;
      for (int w = 0; w < W; ++w) {
        const double* k = a.K + (size_t)w * RK;
        const int l = __ldg(a.wres + w), kind = __ldg(a.lkind + l);
        const double m = __ldg(mass + (size_t)__ldg(a.lch + l) * s.stride);
        const cplx psi = psi_of(kind, a.lshape + (size_t)l * RICH_SP, m);
        const cplx B = prop_of(k, m, psi);
        const cplx c = {k[RK_CR], k[RK_CI]}, e = {k[RK_ER], k[RK_EI]};
        const cplx z = cmul(c, B);
        cplx zd = {0.0, 0.0};
        if (MODE == MODE_FULL) {
          // dD/dM = 2M - i Gamma chi' psi ; dD/dGamma = -i chi psi
          const cplx ipsi = cmuli(psi);
          const cplx DM = {2.0 * k[RK_M] + k[RK_G] * k[RK_CHI1] * psi.im, -k[RK_G] * k[RK_CHI1] * psi.re};
          const cplx DG = cscale(ipsi, -k[RK_CHI]);
          const cplx zB = cmul(z, B);
          // zdot = v_a e B + v_phi i z - v_M z B D_M - v_Gamma z B D_Gamma
          zd = cadd(cadd(cscale(cmul(e, B), k[RK_VA]), cscale(cmuli(z), k[RK_VP])),
                    cscale(cadd(cscale(cmul(zB, DM), k[RK_VM]), cscale(cmul(zB, DG), k[RK_VG])), -1.0));
        }
#pragma unroll
        for (int h = 0; h < H; ++h) {
          const double2 F = __ldg(amp + ((size_t)w * H + h) * s.stride);
          Ar[h] = fma(z.re, F.x, fma(-z.im, F.y, Ar[h]));
          Ai[h] = fma(z.re, F.y, fma(z.im, F.x, Ai[h]));
          if (MODE == MODE_FULL) {
            Dr[h] = fma(zd.re, F.x, fma(-zd.im, F.y, Dr[h]));
            Di[h] = fma(zd.re, F.y, fma(zd.im, F.x, Di[h]));
          }
        }
      }
      double I = 0.0, Idot = 0.0;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        I = fma(Ar[h], Ar[h], fma(Ai[h], Ai[h], I));
        Idot = fma(Ar[h], Dr[h], fma(Ai[h], Di[h], Idot));
      }
      Idot *= 2.0;
      // weights of Eqs. 6, 7: data  g -> w g / I,  H v -> w (g Idot / I^2 - H v / I);  MC  g, H v
      double wg, wh_g, wh_h;
      if (is_data) {
        const double wt = valid ? (s.weight ? __ldg(s.weight + ic) : 1.0) : 0.0;
        const double inv = 1.0 / I;
        wg = wt * inv;
        wh_g = wt * Idot * inv * inv;
        wh_h = -wt * inv;
        s0 += valid ? wt * log(I) : 0.0;
        s1 += wt;
      } else {
        wg = valid ? 1.0 : 0.0;
        wh_g = 0.0;
        wh_h = wg;
        s0 += valid ? I : 0.0;
      }
      if (MODE == MODE_NLL) continue;

      // ---- backward: per wave S = sum_h conj(A_h) F, Sdot = sum_h conj(Adot_h) F and the eight sums -----------
      for (int b = 0; b < a.nb; ++b) {
        double val[32];
#pragma unroll
        for (int j = 0; j < RPB; ++j) {
          const int w = b * RPB + j;
          if (w < W) {
            const double* k = a.K + (size_t)w * RK;
            const int l = __ldg(a.wres + w), kind = __ldg(a.lkind + l);
            const double m = __ldg(mass + (size_t)__ldg(a.lch + l) * s.stride);
            const cplx psi = psi_of(kind, a.lshape + (size_t)l * RICH_SP, m);
            const cplx B = prop_of(k, m, psi);
            const cplx c = {k[RK_CR], k[RK_CI]}, e = {k[RK_ER], k[RK_EI]};
            const cplx z = cmul(c, B);
            cplx S = {0.0, 0.0}, T = {0.0, 0.0};
#pragma unroll
            for (int h = 0; h < H; ++h) {
              const double2 F = __ldg(amp + ((size_t)w * H + h) * s.stride);
              S.re = fma(Ar[h], F.x, fma(Ai[h], F.y, S.re));
              S.im = fma(Ar[h], F.y, fma(-Ai[h], F.x, S.im));
              if (MODE == MODE_FULL) {
                T.re = fma(Dr[h], F.x, fma(Di[h], F.y, T.re));
                T.im = fma(Dr[h], F.y, fma(-Di[h], F.x, T.im));
              }
            }
            const cplx ipsi = cmuli(psi);
            const cplx DM = {2.0 * k[RK_M] + k[RK_G] * k[RK_CHI1] * psi.im, -k[RK_G] * k[RK_CHI1] * psi.re};
            const cplx DG = cscale(ipsi, -k[RK_CHI]);
            const cplx eB = cmul(e, B), zB = cmul(z, B);
            cplx dz[4];
            dz[0] = eB;
            dz[1] = cmuli(z);
            dz[2] = cscale(cmul(zB, DM), -1.0);
            dz[3] = cscale(cmul(zB, DG), -1.0);
            double g4[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) g4[q] = 2.0 * cmul(dz[q], S).re;
#pragma unroll
            for (int q = 0; q < 4; ++q) val[j * VPR + q] = wg * g4[q];
            if (MODE == MODE_FULL) {
              const double va = k[RK_VA], vp = k[RK_VP], vM = k[RK_VM], vG = k[RK_VG];
              // second derivatives of z = a e^{i phi} / D   (D_GG = 0)
              const cplx DMM = {2.0 + k[RK_G] * k[RK_CHI2] * psi.im, -k[RK_G] * k[RK_CHI2] * psi.re};
              const cplx DMG = cscale(ipsi, -k[RK_CHI1]);
              const cplx eBB = cmul(eB, B), zBB = cmul(zB, B);
              const cplx z_ap = cmuli(eB), z_aM = cscale(cmul(eBB, DM), -1.0), z_aG = cscale(cmul(eBB, DG), -1.0);
              const cplx z_pp = cscale(z, -1.0), z_pM = cmuli(dz[2]), z_pG = cmuli(dz[3]);
              const cplx z_MM = cadd(cscale(cmul(zBB, cmul(DM, DM)), 2.0), cscale(cmul(zB, DMM), -1.0));
              const cplx z_MG = cadd(cscale(cmul(zBB, cmul(DM, DG)), 2.0), cscale(cmul(zB, DMG), -1.0));
              const cplx z_GG = cscale(cmul(zBB, cmul(DG, DG)), 2.0);
              cplx w4[4];
              w4[0] = cadd(cadd(cscale(z_ap, vp), cscale(z_aM, vM)), cscale(z_aG, vG));
              w4[1] = cadd(cadd(cscale(z_ap, va), cscale(z_pp, vp)), cadd(cscale(z_pM, vM), cscale(z_pG, vG)));
              w4[2] = cadd(cadd(cscale(z_aM, va), cscale(z_pM, vp)), cadd(cscale(z_MM, vM), cscale(z_MG, vG)));
              w4[3] = cadd(cadd(cscale(z_aG, va), cscale(z_pG, vp)), cadd(cscale(z_MG, vM), cscale(z_GG, vG)));
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const double hq = 2.0 * (cmul(dz[q], T).re + cmul(w4[q], S).re);
                val[j * VPR + 4 + q] = fma(wh_g, g4[q], wh_h * hq);
              }
            } else {
#pragma unroll
              for (int q = 0; q < 4; ++q) val[j * VPR + 4 + q] = 0.0;
            }
          } else {
#pragma unroll
            for (int q = 0; q < VPR; ++q) val[j * VPR + q] = 0.0;
          }
        }
        acc[b * 32 + lane] += bfly32(val, lane);
      }
    }

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

// Second stage for the rich sweep: fixed-order column sums over the per-block rows -> the raw vector in the EXPANDED
// parameter space [W][4] (layout of pwa_raw_sums with P = 4W).  One block of 1024 threads.
template <int MODE>
__global__ void __launch_bounds__(1024) k_reduce_rich(const double* __restrict__ partial, int nblocks, int nb, int W,
                                                      double n_mc, double* sums, double* raw) {
  const int nacc = MODE == MODE_NLL ? 0 : nb * 32, stride = nacc + 2, P = 4 * W;
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
  if (threadIdx.x == 0) {
    raw[0] = sums[stride + nacc];
    raw[1] = sums[stride + nacc + 1];
    raw[2] = sums[nacc];
    raw[3] = n_mc;
  }
  for (int q = threadIdx.x; q < P; q += blockDim.x) {
    const int w = q >> 2, c = q & 3, b = w >> 2, j = w & 3;
    double gd = 0.0, gG = 0.0, hd = 0.0, hG = 0.0;
    if (MODE != MODE_NLL) {
      gG = sums[b * 32 + j * 8 + c];
      hG = sums[b * 32 + j * 8 + 4 + c];
      gd = sums[stride + b * 32 + j * 8 + c];
      hd = sums[stride + b * 32 + j * 8 + 4 + c];
    }
    raw[4 + q] = gd;
    raw[4 + P + q] = gG;
    raw[4 + 2 * P + q] = hd;
    raw[4 + 3 * P + q] = hG;
  }
}

}  // namespace pwa
