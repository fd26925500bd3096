// pwa_fractions.cu - fit fractions (S20; Table 1 of the paper):
//   F_r = sum_j sum_h |z_r(j) F_rh(j)|^2 / sum_j I_j   over the phase-space MC sample.
// One streaming pass over the MC event store (each F element read once: HBM-bound, called once per fit), one thread
// per event, the per-resonance terms summed over the 32 events of a warp by a fixed butterfly and kept per warp in
// shared memory; per-block partial rows, then a fixed-order sum over the blocks.  Deterministic, no atomics.
#include "pwa_internal.h"
#include "pwa_rich.cuh"

namespace pwa {
namespace {

constexpr int FB = 256;  // threads per block

// TILED: the handle keeps its events as 8-event tiles (TiledDev, pwa_common.cuh): same pass, other addresses
template <int H, bool TILED>
__global__ void __launch_bounds__(FB) k_fractions(SampleDev s, TiledDev td, const int* __restrict__ ch,
                                                  const double* __restrict__ theta, int R,
                                                  double* __restrict__ partial /* [grid][R + 1] */) {
  extern __shared__ double sm[];  // [R][4] constants (M^2, (M Gamma)^2, c_re, c_im; M Gamma kept in k[1] as a square root
                                  // would cost precision, so a fifth value) then [FB/32][R + 1] warp sums
  double* K = sm;                 // [R][5]
  double* acc = sm + 5 * R;       // [FB/32][R + 1]
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int r = threadIdx.x; r < R; r += FB) {
    const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
    double sn, cs;
    sincos(phi, &sn, &cs);
    K[5 * r] = M * M;
    K[5 * r + 1] = (M * G) * (M * G);
    K[5 * r + 2] = M * G;
    K[5 * r + 3] = a * cs;
    K[5 * r + 4] = a * sn;
  }
  for (int k = threadIdx.x; k < (FB / 32) * (R + 1); k += FB) acc[k] = 0.0;
  __syncthreads();
  double* mine = acc + w * (R + 1);
  const long long n = TILED ? td.n : s.n, stride = s.stride;
  const long long nwarp_iters = (n + 31) / 32;
  for (long long it = (long long)blockIdx.x * (FB / 32) + w; it < nwarp_iters; it += (long long)gridDim.x * (FB / 32)) {
    const long long i = it * 32 + lane;
    const bool valid = i < n;
    const long long ii = valid ? i : 0;
    double Ar[H], Ai[H];
#pragma unroll
    for (int h = 0; h < H; ++h) Ar[h] = Ai[h] = 0.0;
    for (int r = 0; r < R; ++r) {
      const double m = TILED ? *reinterpret_cast<const double*>(td.base + tiled_mass_off(td, ch[r], ii))
                             : s.mass[(long long)ch[r] * stride + ii];
      const double xx = K[5 * r] - m * m;
      const double inv = 1.0 / (xx * xx + K[5 * r + 1]);
      const double br = xx * inv, bi = K[5 * r + 2] * inv;  // B = conj(D) / |D|^2
      const double zr = K[5 * r + 3] * br - K[5 * r + 4] * bi, zi = K[5 * r + 3] * bi + K[5 * r + 4] * br;
      double own = 0.0;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        const double2 F = TILED ? *reinterpret_cast<const double2*>(td.base + tiled_amp_off(td, r, h, ii))
                                : s.amp[((long long)r * H + h) * stride + ii];
        const double tr = zr * F.x - zi * F.y, ti = zr * F.y + zi * F.x;
        Ar[h] += tr;
        Ai[h] += ti;
        own += tr * tr + ti * ti;
      }
      own = valid ? own : 0.0;
#pragma unroll
      for (int msk = 16; msk > 0; msk >>= 1) own += __shfl_xor_sync(0xffffffffu, own, msk);
      if (lane == 0) mine[r] += own;
    }
    double I = 0.0;
#pragma unroll
    for (int h = 0; h < H; ++h) I += Ar[h] * Ar[h] + Ai[h] * Ai[h];
    I = valid ? I : 0.0;
#pragma unroll
    for (int msk = 16; msk > 0; msk >>= 1) I += __shfl_xor_sync(0xffffffffu, I, msk);
    if (lane == 0) mine[R] += I;
  }
  __syncthreads();
  for (int k = threadIdx.x; k <= R; k += FB) {
    double t = 0.0;
    for (int ww = 0; ww < FB / 32; ++ww) t += acc[ww * (R + 1) + k];
    partial[(size_t)blockIdx.x * (R + 1) + k] = t;
  }
}

__global__ void __launch_bounds__(FB) k_fractions_final(const double* __restrict__ partial, int nblocks, int R,
                                                        double* __restrict__ frac) {
  __shared__ double G;
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int b = 0; b < nblocks; ++b) t += partial[(size_t)b * (R + 1) + R];
    G = t;
  }
  __syncthreads();
  for (int r = threadIdx.x; r < R; r += FB) {
    double t = 0.0;
    for (int b = 0; b < nblocks; ++b) t += partial[(size_t)b * (R + 1) + r];
    frac[r] = t / G;
  }
}

// Rich handles (pwa_create_rich): the fraction of RESONANCE l is the coherent sum of its partial waves,
//   F_l = sum_j sum_h | sum_{m in l} z_m(j) F_mh(j) |^2 / sum_j I_j        (Table 1 lists one fraction per resonance)
// Same event -> thread map as k_fractions; constants K [W][RK] from k_prologue_rich, every lineshape kind.
// wl_off / wl_idx: the waves of each resonance (ascending), partial [grid][L + 1].
template <int H>
__global__ void __launch_bounds__(FB) k_fractions_rich(SampleDev s, const double* __restrict__ K, const int* __restrict__ lch,
                                                       const int* __restrict__ lkind, const double* __restrict__ lshape,
                                                       const int* __restrict__ wl_off, const int* __restrict__ wl_idx, int L,
                                                       double* __restrict__ partial) {
  extern __shared__ double sm[];  // [FB/32][L + 1] warp sums
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int k = threadIdx.x; k < (FB / 32) * (L + 1); k += FB) sm[k] = 0.0;
  __syncthreads();
  double* mine = sm + w * (L + 1);
  const long long n = s.n, stride = s.stride;
  const long long nwarp_iters = (n + 31) / 32;
  for (long long it = (long long)blockIdx.x * (FB / 32) + w; it < nwarp_iters; it += (long long)gridDim.x * (FB / 32)) {
    const long long i = it * 32 + lane;
    const bool valid = i < n;
    const long long ii = valid ? i : 0;
    double Ar[H], Ai[H];
#pragma unroll
    for (int h = 0; h < H; ++h) Ar[h] = Ai[h] = 0.0;
    for (int l = 0; l < L; ++l) {
      const double m = s.mass[(long long)lch[l] * stride + ii];
      const cplx psi = psi_of(lkind[l], lshape + (size_t)l * RICH_SP, m);
      double Lr[H], Li[H];
#pragma unroll
      for (int h = 0; h < H; ++h) Lr[h] = Li[h] = 0.0;
      for (int q = wl_off[l]; q < wl_off[l + 1]; ++q) {
        const int wv = wl_idx[q];
        const double* k = K + (size_t)wv * RK;
        const cplx z = cmul({k[RK_CR], k[RK_CI]}, prop_of(k, m, psi));
#pragma unroll
        for (int h = 0; h < H; ++h) {
          const double2 F = s.amp[((long long)wv * H + h) * stride + ii];
          Lr[h] += z.re * F.x - z.im * F.y;
          Li[h] += z.re * F.y + z.im * F.x;
        }
      }
      double own = 0.0;
#pragma unroll
      for (int h = 0; h < H; ++h) {
        own += Lr[h] * Lr[h] + Li[h] * Li[h];
        Ar[h] += Lr[h];
        Ai[h] += Li[h];
      }
      own = valid ? own : 0.0;
#pragma unroll
      for (int msk = 16; msk > 0; msk >>= 1) own += __shfl_xor_sync(0xffffffffu, own, msk);
      if (lane == 0) mine[l] += own;
    }
    double I = 0.0;
#pragma unroll
    for (int h = 0; h < H; ++h) I += Ar[h] * Ar[h] + Ai[h] * Ai[h];
    I = valid ? I : 0.0;
#pragma unroll
    for (int msk = 16; msk > 0; msk >>= 1) I += __shfl_xor_sync(0xffffffffu, I, msk);
    if (lane == 0) mine[L] += I;
  }
  __syncthreads();
  for (int k = threadIdx.x; k <= L; k += FB) {
    double t = 0.0;
    for (int ww = 0; ww < FB / 32; ++ww) t += sm[ww * (L + 1) + k];
    partial[(size_t)blockIdx.x * (L + 1) + k] = t;
  }
}

typedef void (*frac_rich_fn)(SampleDev, const double*, const int*, const int*, const double*, const int*, const int*, int, double*);
frac_rich_fn frac_rich_kernel(int H) {
  switch (H) {
    case 1: return k_fractions_rich<1>;
    case 2: return k_fractions_rich<2>;
    case 3: return k_fractions_rich<3>;
    case 4: return k_fractions_rich<4>;
    case 5: return k_fractions_rich<5>;
    case 6: return k_fractions_rich<6>;
    case 7: return k_fractions_rich<7>;
    case 8: return k_fractions_rich<8>;
  }
  return nullptr;
}

typedef void (*frac_fn)(SampleDev, TiledDev, const int*, const double*, int, double*);
frac_fn frac_kernel(int H, bool tiled) {
  if (tiled) {  // tiled stores exist for the shapes of the lanes sweep only (n_hel <= 4)
    switch (H) {
      case 1: return k_fractions<1, true>;
      case 2: return k_fractions<2, true>;
      case 3: return k_fractions<3, true>;
      case 4: return k_fractions<4, true>;
    }
    return nullptr;
  }
  switch (H) {
    case 1: return k_fractions<1, false>;
    case 2: return k_fractions<2, false>;
    case 3: return k_fractions<3, false>;
    case 4: return k_fractions<4, false>;
    case 5: return k_fractions<5, false>;
    case 6: return k_fractions<6, false>;
    case 7: return k_fractions<7, false>;
    case 8: return k_fractions<8, false>;
  }
  return nullptr;
}

}  // namespace
}  // namespace pwa

using namespace pwa;

extern "C" pwa_status pwa_fit_fractions(pwa_handle* h, const double* theta, double* frac) {
  if (!h) return PWA_ERR_INVALID_ARG;
  pwa::DeviceGuard guard(h->device);
  if (!theta || !frac) return set_error(h, PWA_ERR_INVALID_ARG, "pwa_fit_fractions: null pointer", cudaSuccess);
  if (h->mapped) {  // one coherent fraction per resonance, any lineshape kind
    pwa_status st = pwa::expand_theta(h, theta);
    if (st != PWA_OK) return st;
    const int W = h->n_res, L = h->n_ls;
    double* K = h->d_full + 2 * (size_t)h->n_full + 4 + 4 * (size_t)h->n_full;
    k_prologue_rich<<<(W + 127) / 128, 128, 0, h->stream>>>(h->d_full, nullptr, W, h->d_wres, h->d_lkind, h->d_lshape, K);
    h->launches++;
    frac_rich_fn rfn = frac_rich_kernel(h->n_hel);
    const int grid = h->num_sms * 2;
    if ((size_t)grid * (L + 1) > h->partial_doubles)
      return set_error(h, PWA_ERR_INVALID_ARG, "pwa_fit_fractions: scratch too small", cudaSuccess);
    rfn<<<grid, FB, (size_t)(FB / 32) * (L + 1) * sizeof(double), h->stream>>>(h->smp[0], K, h->d_lch, h->d_lkind, h->d_lshape,
                                                                              h->d_wl_off, h->d_wl_idx, L, h->d_partial);
    h->launches++;
    if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_fractions_rich", ce);
    k_fractions_final<<<1, FB, 0, h->stream>>>(h->d_partial, grid, L, frac);
    h->launches++;
    if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_fractions_final", ce);
    return PWA_OK;
  }
  frac_fn fn = frac_kernel(h->n_hel, h->tiled);
  if (!fn) return set_error(h, PWA_ERR_INVALID_ARG, "pwa_fit_fractions: n_hel out of range", cudaSuccess);
  const int R = h->n_res;
  // the per-block rows reuse the sweep's partial buffer: [2][grid][10 R + 2] doubles there, [grid][R + 1] needed here
  const int grid = h->num_sms * 2;
  if ((size_t)grid * (R + 1) > h->partial_doubles)
    return set_error(h, PWA_ERR_INVALID_ARG, "pwa_fit_fractions: scratch too small", cudaSuccess);
  const size_t smem = (size_t)(5 * R + (FB / 32) * (R + 1)) * sizeof(double);
  if (smem > 48 * 1024) {
    cudaError_t ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(k_fractions)", ce);
  }
  fn<<<grid, FB, smem, h->stream>>>(h->smp[0], h->tstore[0], h->d_ch, theta, R, h->d_partial);
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_fractions", ce);
  k_fractions_final<<<1, FB, 0, h->stream>>>(h->d_partial, grid, R, frac);
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_fractions_final", ce);
  return PWA_OK;
}
