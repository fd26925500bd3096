// pwa_fit.cu - projected, truncated line-search Newton-CG driver (readings S15', S19).
// All vectors (theta, g, z, r, d, q, p) live on the device; the host reads one small block of scalars
// per CG iteration / line-search trial for control flow.
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>

#include <math_constants.h>

#include "pwa_internal.h"
#include "pwa_kernels.cuh"

namespace {

constexpr int FT = 256;  // threads of the single-block vector kernels

// scalar slots (device array `sc`, mirrored to pinned host memory)
enum { S_F = 0, S_FTRIAL = 1, S_RR = 2, S_GINF = 3, S_GNORM = 4, S_EPS = 5, S_STATUS = 6, S_GP = 7, S_PINF = 8,
       S_NACT = 9, S_N = 16 };

// deterministic block reductions (fixed tree)
__device__ double block_sum(double x, double* red) {
  red[threadIdx.x] = x;
  __syncthreads();
  for (int s = FT / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  const double r = red[0];
  __syncthreads();
  return r;
}
__device__ double block_max(double x, double* red) {
  red[threadIdx.x] = x;
  __syncthreads();
  for (int s = FT / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + s]);
    __syncthreads();
  }
  const double r = red[0];
  __syncthreads();
  return r;
}

// the box of reading S19: only M (k % 4 == 2) and Gamma (k % 4 == 3) are bounded; (0, 0) = no box
struct Box {
  double gmin, gmax, mmin, mmax;
  int split;  // < 0: interleaved (a, phi, M, Gamma) per resonance (S6); >= 0: [a, phi per wave | M, Gamma per resonance] (S21)
};
__device__ __forceinline__ void box_of(const Box& b, int k, double& lo, double& hi) {
  lo = -CUDART_INF;
  hi = CUDART_INF;
  const int kind = b.split < 0 ? (k & 3) : (k < b.split ? (k & 1) : 2 + ((k - b.split) & 1));
  if (kind == 2 && !(b.mmin == 0.0 && b.mmax == 0.0)) { lo = b.mmin; hi = b.mmax; }
  if (kind == 3 && !(b.gmin == 0.0 && b.gmax == 0.0)) { lo = b.gmin; hi = b.gmax; }
}

// step 0 of S15': theta <- clip(theta, lo, hi)
__global__ void __launch_bounds__(FT) k_project(int P, double* theta, Box box) {
  for (int k = threadIdx.x; k < P; k += FT) {
    double lo, hi;
    box_of(box, k, lo, hi);
    theta[k] = fmin(fmax(theta[k], lo), hi);
  }
}

// steps 1-2 of S15': active set -> mask (1 free, 0 frozen), gP = g mask; eps = min(0.5, sqrt|gP|)|gP| ; z = 0, r = gP, d = -gP
__global__ void __launch_bounds__(FT) k_cg_start(int P, const double* theta, const double* g, Box box, double* mask,
                                                 double* z, double* r, double* d, double* sc) {
  __shared__ double red[FT];
  double ss = 0.0, mx = 0.0, full = 0.0, nact = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    const double gk = g[k], th = theta[k];
    double lo, hi;
    box_of(box, k, lo, hi);
    const bool active = (th <= lo && gk > 0.0) || (th >= hi && gk < 0.0);
    const double gp = active ? 0.0 : gk;
    mask[k] = active ? 0.0 : 1.0;
    z[k] = 0.0;
    r[k] = gp;
    d[k] = -gp;
    ss = fma(gp, gp, ss);
    mx = fmax(mx, fabs(gp));
    full = fma(gk, gk, full);
    nact += active ? 1.0 : 0.0;
  }
  ss = block_sum(ss, red);
  mx = block_max(mx, red);
  full = block_sum(full, red);
  nact = block_sum(nact, red);
  if (threadIdx.x == 0) {
    const double gn = sqrt(ss);
    sc[S_RR] = ss;
    sc[S_GINF] = isfinite(full) ? mx : CUDART_NAN;  // a non-finite entry anywhere in g is reported, frozen or not
    sc[S_GNORM] = gn;
    sc[S_EPS] = fmin(0.5, sqrt(gn)) * gn;
    sc[S_NACT] = nact;
    sc[S_STATUS] = 0.0;  // CG running (the speculative launches of the driver test this slot)
  }
}

// step 3 of S15' after q = H d (entries of the active set are dropped).  status: 0 continue, 1 non-positive
// curvature, 2 residual small.  On status != 0 the step p is written.
__global__ void __launch_bounds__(FT) k_cg_iter(int P, int j, const double* g, const double* mask, const double* q,
                                                double* z, double* r, double* d, double* p, double* sc) {
  __shared__ double red[FT];
  if (sc[S_STATUS] != 0.0) return;  // CG already ended: this iteration was enqueued speculatively
  double dq = 0.0, dd = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    dq = fma(d[k], q[k] * mask[k], dq);
    dd = fma(d[k], d[k], dd);
  }
  dq = block_sum(dq, red);
  dd = block_sum(dd, red);
  const double rr = sc[S_RR], eps = sc[S_EPS];
  if (!(dq > 1e-14 * dd)) {  // also catches NaN
    for (int k = threadIdx.x; k < P; k += FT) p[k] = (j == 0) ? -g[k] * mask[k] : z[k];
    if (threadIdx.x == 0) sc[S_STATUS] = 1.0;
    return;
  }
  const double alpha = rr / dq;
  double rn = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    z[k] = fma(alpha, d[k], z[k]);
    const double rk = fma(alpha, q[k] * mask[k], r[k]);
    r[k] = rk;
    rn = fma(rk, rk, rn);
  }
  rn = block_sum(rn, red);
  if (sqrt(rn) <= eps) {
    for (int k = threadIdx.x; k < P; k += FT) p[k] = z[k];
    if (threadIdx.x == 0) sc[S_STATUS] = 2.0;
    return;
  }
  const double beta = rn / rr;
  for (int k = threadIdx.x; k < P; k += FT) d[k] = fma(beta, d[k], -r[k]);
  if (threadIdx.x == 0) {
    sc[S_RR] = rn;
    sc[S_STATUS] = 0.0;
  }
}

__global__ void __launch_bounds__(FT) k_copy(int P, const double* src, double* dst) {
  for (int k = threadIdx.x; k < P; k += FT) dst[k] = src[k];
}

// p = -gP (the restart direction of step 4)
__global__ void __launch_bounds__(FT) k_steepest(int P, const double* g, const double* mask, double* p) {
  for (int k = threadIdx.x; k < P; k += FT) p[k] = -g[k] * mask[k];
}

// step 4 of S15': trial = clip(theta + t p), s = trial - theta; g.s and |s|_inf
__global__ void __launch_bounds__(FT) k_trial(int P, const double* theta, const double* g, const double* p, double t,
                                              double* trial, Box box, double* sc) {
  __shared__ double red[FT];
  double gs = 0.0, mx = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    double lo, hi;
    box_of(box, k, lo, hi);
    const double th = theta[k];
    const double x = fmin(fmax(fma(t, p[k], th), lo), hi);
    trial[k] = x;
    const double s = x - th;
    gs = fma(g[k], s, gs);
    mx = fmax(mx, fabs(s));
  }
  gs = block_sum(gs, red);
  mx = block_max(mx, red);
  if (threadIdx.x == 0) {
    sc[S_GP] = gs;
    sc[S_PINF] = mx;
  }
}

}  // namespace

extern "C" void pwa_fit_opts_default(pwa_fit_opts* o) {
  if (!o) return;
  o->max_outer = 500;
  o->max_cg = 50;
  o->gtol = 1e-5;
  o->xtol = 1e-8;
  o->ftol = 1e-12;
  o->armijo_c1 = 1e-4;
  o->backtrack = 0.5;
  o->max_backtrack = 40;
  o->max_seconds = 0.0;
  o->gamma_min = 5e-3;
  o->gamma_max = 2.0;
  o->mass_min = 0.1;
  o->mass_max = 4.0;
  o->gconv = 1.0;
}

extern "C" pwa_status pwa_fit_newton_cg(pwa_handle* h, double* theta, const pwa_fit_opts* opts_in, pwa_fit_result* res) {
  if (!h) return PWA_ERR_INVALID_ARG;
  if (!theta || !res) return pwa::set_error(h, PWA_ERR_INVALID_ARG, "pwa_fit_newton_cg: null pointer", cudaSuccess);
  pwa::DeviceGuard guard(h->device);
  pwa_fit_opts o;
  if (opts_in) o = *opts_in; else pwa_fit_opts_default(&o);
  if (o.max_outer < 0 || o.max_cg < 1 || o.max_backtrack < 0 || !(o.backtrack > 0.0 && o.backtrack < 1.0))
    return pwa::set_error(h, PWA_ERR_INVALID_ARG, "pwa_fit_newton_cg: bad options", cudaSuccess);
  const bool trace = std::getenv("PWA_FIT_TRACE") != nullptr;  // per-iteration diagnostics on stderr
  const auto t0 = std::chrono::steady_clock::now();
  auto elapsed = [&] { return std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count(); };
  *res = pwa_fit_result{};
  struct Events {
    cudaEvent_t e[2] = {nullptr, nullptr};
    ~Events() { for (cudaEvent_t x : e) if (x) cudaEventDestroy(x); }
    cudaEvent_t& operator[](int i) { return e[i]; }
  } ev;
  for (int i = 0; i < 2; ++i)
    if (cudaError_t ce = cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming)) return pwa::set_error(h, PWA_ERR_CUDA, "cudaEventCreate", ce);
  const int P = h->n_par;
  cudaStream_t st = h->stream;
  double *g = h->d_fit, *z = g + P, *r = z + P, *d = r + P, *q = d + P, *p = q + P, *trial = p + P, *mask = trial + P,
         *sc = mask + P;
  double* hs = h->h_fit;
  const Box box = {o.gamma_min, o.gamma_max, o.mass_min, o.mass_max, h->mapped ? 2 * h->n_res : -1};
  auto fetch = [&]() -> cudaError_t {
    cudaError_t ce = cudaMemcpyAsync(hs, sc, sizeof(double) * S_N, cudaMemcpyDeviceToHost, st);
    if (ce != cudaSuccess) return ce;
    return cudaStreamSynchronize(st);
  };
#define FIT_CHECK(call) PWA_CUDA_CHECK(h, (call))
#define FIT_EVAL(call)                   \
  do {                                   \
    pwa_status s__ = (call);             \
    if (s__ != PWA_OK) return s__;       \
  } while (0)

  // step 0: the start point projected into the box; step 1: f, g there
  k_project<<<1, FT, 0, st>>>(P, theta, box);
  h->launches++;
  FIT_EVAL(pwa::eval_grad_keep(h, theta, sc + S_F, g));
  res->n_grad++;
  int stop = 0;
  double f = 0.0, ginf = 0.0;
  for (int outer = 0;; ++outer) {
    k_cg_start<<<1, FT, 0, st>>>(P, theta, g, box, mask, z, r, d, sc);
    h->launches++;
    FIT_CHECK(fetch());
    f = hs[S_F];
    ginf = hs[S_GINF];
    res->n_active = (int32_t)hs[S_NACT];
    if (!std::isfinite(f) || !std::isfinite(ginf)) {
      res->nll = f;
      res->grad_inf_norm = ginf;
      res->status = PWA_ERR_NONFINITE;
      res->seconds = elapsed();
      return pwa::set_error(h, PWA_ERR_NONFINITE, "fit: NLL or gradient not finite", cudaSuccess);
    }
    if (ginf <= o.gtol) { stop = 1; break; }
    if (outer >= o.max_outer) { stop = 4; break; }
    if (o.max_seconds > 0.0 && elapsed() > o.max_seconds) { stop = 5; break; }
    res->outer_iters = outer + 1;

    // step 3: truncated CG on the free variables.  Iteration j + 1 is enqueued BEFORE the host has seen the verdict of
    // iteration j (a copy of the status slot into pinned memory + an event per iteration): its kernels test the
    // device-side status and return at once if CG has ended, so the host round trip hides behind the next sweep.
    // Shapes on the generic kernel have no such test and run one iteration at a time.
    bool have_p = false;
    const bool pipelined = h->variant >= 2 && !h->mapped;
    int done_at = -1;
    double cg_end = 0.0;
    for (int j = 0; j < o.max_cg; ++j) {
      if (pipelined) {
        // the CG update runs in the tail of the HVP's reduction launch and leaves its verdict in mapped pinned memory:
        // per iteration two launches (sweep, reduction + CG) and an event, no copy
        const pwa::CgTail cg = {g, mask, z, r, d, p, sc, hs + S_N + (j & 1), P, j};
        FIT_EVAL(pwa::eval_hvp_kept(h, d, q, sc + S_STATUS, &cg));
        FIT_CHECK(cudaEventRecord(ev[j & 1], st));
        if (j >= 1) {
          FIT_CHECK(cudaEventSynchronize(ev[(j - 1) & 1]));
          if (hs[S_N + ((j - 1) & 1)] != 0.0) { done_at = j - 1; cg_end = hs[S_N + ((j - 1) & 1)]; break; }
        }
        if (j == o.max_cg - 1) {
          FIT_CHECK(cudaEventSynchronize(ev[j & 1]));
          if (hs[S_N + (j & 1)] != 0.0) { done_at = j; cg_end = hs[S_N + (j & 1)]; }
        }
        continue;
      }
      FIT_EVAL(pwa::eval_hvp_kept(h, d, q, nullptr));
      k_cg_iter<<<1, FT, 0, st>>>(P, j, g, mask, q, z, r, d, p, sc);
      h->launches++;
      FIT_CHECK(fetch());
      if (hs[S_STATUS] != 0.0) { done_at = j; cg_end = hs[S_STATUS]; break; }
    }
    have_p = done_at >= 0;
    const int iters = have_p ? done_at + 1 : o.max_cg;
    res->n_hvp += iters;
    res->cg_iters += iters;
    if (!have_p) {
      k_copy<<<1, FT, 0, st>>>(P, z, p);
      h->launches++;
    }

    // step 4: projected Armijo backtracking; one restart along -gP if the search along p fails
    bool is_sd = have_p && done_at == 0 && cg_end == 1.0;  // p is already -gP
    double t = 1.0, fnew = 0.0, gs = 0.0, sinf = 0.0;
    bool accepted = false;
    for (;;) {
      t = 1.0;
      for (int bt = 0; bt <= o.max_backtrack; ++bt) {
        k_trial<<<1, FT, 0, st>>>(P, theta, g, p, t, trial, box, sc);
        h->launches++;
        FIT_EVAL(pwa::eval(h, pwa::MODE_NLL, trial, nullptr, sc + S_FTRIAL, nullptr, nullptr));
        res->n_nll++;
        FIT_CHECK(fetch());
        gs = hs[S_GP];
        sinf = hs[S_PINF];
        fnew = hs[S_FTRIAL];
        if (std::isfinite(fnew) && fnew <= f + o.armijo_c1 * gs) { accepted = true; break; }
        t *= o.backtrack;
      }
      if (accepted || is_sd) break;
      k_steepest<<<1, FT, 0, st>>>(P, g, mask, p);
      h->launches++;
      is_sd = true;
    }
    if (trace)
      std::fprintf(stderr, "pwa_fit: outer %d f %.10e |gP|inf %.3e active %d cg %d (end %d) g.s %.3e |s|inf %.3e t %.3e%s f_new %.10e %s\n",
                   outer, f, ginf, res->n_active, iters, (int)cg_end, gs, sinf, t, is_sd ? " (-gP)" : "", fnew,
                   accepted ? "ok" : "LINE SEARCH FAILED");
    if (!accepted) { stop = 6; break; }
    // step 5: accept
    FIT_CHECK(cudaMemcpyAsync(theta, trial, sizeof(double) * P, cudaMemcpyDeviceToDevice, st));
    FIT_EVAL(pwa::eval_grad_keep(h, theta, sc + S_F, g));
    res->n_grad++;
    const bool small_step = sinf <= o.xtol;
    const bool small_df = std::fabs(fnew - f) <= o.ftol * std::fmax(1.0, std::fabs(f));
    if (small_step || small_df) {
      stop = small_step ? 2 : 3;
      k_cg_start<<<1, FT, 0, st>>>(P, theta, g, box, mask, z, r, d, sc);  // refresh f, |gP|_inf at the final point
      h->launches++;
      FIT_CHECK(fetch());
      f = hs[S_F];
      ginf = hs[S_GINF];
      res->n_active = (int32_t)hs[S_NACT];
      break;
    }
  }
  res->nll = f;
  res->grad_inf_norm = ginf;
  res->stop_reason = stop;
  const bool stopped_on_test = stop == 1 || stop == 2 || stop == 3;
  res->status = (stopped_on_test && ginf <= o.gconv) ? PWA_OK : PWA_ERR_NOT_CONVERGED;
  res->seconds = elapsed();
  return (pwa_status)res->status;
}
