// pwa_fit.cu - truncated line-search Newton-CG driver (DESIGN.md (c-F)).
// All vectors (theta, g, z, r, d, q, p) live on the device; the host reads one small block of scalars
// per CG iteration / line-search trial for control flow.
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>

#include <math_constants.h>

#include "pwa_internal.h"

namespace {

constexpr int FT = 256;  // threads of the single-block vector kernels

// scalar slots (device array `sc`, mirrored to pinned host memory)
enum { S_F = 0, S_FTRIAL = 1, S_RR = 2, S_GINF = 3, S_GNORM = 4, S_EPS = 5, S_STATUS = 6, S_GP = 7, S_PINF = 8,
       S_FEAS = 9, S_N = 16 };

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

// step 2 of (c-F): eps = min(0.5, sqrt|g|)|g| ; z = 0, r = g, d = -g
__global__ void __launch_bounds__(FT) k_cg_start(int P, const double* g, double* z, double* r, double* d, double* sc) {
  __shared__ double red[FT];
  double ss = 0.0, mx = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    const double gk = g[k];
    z[k] = 0.0;
    r[k] = gk;
    d[k] = -gk;
    ss = fma(gk, gk, ss);
    mx = fmax(mx, fabs(gk));
  }
  ss = block_sum(ss, red);
  mx = block_max(mx, red);
  if (threadIdx.x == 0) {
    const double gn = sqrt(ss);
    sc[S_RR] = ss;
    sc[S_GINF] = isfinite(ss) ? mx : CUDART_NAN;
    sc[S_GNORM] = gn;
    sc[S_EPS] = fmin(0.5, sqrt(gn)) * gn;
    sc[S_STATUS] = 0.0;  // CG running (the speculative launches of the driver test this slot)
  }
}

// step 3 of (c-F) after q = H d.  status: 0 continue, 1 non-positive curvature, 2 residual small.
// On status != 0 the step p is written.
__global__ void __launch_bounds__(FT) k_cg_iter(int P, int j, const double* g, const double* q, double* z, double* r,
                                                double* d, double* p, double* sc) {
  __shared__ double red[FT];
  if (sc[S_STATUS] != 0.0) return;  // CG already ended: this iteration was enqueued speculatively
  double dq = 0.0, dd = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    dq = fma(d[k], q[k], dq);
    dd = fma(d[k], d[k], dd);
  }
  dq = block_sum(dq, red);
  dd = block_sum(dd, red);
  const double rr = sc[S_RR], eps = sc[S_EPS];
  if (!(dq > 1e-14 * dd)) {  // also catches NaN
    for (int k = threadIdx.x; k < P; k += FT) p[k] = (j == 0) ? -g[k] : z[k];
    if (threadIdx.x == 0) sc[S_STATUS] = 1.0;
    return;
  }
  const double alpha = rr / dq;
  double rn = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    z[k] = fma(alpha, d[k], z[k]);
    const double rk = fma(alpha, q[k], r[k]);
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

// g.p and |p|_inf
__global__ void __launch_bounds__(FT) k_dirstats(int P, const double* g, const double* p, double* sc) {
  __shared__ double red[FT];
  double gp = 0.0, mx = 0.0;
  for (int k = threadIdx.x; k < P; k += FT) {
    gp = fma(g[k], p[k], gp);
    mx = fmax(mx, fabs(p[k]));
  }
  gp = block_sum(gp, red);
  mx = block_max(mx, red);
  if (threadIdx.x == 0) {
    sc[S_GP] = gp;
    sc[S_PINF] = mx;
  }
}

// trial = theta + t p ; feasibility of the fit box (S19)
__global__ void __launch_bounds__(FT) k_trial(int P, const double* theta, const double* p, double t, double* trial,
                                              double gmin, double gmax, double mmin, double mmax, double* sc) {
  __shared__ double red[FT];
  double bad = 0.0;
  const bool gbox = !(gmin == 0.0 && gmax == 0.0), mbox = !(mmin == 0.0 && mmax == 0.0);
  for (int k = threadIdx.x; k < P; k += FT) {
    const double x = fma(t, p[k], theta[k]);
    trial[k] = x;
    const int kind = k & 3;
    if (kind == 2 && mbox && !(x >= mmin && x <= mmax)) bad = 1.0;
    if (kind == 3 && gbox && !(x >= gmin && x <= gmax)) bad = 1.0;
    if (!isfinite(x)) bad = 1.0;
  }
  bad = block_max(bad, red);
  if (threadIdx.x == 0) sc[S_FEAS] = bad > 0.0 ? 0.0 : 1.0;
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
  double *g = h->d_fit, *z = g + P, *r = z + P, *d = r + P, *q = d + P, *p = q + P, *trial = p + P, *sc = trial + P;
  double* hs = h->h_fit;
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

  // step 1: f, g at theta
  FIT_EVAL(pwa::eval_grad_keep(h, theta, sc + S_F, g));
  res->n_grad++;
  int stop = 0;
  double f = 0.0, ginf = 0.0;
  for (int outer = 0;; ++outer) {
    k_cg_start<<<1, FT, 0, st>>>(P, g, z, r, d, sc);
    h->launches++;
    FIT_CHECK(fetch());
    f = hs[S_F];
    ginf = hs[S_GINF];
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

    // step 3: truncated CG on H p = -g.  Iteration j + 1 is enqueued BEFORE the host has seen the verdict of iteration
    // j (a copy of the status slot into pinned memory + an event per iteration): its kernels test the device-side
    // status and return at once if CG has ended, so the host round trip hides behind the next sweep.  Shapes on the
    // generic kernel have no such test and run one iteration at a time.
    bool have_p = false;
    const bool pipelined = h->variant >= 2;
    int done_at = -1;
    for (int j = 0; j < o.max_cg; ++j) {
      FIT_EVAL(pwa::eval_hvp_kept(h, d, q, pipelined ? sc + S_STATUS : nullptr));
      k_cg_iter<<<1, FT, 0, st>>>(P, j, g, q, z, r, d, p, sc);
      h->launches++;
      if (!pipelined) {
        FIT_CHECK(fetch());
        if (hs[S_STATUS] != 0.0) { done_at = j; break; }
        continue;
      }
      FIT_CHECK(cudaMemcpyAsync(hs + S_N + (j & 1), sc + S_STATUS, sizeof(double), cudaMemcpyDeviceToHost, st));
      FIT_CHECK(cudaEventRecord(ev[j & 1], st));
      if (j >= 1) {
        FIT_CHECK(cudaEventSynchronize(ev[(j - 1) & 1]));
        if (hs[S_N + ((j - 1) & 1)] != 0.0) { done_at = j - 1; break; }
      }
      if (j == o.max_cg - 1) {
        FIT_CHECK(cudaEventSynchronize(ev[j & 1]));
        if (hs[S_N + (j & 1)] != 0.0) done_at = j;
      }
    }
    have_p = done_at >= 0;
    const int iters = have_p ? done_at + 1 : o.max_cg;
    res->n_hvp += iters;
    res->cg_iters += iters;
    if (!have_p) {
      k_copy<<<1, FT, 0, st>>>(P, z, p);
      h->launches++;
    }
    k_dirstats<<<1, FT, 0, st>>>(P, g, p, sc);
    h->launches++;

    // step 4: Armijo backtracking
    double t = 1.0, fnew = 0.0;
    bool accepted = false;
    double gp = 0.0, pinf = 0.0;
    int n_infeasible = 0;
    for (int bt = 0; bt <= o.max_backtrack; ++bt) {
      k_trial<<<1, FT, 0, st>>>(P, theta, p, t, trial, o.gamma_min, o.gamma_max, o.mass_min, o.mass_max, sc);
      h->launches++;
      FIT_EVAL(pwa::eval(h, pwa::MODE_NLL, trial, nullptr, sc + S_FTRIAL, nullptr, nullptr));
      res->n_nll++;
      FIT_CHECK(fetch());
      gp = hs[S_GP];
      pinf = hs[S_PINF];
      fnew = hs[S_FTRIAL];
      if (hs[S_FEAS] != 0.0 && std::isfinite(fnew) && fnew <= f + o.armijo_c1 * t * gp) { accepted = true; break; }
      if (hs[S_FEAS] == 0.0) ++n_infeasible;
      t *= o.backtrack;
    }
    if (trace)
      std::fprintf(stderr, "pwa_fit: outer %d f %.10e |g|inf %.3e cg %d (end %d) g.p %.3e |p|inf %.3e t %.3e infeasible %d f_new %.10e %s\n",
                   outer, f, ginf, iters, have_p ? (int)hs[S_STATUS] : 0, gp, pinf, t, n_infeasible, fnew, accepted ? "ok" : "LINE SEARCH FAILED");
    if (!accepted) { stop = 6; break; }
    // step 5: accept
    FIT_CHECK(cudaMemcpyAsync(theta, trial, sizeof(double) * P, cudaMemcpyDeviceToDevice, st));
    FIT_EVAL(pwa::eval_grad_keep(h, theta, sc + S_F, g));
    res->n_grad++;
    const bool small_step = t * pinf <= o.xtol;
    const bool small_df = std::fabs(fnew - f) <= o.ftol * std::fmax(1.0, std::fabs(f));
    if (small_step || small_df) {
      stop = small_step ? 2 : 3;
      k_cg_start<<<1, FT, 0, st>>>(P, g, z, r, d, sc);  // refresh f, |g|_inf at the final point
      h->launches++;
      FIT_CHECK(fetch());
      f = hs[S_F];
      ginf = hs[S_GINF];
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
