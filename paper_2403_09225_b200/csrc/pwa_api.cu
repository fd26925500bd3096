// pwa_api.cu - the C ABI of include/pwa.h: handle, event store, evaluation entry points.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <new>

#include "pwa_internal.h"
#include "pwa_kernels.cuh"
#include "pwa_batch.cuh"
#include "pwa_rich.cuh"

namespace {
std::mutex g_err_mutex;
std::string g_create_err;

void set_create_error(const std::string& s) {
  std::lock_guard<std::mutex> lk(g_err_mutex);
  g_create_err = s;
}

inline long long round_up(long long x, long long m) { return (x + m - 1) / m * m; }
}  // namespace

namespace pwa {

pwa_status set_error(pwa_handle* h, pwa_status st, const char* what, cudaError_t ce) {
  std::string msg = what ? what : "";
  if (ce != cudaSuccess) {
    msg += ": ";
    msg += cudaGetErrorString(ce);
  }
  if (h) h->err = msg; else set_create_error(msg);
  return st;
}

// ---- sweep dispatch -------------------------------------------------------------------------------
typedef void (*sweep_fn)(const SweepArgs);

template <int MODE>
static sweep_fn generic_for_h(int H) {
  switch (H) {
    case 1: return k_sweep_generic<1, MODE>;
    case 2: return k_sweep_generic<2, MODE>;
    case 3: return k_sweep_generic<3, MODE>;
    case 4: return k_sweep_generic<4, MODE>;
    case 5: return k_sweep_generic<5, MODE>;
    case 6: return k_sweep_generic<6, MODE>;
    case 7: return k_sweep_generic<7, MODE>;
    case 8: return k_sweep_generic<8, MODE>;
  }
  return nullptr;
}

static sweep_fn generic_fn(int H, int mode) {
  switch (mode) {
    case MODE_NLL: return generic_for_h<MODE_NLL>(H);
    case MODE_GRAD: return generic_for_h<MODE_GRAD>(H);
    default: return generic_for_h<MODE_FULL>(H);
  }
}

// blocks of the second reduction stage (phase 1 is spread over them, the last one to finish does the rest)
static constexpr int kReduceBlocks = 16;

static inline int nb_of(int R, int mode) {
  if (mode == MODE_NLL) return 0;
  const int rpb = rpb_of(mode);
  return (R + rpb - 1) / rpb;
}

static size_t generic_smem(int block, int nb) { return (size_t)(block / 32) * ((size_t)nb * 32 + 2) * sizeof(double); }

// Runs prologue + sweep + stage-2 reduction/unpack; leaves the public raw vector in `raw` (device).
static pwa_status raw_sums_impl(pwa_handle* h, int mode, const double* theta, const double* v, double* raw,
                                bool combine = false, double* nll = nullptr, double* grad = nullptr, double* hv = nullptr,
                                const double* skip = nullptr, const CgTail* cg = nullptr) {
  const int R = h->n_res;
  if (mode == MODE_FULL && !v) mode = MODE_GRAD;
  const bool prof = h->profiling && h->prof_used + 2 <= h->prof_events.size();
  const int packed = h->variant >= 1;
  int nb = 0;
  if (packed) {
    // lanes sweep: the per-resonance constants are formed by every block itself (no prologue launch)
    if (mode == MODE_FULL && pair_available(h, MODE_FULLP)) mode = MODE_FULLP;  // two events per lane (pwa_sweep_pair.cuh)
    const bool pair = pair_available(h, mode);  // every mode of the 4 x 8-slice shape with H <= 2
    if (prof) cudaEventRecord(h->prof_events[h->prof_used], h->stream);
    pwa_status st = pair ? pair_launch(h, mode, theta, mode_q(mode) ? v : nullptr, skip)
                         : lanes_launch(h, mode, theta, mode_q(mode) ? v : nullptr, skip);
    if (st != PWA_OK) return st;
    h->launches++;
    if (prof) {
      cudaEventRecord(h->prof_events[h->prof_used + 1], h->stream);
      h->prof_used += 2;
    }
  } else {
    k_prologue<<<(R + 127) / 128, 128, 0, h->stream>>>(theta, mode == MODE_FULL ? v : nullptr, R, h->d_K);
    h->launches++;
    if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_prologue", ce);
    SweepArgs a;
    a.s[0] = h->smp[0];
    a.s[1] = h->smp[1];
    a.K = h->d_K;
    a.ch = h->d_ch;
    a.R = R;
    a.C = h->n_chan;
    a.nb = nb = nb_of(R, mode);
    a.partial = h->d_partial;
    sweep_fn fn = generic_fn(h->n_hel, mode);
    if (prof) cudaEventRecord(h->prof_events[h->prof_used], h->stream);
    fn<<<h->grid, h->block, generic_smem(h->block, a.nb), h->stream>>>(a);
    h->launches++;
    if (prof) {
      cudaEventRecord(h->prof_events[h->prof_used + 1], h->stream);
      h->prof_used += 2;
    }
    if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch sweep kernel", ce);
  }
  const double n_mc = (double)h->smp[0].n;
  CgTail cgt = {};
  if (cg && mode == MODE_HVPQ && combine) cgt = *cg;
#define PWA_REDUCE(M)                                                                                              \
  k_reduce_unpack<M><<<kReduceBlocks, 1024, 0, h->stream>>>(h->d_partial, h->grid, nb, R, packed, theta, v, n_mc,  \
                                                             h->d_sums, raw, combine ? 1 : 0, nll, grad, hv,        \
                                                             h->d_flags, h->d_flags + 1, h->d_pcache, skip, cgt)
  switch (mode) {
    case MODE_NLL: PWA_REDUCE(MODE_NLL); break;
    case MODE_GRAD: PWA_REDUCE(MODE_GRAD); break;
    case MODE_GRAD3: PWA_REDUCE(MODE_GRAD3); break;
    case MODE_HVPQ: PWA_REDUCE(MODE_HVPQ); break;
    case MODE_FULLP: PWA_REDUCE(MODE_FULLP); break;
    default: PWA_REDUCE(MODE_FULL); break;
  }
#undef PWA_REDUCE
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_reduce_unpack", ce);
  return PWA_OK;
}

static pwa_status combine_impl(pwa_handle* h, const double* raw, const double* v, double* nll, double* grad,
                               double* hv) {
  k_combine<<<1, 1024, 0, h->stream>>>(raw, v, h->n_par, nll, grad, hv, h->d_flags);
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_combine", ce);
  return PWA_OK;
}

// ---- richer model (readings S21, S22): user vectors <-> the expanded space [n_res][4] the sweeps work in ----------
// full[q] = user[map[q]] for theta (and v): exact, the expanded parameters are a linear (selection) map E of the user's
static __global__ void k_expand(int n_full, const int* __restrict__ map, const double* __restrict__ theta,
                                const double* __restrict__ v, double* __restrict__ theta_full, double* __restrict__ v_full) {
  for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < n_full; q += gridDim.x * blockDim.x) {
    const int p = map[q];
    if (theta) theta_full[q] = theta[p];
    if (v) v_full[q] = v[p];
  }
}

// raw_user = E^T raw_full block by block (every user parameter adds its expanded entries in ascending order), then -
// with `combine` - Eqs. 4, 6, 7 on the user-sized vectors.  One block of 1024 threads.
static __global__ void __launch_bounds__(1024) k_contract_combine(const double* __restrict__ raw_full, int n_full, int P,
                                                                  const int* __restrict__ off, const int* __restrict__ idx,
                                                                  double* raw, const double* __restrict__ v, int combine,
                                                                  double* __restrict__ nll, double* __restrict__ grad,
                                                                  double* __restrict__ hv, unsigned* __restrict__ flags) {
  if (threadIdx.x < 4) raw[threadIdx.x] = raw_full[threadIdx.x];
  for (int k = threadIdx.x; k < 4 * P; k += blockDim.x) {
    const int blk = k / P, p = k - blk * P;
    double t = 0.0;
    for (int j = off[p]; j < off[p + 1]; ++j) t += raw_full[4 + (size_t)blk * n_full + idx[j]];
    raw[4 + k] = t;
  }
  if (combine) {
    __syncthreads();
    combine_block(raw, v, P, nll, grad, hv, flags);
  }
}

template <int MODE>
static sweep_rich_fn rich_for_h(int H) {
  switch (H) {
    case 1: return k_sweep_rich<1, MODE>;
    case 2: return k_sweep_rich<2, MODE>;
    case 3: return k_sweep_rich<3, MODE>;
    case 4: return k_sweep_rich<4, MODE>;
  }
  return nullptr;
}

// general-lineshape sweep (pwa_rich.cuh): prologue + sweep + reduction -> raw_full
static pwa_status rich_raw(pwa_handle* h, int mode, const double* theta_full, const double* v_full, double* raw_full) {
  const int W = h->n_res;
  if (mode != MODE_NLL && mode != MODE_GRAD) mode = v_full ? MODE_FULL : MODE_GRAD;
  double* K = h->d_full + 2 * (size_t)h->n_full + 4 + 4 * (size_t)h->n_full;
  k_prologue_rich<<<(W + 127) / 128, 128, 0, h->stream>>>(theta_full, mode == MODE_FULL ? v_full : nullptr, W, h->d_wres,
                                                         h->d_lkind, h->d_lshape, K);
  h->launches++;
  RichArgs a;
  a.s[0] = h->smp[0];
  a.s[1] = h->smp[1];
  a.K = K;
  a.wres = h->d_wres;
  a.lch = h->d_lch;
  a.lkind = h->d_lkind;
  a.lshape = h->d_lshape;
  a.W = W;
  a.nb = (W + 3) / 4;
  a.partial = h->d_partial;
  sweep_rich_fn fn = mode == MODE_NLL ? rich_for_h<MODE_NLL>(h->n_hel) : mode == MODE_GRAD ? rich_for_h<MODE_GRAD>(h->n_hel) : rich_for_h<MODE_FULL>(h->n_hel);
  if (!fn) return set_error(h, PWA_ERR_INVALID_ARG, "general-lineshape kernel: n_hel > 4", cudaSuccess);
  const size_t smem = (size_t)(h->block / 32) * ((size_t)(mode == MODE_NLL ? 0 : a.nb * 32) + 2) * sizeof(double);
  const bool prof = h->profiling && h->prof_used + 2 <= h->prof_events.size();
  if (prof) cudaEventRecord(h->prof_events[h->prof_used], h->stream);
  fn<<<h->grid, h->block, smem, h->stream>>>(a);
  if (prof) {
    cudaEventRecord(h->prof_events[h->prof_used + 1], h->stream);
    h->prof_used += 2;
  }
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_sweep_rich", ce);
  const double n_mc = (double)h->smp[0].n;
  if (mode == MODE_NLL) k_reduce_rich<MODE_NLL><<<1, 1024, 0, h->stream>>>(h->d_partial, h->grid, a.nb, W, n_mc, h->d_sums, raw_full);
  else k_reduce_rich<MODE_FULL><<<1, 1024, 0, h->stream>>>(h->d_partial, h->grid, a.nb, W, n_mc, h->d_sums, raw_full);
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_reduce_rich", ce);
  return PWA_OK;
}

// One evaluation of a pwa_create_rich handle.  theta == nullptr: the expanded theta kept in d_theta_keep is used
// (split evaluation).  raw_user: where the contracted raw vector goes (h->d_raw or the caller's buffer).
static pwa_status eval_mapped(pwa_handle* h, int mode, const double* theta, const double* v, double* raw_user, bool combine,
                              double* nll, double* grad, double* hv, bool keep = false) {
  const int nf = h->n_full;
  double* th_full = (theta == nullptr || keep) ? h->d_theta_keep : h->d_full;
  double* v_full = h->d_full + nf;
  double* raw_full = h->d_full + 2 * (size_t)nf;
  if (theta || v) {
    k_expand<<<(nf + 255) / 256, 256, 0, h->stream>>>(nf, h->d_map, theta, v, th_full, v_full);
    h->launches++;
  }
  pwa_status st = h->rich_kernel ? rich_raw(h, mode, th_full, v ? v_full : nullptr, raw_full)
                                 : raw_sums_impl(h, mode, th_full, v ? v_full : nullptr, raw_full);
  if (st != PWA_OK) return st;
  k_contract_combine<<<1, 1024, 0, h->stream>>>(raw_full, nf, h->n_par, h->d_csr_off, h->d_csr_idx, raw_user, v, combine ? 1 : 0,
                                                nll, grad, v ? hv : nullptr, h->d_flags);
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_contract_combine", ce);
  return PWA_OK;
}

pwa_status expand_theta(pwa_handle* h, const double* theta) {
  k_expand<<<(h->n_full + 255) / 256, 256, 0, h->stream>>>(h->n_full, h->d_map, theta, nullptr, h->d_full, nullptr);
  h->launches++;
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch k_expand", ce);
  return PWA_OK;
}

pwa_status eval(pwa_handle* h, int mode, const double* theta, const double* v, double* nll, double* grad, double* hv) {
  if (h->mapped) return eval_mapped(h, mode, theta, mode == MODE_FULL ? v : nullptr, h->d_raw, true, nll, grad, hv);
  // sweep, then ONE launch for the second reduction stage, the unpacking and Eqs. 4, 6, 7
  return raw_sums_impl(h, mode, theta, v, h->d_raw, true, nll, grad, hv);
}

// Split evaluation for Newton-CG: the gradient call keeps theta and the direction-independent compact
// sums P1, P2, P3 in the handle; every following HVP at that theta only accumulates Q1, Q2 (MODE_HVPQ).
// Shapes served by the generic kernel have no such modes: they fall back to the fused sweep at the kept theta.
pwa_status eval_grad_keep(pwa_handle* h, const double* theta, double* nll, double* grad) {
  h->keep_valid = false;  // valid again only once everything that refreshes the kept state has been enqueued
  if (h->mapped) {  // the kept theta is the expanded one
    const int mode = (h->rich_kernel || h->variant < 2) ? MODE_GRAD : MODE_GRAD3;
    const pwa_status stm = eval_mapped(h, mode, theta, nullptr, h->d_raw, true, nll, grad, nullptr, true);
    h->keep_valid = stm == PWA_OK;
    return stm;
  }
  PWA_CUDA_CHECK(h, cudaMemcpyAsync(h->d_theta_keep, theta, sizeof(double) * h->n_par, cudaMemcpyDeviceToDevice, h->stream));
  const pwa_status st = h->variant < 2 ? eval(h, MODE_GRAD, theta, nullptr, nll, grad, nullptr)
                                       : raw_sums_impl(h, MODE_GRAD3, h->d_theta_keep, nullptr, h->d_raw, true, nll, grad, nullptr);
  h->keep_valid = st == PWA_OK;
  return st;
}

pwa_status eval_hvp_kept(pwa_handle* h, const double* v, double* hv, const double* skip, const CgTail* cg) {
  if (!h->keep_valid) return set_error(h, PWA_ERR_INVALID_ARG, "pwa_hvp_cached: no pwa_nll_grad_for_hvp call before", cudaSuccess);
  if (h->mapped) {
    const int mode = (h->rich_kernel || h->variant < 2) ? MODE_FULL : MODE_HVPQ;
    return eval_mapped(h, mode, nullptr, v, h->d_raw, true, nullptr, nullptr, hv);
  }
  if (h->variant < 2) return eval(h, MODE_FULL, h->d_theta_keep, v, nullptr, nullptr, hv);
  return raw_sums_impl(h, MODE_HVPQ, h->d_theta_keep, v, h->d_raw, true, nullptr, nullptr, hv, skip, cg);
}

}  // namespace pwa

using namespace pwa;

// ---- creation -------------------------------------------------------------------------------------
static pwa_status fail_create(pwa_handle* h, pwa_status st, const std::string& msg) {
  set_create_error(msg);
  if (h) pwa_destroy(h);
  return st;
}

static bool validate_sample(const pwa_sample& s, const char* name, std::string& why) {
  if (s.n_events < 1) { why = std::string(name) + ".n_events < 1"; return false; }
  if (s.stride != 0 && s.stride < s.n_events) { why = std::string(name) + ".stride < n_events"; return false; }
  if (!s.mass || !s.amp) { why = std::string(name) + ": null mass or amp"; return false; }
  return true;
}

// Uploads or adopts one sample.  own[0..2] receive owned allocations (mass, amp, weight).
static pwa_status store_sample(pwa_handle* h, const pwa_model_desc* m, const pwa_sample& s, int which, void** own) {
  const long long n = s.n_events, sin = s.stride ? s.stride : s.n_events;
  const int C = m->n_chan, planes = m->n_res * m->n_hel;
  SampleDev& d = h->smp[which];
  d.n = n;
  if (m->mem == PWA_MEM_DEVICE && m->borrow) {
    if (((uintptr_t)s.amp & 15) || ((uintptr_t)s.mass & 7) || (s.weight && ((uintptr_t)s.weight & 7)))
      return set_error(nullptr, PWA_ERR_INVALID_ARG, "borrowed buffers are misaligned (amp 16 B, mass/weight 8 B)", cudaSuccess);
    d.mass = s.mass;
    d.amp = reinterpret_cast<const double2*>(s.amp);
    d.weight = s.weight;
    d.stride = sin;
    return PWA_OK;
  }
  const long long so = round_up(n, 8);
  d.stride = so;
  const cudaMemcpyKind kind = m->mem == PWA_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  double *dm = nullptr, *da = nullptr, *dw = nullptr;
  if (cudaMalloc(&dm, sizeof(double) * C * so) != cudaSuccess ||
      cudaMalloc(&da, sizeof(double) * 2 * planes * so) != cudaSuccess ||
      (s.weight && cudaMalloc(&dw, sizeof(double) * so) != cudaSuccess)) {
    cudaGetLastError();
    if (dm) cudaFree(dm);
    if (da) cudaFree(da);
    if (dw) cudaFree(dw);
    return set_error(nullptr, PWA_ERR_OOM, "device allocation of the event store failed", cudaSuccess);
  }
  own[0] = dm; own[1] = da; own[2] = dw;
  // zero the padding so that clamped tail lanes read defined values
  PWA_CUDA_CHECK(nullptr, cudaMemsetAsync(dm, 0, sizeof(double) * C * so, h->stream));
  PWA_CUDA_CHECK(nullptr, cudaMemsetAsync(da, 0, sizeof(double) * 2 * planes * so, h->stream));
  for (int c = 0; c < C; ++c)
    PWA_CUDA_CHECK(nullptr, cudaMemcpyAsync(dm + (size_t)c * so, s.mass + (size_t)c * sin, sizeof(double) * n, kind, h->stream));
  for (int p = 0; p < planes; ++p)
    PWA_CUDA_CHECK(nullptr, cudaMemcpyAsync(da + (size_t)p * so * 2, s.amp + (size_t)p * sin * 2, sizeof(double) * 2 * n, kind, h->stream));
  if (s.weight) {
    PWA_CUDA_CHECK(nullptr, cudaMemsetAsync(dw, 0, sizeof(double) * so, h->stream));
    PWA_CUDA_CHECK(nullptr, cudaMemcpyAsync(dw, s.weight, sizeof(double) * n, kind, h->stream));
  }
  d.mass = dm;
  d.amp = reinterpret_cast<const double2*>(da);
  d.weight = dw;
  return PWA_OK;
}

// Planes -> tiled store (TiledDev, pwa_common.cuh).  The source holds `cnt` events starting at event i0 (a multiple of
// 32) of the sample, planes `stride` events apart; a warp moves one plane row of a 32-event group at a time (512
// contiguous bytes in, four 128-byte tile rows out).  Events from i0 + cnt to the end of their last tile are zeroed.
static __global__ void __launch_bounds__(256) k_retile(const double2* __restrict__ amp, const double* __restrict__ mass,
                                                       const double* __restrict__ weight, long long i0, long long cnt,
                                                       long long stride, int R, int C, TiledDev t, unsigned char* dst) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const long long groups = (cnt + 31) / 32, cap = (t.n + 7) / 8 * 8;
  for (long long g = blockIdx.x; g < groups; g += gridDim.x) {
    const long long k = g * 32 + lane, i = i0 + k;  // source-local and sample-wide event index
    if (i >= cap) continue;
    const bool valid = k < cnt;
    const int rows = R * t.H;
    for (int row = warp; row < rows + C + 1; row += nwarp) {
      if (row < rows) {
        const double2 f = valid ? amp[(size_t)row * stride + k] : make_double2(0.0, 0.0);
        *reinterpret_cast<double2*>(dst + tiled_amp_off(t, row / t.H, row % t.H, i)) = f;
      } else if (row < rows + C) {
        const int c = row - rows;
        *reinterpret_cast<double*>(dst + tiled_mass_off(t, c, i)) = valid ? mass[(size_t)c * stride + k] : 0.0;
      } else {
        *reinterpret_cast<double*>(dst + tiled_weight_off(t, i)) = (valid && weight) ? weight[k] : 0.0;
      }
    }
  }
}

// Builds the tiled store of one sample (h->tstore[which], layout already filled in) from the caller's planes.
static pwa_status store_sample_tiled(pwa_handle* h, const pwa_model_desc* m, const pwa_sample& s, int which, void** own) {
  const long long n = s.n_events, sin = s.stride ? s.stride : s.n_events;
  const int R = m->n_res, H = m->n_hel, C = m->n_chan, planes = R * H;
  TiledDev& t = h->tstore[which];
  t.n = n;
  t.weighted = s.weight != nullptr;
  h->smp[which].n = n;
  h->smp[which].stride = 0;
  h->smp[which].mass = nullptr;
  h->smp[which].amp = nullptr;
  h->smp[which].weight = nullptr;
  const size_t bytes = (size_t)((n + 7) / 8) * t.tile_bytes;
  unsigned char* dst = nullptr;
  if (cudaMalloc(&dst, bytes) != cudaSuccess) {
    cudaGetLastError();
    return set_error(nullptr, PWA_ERR_OOM, "device allocation of the (tiled) event store failed", cudaSuccess);
  }
  own[0] = dst;
  t.base = dst;
  const int grid = 8 * h->num_sms;
  if (m->mem == PWA_MEM_DEVICE) {
    k_retile<<<grid, 256, 0, h->stream>>>(reinterpret_cast<const double2*>(s.amp), s.mass, s.weight, 0, n, sin, R, C, t, dst);
    PWA_CUDA_CHECK(nullptr, cudaGetLastError());
    PWA_CUDA_CHECK(nullptr, cudaStreamSynchronize(h->stream));  // the caller may free its buffers when pwa_create returns
    return PWA_OK;
  }
  // host planes: staged through a device buffer of E events per plane (about 256 MB), chunk by chunk
  const size_t per_event = (size_t)planes * 16 + (size_t)C * 8 + 8;
  long long E = (long long)((256u << 20) / per_event) / 32 * 32;
  E = std::max<long long>(32, std::min<long long>(E, round_up(n, 32)));
  double *ta = nullptr, *tm = nullptr, *tw = nullptr;
  if (cudaMalloc(&ta, (size_t)planes * E * 16) != cudaSuccess || cudaMalloc(&tm, (size_t)C * E * 8) != cudaSuccess ||
      cudaMalloc(&tw, (size_t)E * 8) != cudaSuccess) {
    cudaGetLastError();
    if (ta) cudaFree(ta);
    if (tm) cudaFree(tm);
    return set_error(nullptr, PWA_ERR_OOM, "device allocation of the staging buffers failed", cudaSuccess);
  }
  cudaError_t ce = cudaSuccess;
  for (long long i0 = 0; i0 < n && ce == cudaSuccess; i0 += E) {
    const long long cnt = std::min(E, n - i0);
    ce = cudaMemcpy2DAsync(ta, (size_t)E * 16, s.amp + (size_t)i0 * 2, (size_t)sin * 16, (size_t)cnt * 16, planes, cudaMemcpyHostToDevice, h->stream);
    if (ce == cudaSuccess)
      ce = cudaMemcpy2DAsync(tm, (size_t)E * 8, s.mass + i0, (size_t)sin * 8, (size_t)cnt * 8, C, cudaMemcpyHostToDevice, h->stream);
    if (ce == cudaSuccess && s.weight) ce = cudaMemcpyAsync(tw, s.weight + i0, (size_t)cnt * 8, cudaMemcpyHostToDevice, h->stream);
    if (ce != cudaSuccess) break;
    k_retile<<<grid, 256, 0, h->stream>>>(reinterpret_cast<const double2*>(ta), tm, s.weight ? tw : nullptr, i0, cnt, E, R, C, t, dst);
    ce = cudaGetLastError();
  }
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(h->stream);
  cudaFree(ta);
  cudaFree(tm);
  cudaFree(tw);
  if (ce != cudaSuccess) return set_error(nullptr, PWA_ERR_CUDA, "upload of the (tiled) event store", ce);
  return PWA_OK;
}

extern "C" pwa_status pwa_create(const pwa_model_desc* m, pwa_handle** out) { return pwa_create_rich(m, nullptr, out); }

extern "C" pwa_status pwa_create_rich(const pwa_model_desc* m, const pwa_rich_desc* rich, pwa_handle** out) {
  if (out) *out = nullptr;
  if (!m || !out) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "null descriptor or output pointer");
  if (m->n_res < 1 || m->n_res > PWA_MAX_RES) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "n_res out of range");
  if (m->n_hel < 1 || m->n_hel > PWA_MAX_HEL) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "n_hel out of range");
  if (m->n_chan < 1 || m->n_chan > PWA_MAX_CHAN) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "n_chan out of range");
  std::vector<int> wave_chan(m->n_res);  // mass channel of every plane group (wave)
  bool rich_kernel = false;
  if (rich) {
    if (rich->n_lineshape < 1 || rich->n_lineshape > m->n_res) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "n_lineshape out of range");
    if (!rich->wave_res || !rich->ls_chan) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "null wave_res or ls_chan");
    for (int l = 0; l < rich->n_lineshape; ++l) {
      if (rich->ls_chan[l] < 0 || rich->ls_chan[l] >= m->n_chan) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "ls_chan value out of range");
      const int kind = rich->ls_kind ? rich->ls_kind[l] : PWA_LS_CONST;
      if (kind < PWA_LS_CONST || kind > PWA_LS_FLATTE) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "ls_kind value out of range");
      if (kind != PWA_LS_CONST) rich_kernel = true;
    }
    if (rich_kernel && !rich->ls_shape) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "null ls_shape with a non-constant-width resonance");
    if (rich_kernel && m->n_hel > 4) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "the general-lineshape kernel serves n_hel <= 4");
    for (int w = 0; w < m->n_res; ++w) {
      if (rich->wave_res[w] < 0 || rich->wave_res[w] >= rich->n_lineshape) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "wave_res value out of range");
      wave_chan[w] = rich->ls_chan[rich->wave_res[w]];
    }
  } else {
    if (!m->res_chan) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "null res_chan");
    for (int r = 0; r < m->n_res; ++r) {
      if (m->res_chan[r] < 0 || m->res_chan[r] >= m->n_chan)
        return fail_create(nullptr, PWA_ERR_INVALID_ARG, "res_chan value out of range");
      wave_chan[r] = m->res_chan[r];
    }
  }
  std::string why;
  if (!validate_sample(m->data, "data", why) || !validate_sample(m->mc, "mc", why))
    return fail_create(nullptr, PWA_ERR_INVALID_ARG, why);
  if (m->mc.weight) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "mc.weight must be NULL (unweighted phase space)");
  if (m->mem != PWA_MEM_HOST && m->mem != PWA_MEM_DEVICE) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "bad mem kind");
  if (m->borrow && m->mem != PWA_MEM_DEVICE) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "borrow needs PWA_MEM_DEVICE");

  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return fail_create(nullptr, PWA_ERR_CUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(ce));
  }
  if (m->device < 0 || m->device >= ndev) return fail_create(nullptr, PWA_ERR_INVALID_ARG, "device ordinal out of range");
  DeviceGuard guard(m->device);  // restores the caller's current device on every return path
  {
    int cur = -1;
    if ((ce = cudaGetDevice(&cur)) != cudaSuccess || cur != m->device)
      return fail_create(nullptr, PWA_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(ce));
  }

  pwa_handle* h = new (std::nothrow) pwa_handle();
  if (!h) return fail_create(nullptr, PWA_ERR_OOM, "host allocation failed");
  h->device = m->device;
  h->stream = static_cast<cudaStream_t>(m->stream);
  h->n_res = m->n_res;
  h->n_hel = m->n_hel;
  h->n_chan = m->n_chan;
  h->n_full = 4 * m->n_res;
  h->mapped = rich != nullptr;
  h->rich_kernel = rich_kernel;
  h->n_ls = rich ? rich->n_lineshape : m->n_res;
  h->n_par = rich ? 2 * m->n_res + 2 * rich->n_lineshape : h->n_full;
  h->weighted = m->data.weight != nullptr;
  cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, m->device);

  // Copy-mode handles of shapes that need 8-event tiles keep the events tiled (one bulk copy per stage instead of
  // tensor copies of 128-byte rows: pwa_sweep_lanes.cuh, PROD 4)
  const char* force = std::getenv("PWA_VARIANT");
  const bool want_lanes = (!force || std::strcmp(force, "lanes") == 0) && !rich_kernel;
  if (want_lanes && !rich && !m->borrow && m->data.n_events < (1LL << 30) && m->mc.n_events < (1LL << 30) &&
      !(m->mem == PWA_MEM_DEVICE && (((uintptr_t)m->data.amp | (uintptr_t)m->mc.amp) & 15))) {
    int phase_mul = 0;
    unsigned tile_bytes = 0, off_mass = 0, off_wgt = 0;
    if (lanes_wants_tiled(m->device, m->n_res, m->n_hel, m->n_chan, &phase_mul, &tile_bytes, &off_mass, &off_wgt)) {
      h->tiled = true;
      for (int k = 0; k < 2; ++k) {
        h->tstore[k].base = nullptr;
        h->tstore[k].tile_bytes = tile_bytes;
        h->tstore[k].off_mass = off_mass;
        h->tstore[k].off_wgt = off_wgt;
        h->tstore[k].H = m->n_hel;
        h->tstore[k].phase_mul = phase_mul;
      }
    }
  }
  pwa_status st = h->tiled ? store_sample_tiled(h, m, m->mc, 0, h->owned) : store_sample(h, m, m->mc, 0, h->owned);
  if (st == PWA_OK) st = h->tiled ? store_sample_tiled(h, m, m->data, 1, h->owned + 3) : store_sample(h, m, m->data, 1, h->owned + 3);
  if (st != PWA_OK) {
    std::string msg;
    { std::lock_guard<std::mutex> lk(g_err_mutex); msg = g_create_err; }
    return fail_create(h, st, msg);
  }

  // ---- launch configuration of the sweep (fixed for the life of the handle) ------------------------
  const int R = h->n_res, P = h->n_full;  // scratch is sized for the expanded space
  const int nb_full = std::max(nb_of(R, MODE_FULL), (R + 3) / 4);
  if (cudaMalloc(&h->d_ch, sizeof(int) * R) != cudaSuccess) {
    cudaGetLastError();
    return fail_create(h, PWA_ERR_OOM, "scratch allocation failed");
  }
  why.clear();
  h->weight_padded = h->owned[5] != nullptr;
  if (want_lanes) {
    st = lanes_configure(h, why);
    if (st != PWA_OK) return fail_create(h, st, h->err);
  }
  if (h->tiled && h->variant == 0) return fail_create(h, PWA_ERR_CUDA, "the tiled event store needs the lanes kernel (internal): " + why);
  if (h->variant == 0 && force) why = std::string("PWA_VARIANT=") + force + (why.empty() ? "" : "; " + why);
  if (h->variant == 0) {
    int block = 256;
    while (block > 32 && generic_smem(block, nb_full) > 160 * 1024) block /= 2;
    // the opt-in limit is a property of the function, shared by every handle: always raise it to one fixed cap
    const size_t smem = 200 * 1024;
    int occ_min = 1 << 30;
    for (int mode = 0; mode < 3; ++mode) {
      sweep_fn fn = generic_fn(h->n_hel, mode);
      if ((ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess)
        return fail_create(h, PWA_ERR_CUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(ce));
      int occ = 0;
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, block, generic_smem(block, nb_of(R, mode)));
      if (occ < 1) occ = 1;
      if (occ < occ_min) occ_min = occ;
    }
    h->block = block;
    h->grid = h->num_sms * occ_min;
    std::snprintf(h->variant_name, sizeof(h->variant_name), "generic(%s)", why.c_str());
    if (rich_kernel) {
      const size_t rsmem = (size_t)(block / 32) * ((size_t)((R + 3) / 4) * 32 + 2) * sizeof(double);
      int occ_r = 1 << 30;
      for (int mode = 0; mode < 3; ++mode) {
        sweep_rich_fn fn = mode == MODE_NLL ? rich_for_h<MODE_NLL>(h->n_hel) : mode == MODE_GRAD ? rich_for_h<MODE_GRAD>(h->n_hel) : rich_for_h<MODE_FULL>(h->n_hel);
        if ((ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess)
          return fail_create(h, PWA_ERR_CUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(ce));
        int occ = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, block, mode == MODE_NLL ? (size_t)(block / 32) * 16 : rsmem);
        occ_r = std::min(occ_r, std::max(occ, 1));
      }
      h->grid = h->num_sms * occ_r;
      std::snprintf(h->variant_name, sizeof(h->variant_name), "rich(general lineshape, one thread per event)");
    }
  }
  if (h->mapped && !rich_kernel) {
    const size_t len = std::strlen(h->variant_name);
    std::snprintf(h->variant_name + len, sizeof(h->variant_name) - len, "+shared");
  }

  const size_t pstride = std::max((size_t)nb_full * 32, (size_t)R * 10) + 2;
  h->partial_doubles = 2 * (size_t)h->grid * pstride;
  const size_t io = 1 + 4 * (size_t)P + 8;
  bool ok = cudaMalloc(&h->d_K, sizeof(double) * KSTRIDE * R) == cudaSuccess &&
            cudaMalloc(&h->d_partial, sizeof(double) * h->partial_doubles) == cudaSuccess &&
            cudaMalloc(&h->d_sums, sizeof(double) * 2 * pstride) == cudaSuccess &&
            cudaMalloc(&h->d_raw, sizeof(double) * (4 + 4 * (size_t)P)) == cudaSuccess &&
            cudaMalloc(&h->d_flags, 2 * sizeof(unsigned)) == cudaSuccess &&
            cudaMalloc(&h->d_pcache, sizeof(double) * 2 * (6 * (size_t)h->n_res + 2)) == cudaSuccess &&
            cudaMalloc(&h->d_theta_keep, sizeof(double) * h->n_full) == cudaSuccess &&
            cudaMalloc(&h->d_io, sizeof(double) * io) == cudaSuccess &&
            cudaMalloc(&h->d_fit, sizeof(double) * (8 * (size_t)P + 64)) == cudaSuccess &&
            cudaMallocHost(&h->h_pin, sizeof(double) * io) == cudaSuccess &&
            cudaMallocHost(&h->h_fit, sizeof(double) * 64) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    return fail_create(h, PWA_ERR_OOM, "scratch allocation failed");
  }
  if (h->mapped) {
    const int L = h->n_ls, nf = h->n_full, Pu = h->n_par;
    std::vector<int> map(nf), off(Pu + 1, 0), idx(nf), kind(L, PWA_LS_CONST);
    for (int w = 0; w < R; ++w) {
      map[4 * w] = 2 * w;
      map[4 * w + 1] = 2 * w + 1;
      map[4 * w + 2] = 2 * R + 2 * rich->wave_res[w];
      map[4 * w + 3] = 2 * R + 2 * rich->wave_res[w] + 1;
    }
    for (int q = 0; q < nf; ++q) off[map[q] + 1]++;
    for (int p2 = 0; p2 < Pu; ++p2) off[p2 + 1] += off[p2];
    {
      std::vector<int> fill(off.begin(), off.end() - 1);
      for (int q = 0; q < nf; ++q) idx[fill[map[q]]++] = q;  // ascending q within each user parameter
    }
    if (rich->ls_kind) kind.assign(rich->ls_kind, rich->ls_kind + L);
    std::vector<double> shape((size_t)L * RICH_SP, 0.0);
    if (rich->ls_shape) shape.assign(rich->ls_shape, rich->ls_shape + (size_t)L * RICH_SP);
    std::vector<int> wl_off(L + 1, 0), wl_idx(R);
    for (int w = 0; w < R; ++w) wl_off[rich->wave_res[w] + 1]++;
    for (int l = 0; l < L; ++l) wl_off[l + 1] += wl_off[l];
    {
      std::vector<int> fill(wl_off.begin(), wl_off.end() - 1);
      for (int w = 0; w < R; ++w) wl_idx[fill[rich->wave_res[w]]++] = w;
    }
    const size_t full_doubles = 2 * (size_t)nf + 4 + 4 * (size_t)nf + (size_t)R * RK;
    bool okr = cudaMalloc(&h->d_map, sizeof(int) * nf) == cudaSuccess && cudaMalloc(&h->d_csr_off, sizeof(int) * (Pu + 1)) == cudaSuccess &&
               cudaMalloc(&h->d_csr_idx, sizeof(int) * nf) == cudaSuccess && cudaMalloc(&h->d_wres, sizeof(int) * R) == cudaSuccess &&
               cudaMalloc(&h->d_lch, sizeof(int) * L) == cudaSuccess && cudaMalloc(&h->d_lkind, sizeof(int) * L) == cudaSuccess &&
               cudaMalloc(&h->d_lshape, sizeof(double) * L * RICH_SP) == cudaSuccess &&
               cudaMalloc(&h->d_wl_off, sizeof(int) * (L + 1)) == cudaSuccess && cudaMalloc(&h->d_wl_idx, sizeof(int) * R) == cudaSuccess &&
               cudaMalloc(&h->d_full, sizeof(double) * full_doubles) == cudaSuccess;
    if (!okr) {
      cudaGetLastError();
      return fail_create(h, PWA_ERR_OOM, "scratch allocation failed");
    }
    // pageable sources: cudaMemcpyAsync returns after staging them, the vectors may go out of scope
    if ((ce = cudaMemcpyAsync(h->d_map, map.data(), sizeof(int) * nf, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_csr_off, off.data(), sizeof(int) * (Pu + 1), cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_csr_idx, idx.data(), sizeof(int) * nf, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_wres, rich->wave_res, sizeof(int) * R, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_lch, rich->ls_chan, sizeof(int) * L, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_lkind, kind.data(), sizeof(int) * L, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_lshape, shape.data(), sizeof(double) * L * RICH_SP, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_wl_off, wl_off.data(), sizeof(int) * (L + 1), cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(h->d_wl_idx, wl_idx.data(), sizeof(int) * R, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
        (ce = cudaStreamSynchronize(h->stream)) != cudaSuccess)
      return fail_create(h, PWA_ERR_CUDA, std::string("upload: ") + cudaGetErrorString(ce));
  }
  if ((ce = cudaMemcpyAsync(h->d_ch, wave_chan.data(), sizeof(int) * R, cudaMemcpyHostToDevice, h->stream)) != cudaSuccess ||
      (ce = cudaMemsetAsync(h->d_flags, 0, 2 * sizeof(unsigned), h->stream)) != cudaSuccess ||
      (ce = cudaStreamSynchronize(h->stream)) != cudaSuccess)
    return fail_create(h, PWA_ERR_CUDA, std::string("upload: ") + cudaGetErrorString(ce));
  *out = h;
  return PWA_OK;
}

extern "C" pwa_status pwa_destroy(pwa_handle* h) {
  if (!h) return PWA_OK;
  DeviceGuard guard(h->device);
  cudaStreamSynchronize(h->stream);
  for (void* p : h->owned) if (p) cudaFree(p);
  void* dev[] = {h->d_ch, h->d_K, h->d_partial, h->d_sums, h->d_raw, h->d_flags, h->d_io, h->d_fit, h->d_pcache, h->d_theta_keep, h->d_batch,
                 h->d_map, h->d_csr_off, h->d_csr_idx, h->d_wres, h->d_lch, h->d_lkind, h->d_lshape, h->d_full,
                 h->d_wl_off, h->d_wl_idx};
  for (void* p : dev) if (p) cudaFree(p);
  for (cudaEvent_t e : h->prof_events) cudaEventDestroy(e);
  if (h->h_pin) cudaFreeHost(h->h_pin);
  if (h->h_fit) cudaFreeHost(h->h_fit);
  cudaGetLastError();
  delete h;
  return PWA_OK;
}

extern "C" int32_t pwa_n_params(const pwa_handle* h) { return h ? h->n_par : -1; }
extern "C" int32_t pwa_raw_size(const pwa_handle* h) { return h ? 4 + 4 * h->n_par : -1; }

// ---- evaluation -------------------------------------------------------------------------------------
#define PWA_REQUIRE(h, cond, msg) \
  do { if (!(cond)) return pwa::set_error((h), PWA_ERR_INVALID_ARG, msg, cudaSuccess); } while (0)

extern "C" pwa_status pwa_nll(pwa_handle* h, const double* theta, double* nll) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta && nll, "pwa_nll: null pointer");
  return eval(h, MODE_NLL, theta, nullptr, nll, nullptr, nullptr);
}

extern "C" pwa_status pwa_nll_grad(pwa_handle* h, const double* theta, double* nll, double* grad) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta && nll && grad, "pwa_nll_grad: null pointer");
  return eval(h, MODE_GRAD, theta, nullptr, nll, grad, nullptr);
}

extern "C" pwa_status pwa_hvp(pwa_handle* h, const double* theta, const double* v, double* hv) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta && v && hv, "pwa_hvp: null pointer");
  return eval(h, MODE_FULL, theta, v, nullptr, nullptr, hv);
}

extern "C" pwa_status pwa_nll_grad_hvp(pwa_handle* h, const double* theta, const double* v, double* nll, double* grad,
                                       double* hv) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta && v && nll && grad && hv, "pwa_nll_grad_hvp: null pointer");
  return eval(h, MODE_FULL, theta, v, nll, grad, hv);
}

extern "C" pwa_status pwa_raw_sums(pwa_handle* h, const double* theta, const double* v, double* raw) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta && raw, "pwa_raw_sums: null pointer");
  if (h->mapped) return eval_mapped(h, v ? MODE_FULL : MODE_GRAD, theta, v, raw, false, nullptr, nullptr, nullptr);
  return raw_sums_impl(h, v ? MODE_FULL : MODE_GRAD, theta, v, raw);
}

extern "C" pwa_status pwa_combine(pwa_handle* h, const double* raw, const double* v, double* nll, double* grad,
                                  double* hv) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, raw, "pwa_combine: null raw");
  PWA_REQUIRE(h, !hv || v, "pwa_combine: hv requires v");
  return combine_impl(h, raw, v, nll, grad, hv);
}

extern "C" pwa_status pwa_nll_grad_hvp_host(pwa_handle* h, const double* theta_host, const double* v_host,
                                            double* nll_host, double* grad_host, double* hv_host) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta_host, "pwa_nll_grad_hvp_host: null theta");
  PWA_REQUIRE(h, !hv_host || v_host, "pwa_nll_grad_hvp_host: hv requires v");
  const size_t P = h->n_par;
  double* d_theta = h->d_io;
  double* d_v = h->d_io + P;
  double* d_out = h->d_io + 2 * P;  // nll | grad | hv
  std::memcpy(h->h_pin, theta_host, sizeof(double) * P);
  if (v_host) std::memcpy(h->h_pin + P, v_host, sizeof(double) * P);
  PWA_CUDA_CHECK(h, cudaMemcpyAsync(d_theta, h->h_pin, sizeof(double) * (v_host ? 2 * P : P), cudaMemcpyHostToDevice, h->stream));
  pwa_status st = eval(h, v_host ? MODE_FULL : MODE_GRAD, d_theta, v_host ? d_v : nullptr, d_out, d_out + 1,
                       v_host ? d_out + 1 + P : nullptr);
  if (st != PWA_OK) return st;
  const size_t nout = 1 + P + (v_host ? P : 0);
  PWA_CUDA_CHECK(h, cudaMemcpyAsync(h->h_pin + 2 * P, d_out, sizeof(double) * nout, cudaMemcpyDeviceToHost, h->stream));
  PWA_CUDA_CHECK(h, cudaStreamSynchronize(h->stream));
  if (nll_host) *nll_host = h->h_pin[2 * P];
  if (grad_host) std::memcpy(grad_host, h->h_pin + 2 * P + 1, sizeof(double) * P);
  if (hv_host) std::memcpy(hv_host, h->h_pin + 2 * P + 1 + P, sizeof(double) * P);
  return PWA_OK;
}

// ---- diagnostics --------------------------------------------------------------------------------------
extern "C" pwa_status pwa_status_flags(pwa_handle* h, uint32_t* flags_host) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, flags_host, "pwa_status_flags: null pointer");
  unsigned f = 0;
  PWA_CUDA_CHECK(h, cudaMemcpyAsync(&f, h->d_flags, sizeof(unsigned), cudaMemcpyDeviceToHost, h->stream));
  PWA_CUDA_CHECK(h, cudaStreamSynchronize(h->stream));
  *flags_host = f;
  return PWA_OK;
}

extern "C" pwa_status pwa_profile_enable(pwa_handle* h, int32_t on) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  if (on && h->prof_events.empty()) {
    h->prof_events.resize(2 * 4096);
    for (size_t i = 0; i < h->prof_events.size(); ++i) {
      cudaError_t ce = cudaEventCreate(&h->prof_events[i]);
      if (ce != cudaSuccess) {
        for (size_t j = 0; j < i; ++j) cudaEventDestroy(h->prof_events[j]);
        h->prof_events.clear();
        return pwa::set_error(h, PWA_ERR_CUDA, "cudaEventCreate", ce);
      }
    }
  }
  h->profiling = on != 0;
  return PWA_OK;
}

extern "C" pwa_status pwa_profile_read(pwa_handle* h, double* total_ms, int64_t* n_launches) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_CUDA_CHECK(h, cudaStreamSynchronize(h->stream));
  double tot = 0.0;
  for (size_t i = 0; i + 1 < h->prof_used; i += 2) {
    float ms = 0.f;
    PWA_CUDA_CHECK(h, cudaEventElapsedTime(&ms, h->prof_events[i], h->prof_events[i + 1]));
    tot += ms;
  }
  if (total_ms) *total_ms = tot;
  if (n_launches) *n_launches = (int64_t)(h->prof_used / 2);
  h->prof_used = 0;
  return PWA_OK;
}

extern "C" pwa_status pwa_nll_grad_for_hvp(pwa_handle* h, const double* theta, double* nll, double* grad) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  if (!theta) return set_error(h, PWA_ERR_INVALID_ARG, "pwa_nll_grad_for_hvp: null theta", cudaSuccess);
  return eval_grad_keep(h, theta, nll, grad);
}

extern "C" pwa_status pwa_hvp_cached(pwa_handle* h, const double* v, double* hv) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  if (!v || !hv) return set_error(h, PWA_ERR_INVALID_ARG, "pwa_hvp_cached: null pointer", cudaSuccess);
  return eval_hvp_kept(h, v, hv);
}

// ---- K evaluations per pass over the event store -----------------------------------
// Greedy split of K into the batch counts the kernels are instantiated for; shapes without a batch kernel (and a
// remainder of one) go through the single-evaluation sweep: same results, one pass each.
extern "C" pwa_status pwa_nll_batch(pwa_handle* h, int32_t K, const double* theta, double* nll) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, K >= 1 && theta && nll, "pwa_nll_batch: K < 1 or null pointer");
  const int P = h->n_par;
  int k = 0;
  unsigned bad = 0;
  (void)bad;
  while (k < K) {
    const int left = K - k;
    int kb = 1;
    if (left >= 4 && batch_supported(h, BK_NLL, 4)) kb = 4;
    else if (left >= 2 && batch_supported(h, BK_NLL, 2)) kb = 2;
    pwa_status st = kb == 1 ? eval(h, MODE_NLL, theta + (size_t)k * P, nullptr, nll + k, nullptr, nullptr)
                            : batch_launch(h, BK_NLL, kb, theta + (size_t)k * P, nullptr, nll + k);
    if (st != PWA_OK) return st;
    k += kb;
  }
  return PWA_OK;
}

extern "C" pwa_status pwa_hvp_cached_batch(pwa_handle* h, int32_t K, const double* v, double* hv) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, K >= 1 && v && hv, "pwa_hvp_cached_batch: K < 1 or null pointer");
  if (!h->keep_valid) return set_error(h, PWA_ERR_INVALID_ARG, "pwa_hvp_cached_batch: no pwa_nll_grad_for_hvp call before", cudaSuccess);
  const int P = h->n_par;
  const int pref = std::getenv("PWA_HVP_BATCH") ? std::atoi(std::getenv("PWA_HVP_BATCH")) : 3;  // A/B runs
  int k = 0;
  while (k < K) {
    const int left = K - k;
    int kb = 1;
    if (pref >= 3 && left >= 3 && batch_supported(h, BK_HVPQ, 3)) kb = 3;
    else if (pref >= 2 && left >= 2 && batch_supported(h, BK_HVPQ, 2)) kb = 2;
    pwa_status st = kb == 1 ? eval_hvp_kept(h, v + (size_t)k * P, hv + (size_t)k * P)
                            : batch_launch(h, BK_HVPQ, kb, h->d_theta_keep, v + (size_t)k * P, hv + (size_t)k * P);
    if (st != PWA_OK) return st;
    k += kb;
  }
  return PWA_OK;
}

namespace {
__global__ void k_identity(int P, double* V) {
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < P * P; k += gridDim.x * blockDim.x) V[k] = (k / P == k % P) ? 1.0 : 0.0;
}
}  // namespace

extern "C" pwa_status pwa_hessian(pwa_handle* h, const double* theta, double* hess) {
  if (!h) return PWA_ERR_INVALID_ARG;
  DeviceGuard guard(h->device);
  PWA_REQUIRE(h, theta && hess, "pwa_hessian: null pointer");
  const int P = h->n_par;
  double* V = nullptr;
  if (cudaMallocAsync(&V, sizeof(double) * P * P, h->stream) != cudaSuccess) {
    cudaGetLastError();
    return set_error(h, PWA_ERR_OOM, "pwa_hessian: scratch allocation failed", cudaSuccess);
  }
  k_identity<<<(P * P + 255) / 256, 256, 0, h->stream>>>(P, V);
  h->launches++;
  pwa_status st = eval_grad_keep(h, theta, h->d_io, h->d_io + 1);  // nll, grad into the staging area (not returned)
  if (st == PWA_OK) st = pwa_hvp_cached_batch(h, P, V, hess);
  cudaFreeAsync(V, h->stream);
  return st;
}

extern "C" int64_t pwa_kernel_launches(const pwa_handle* h) { return h ? h->launches : -1; }

extern "C" int64_t pwa_bytes_per_eval(const pwa_handle* h) {
  if (!h) return -1;
  const long long per = 16LL * h->n_res * h->n_hel + 8LL * h->n_chan;
  return h->smp[0].n * per + h->smp[1].n * (per + (h->weighted ? 8 : 0));
}

extern "C" const char* pwa_kernel_variant(const pwa_handle* h) { return h ? h->variant_name : ""; }

extern "C" const char* pwa_last_error(const pwa_handle* h) {
  if (h) return h->err.c_str();
  static thread_local std::string copy;
  std::lock_guard<std::mutex> lk(g_err_mutex);
  copy = g_create_err;
  return copy.c_str();
}

extern "C" const char* pwa_version(void) { return "pwa-b200 0.1 (sm_100a)"; }
