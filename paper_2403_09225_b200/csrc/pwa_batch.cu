// pwa_batch.cu - host side of the batch sweeps (pwa_batch.cuh): kernel lookup, shared-memory plan, launch.
#include <algorithm>
#include <cstdlib>

#include "pwa_internal.h"
#include "pwa_batch.cuh"
#include "pwa_sweep_pair.cuh"

namespace pwa {

namespace {
inline unsigned up(unsigned x, unsigned m) { return (x + m - 1) / m * m; }
}  // namespace

// ---- the fused sweep with two events per lane (pwa_sweep_pair.cuh) -------------------------------------------------
static pair_fn pair_kernel(const pwa_handle* h, int mode) {
  if (h->variant < 2 || h->lanes_combo < 0) return nullptr;
  const LanesCombo& c = kLanesCombos[h->lanes_combo];
  if (!(c.rho == 4 && c.log_sw == 3 && c.nw == 8 && c.prod == 2 && c.tile == 32)) return nullptr;
  const char* env = std::getenv("PWA_PAIR");  // PWA_PAIR=0: the one-event kernel (A/B runs, tests of that path)
  if (env && std::atoi(env) == 0) return nullptr;
  switch (h->n_hel) {
    case 1: return pair_kernel_h1(mode);
    case 2: return pair_kernel_h2(mode);
  }
  return nullptr;
}

static bool pair_plan(const pwa_handle* h, PairArgs& p, size_t& smem) {
  const int NW = 8, EW = 4, RP = 32, H = h->n_hel;
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  const unsigned k_bytes = up((unsigned)RP * lanes::KSP * 8, 128);
  const unsigned red_bytes = up((unsigned)NW * (h->n_res * 8 + 2) * 8, 128);
  const unsigned xch_bytes = up((unsigned)NW * 2 * EW * (4 * H + 2) * 8, 128);
  const unsigned fixed = k_bytes + red_bytes + xch_bytes + 32u * 2 * 8 + 128;
  const long long fit = ((long long)dev_smem - fixed) / h->largs.stage_bytes;
  const int stages = ring_stages((int)std::min<long long>(fit, h->largs.stages), 2);  // two tiles are consumed at a time
  if (stages < 4) return false;
  p.stages = stages;
  p.off_K = (unsigned)stages * h->largs.stage_bytes;
  p.off_red = p.off_K + k_bytes;
  p.off_xch = p.off_red + red_bytes;
  p.off_bar = p.off_xch + xch_bytes;
  smem = (size_t)stages * h->largs.stage_bytes + fixed;
  return true;
}

bool pair_available(const pwa_handle* h, int mode) {
  if (!pair_kernel(h, mode)) return false;
  PairArgs p;
  size_t smem;
  return pair_plan(h, p, smem);
}

pwa_status pair_launch(pwa_handle* h, int mode, const double* theta, const double* v, const double* skip) {
  pair_fn fn = pair_kernel(h, mode);
  PairArgs p;
  size_t smem = 0;
  if (!fn || !pair_plan(h, p, smem)) return set_error(h, PWA_ERR_INVALID_ARG, "no two-event kernel for this shape", cudaSuccess);
  cudaError_t ce = cudaSuccess;
  if (!(h->attr_done & (1u << mode))) {  // once per handle and mode, not per launch
    // the attribute belongs to the FUNCTION, shared by every handle of the process: always raise it to the device limit
    int dev_smem = 0;
    cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(two-event sweep)", ce);
    h->attr_done |= 1u << mode;
  }
  LaneArgs a = h->largs;
  a.theta = theta;
  a.v = v;
  a.skip = skip;
  a.partial = h->d_partial;
  a.nprod = producers_for(p.stages);
  fn<<<h->grid, lanes::lanes_threads(8, 2), smem, h->stream>>>(a, p);
  if ((ce = cudaGetLastError()) != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "launch two-event sweep kernel", ce);
  return PWA_OK;
}

// ---- batch sweeps (pwa_batch.cuh) ---------------------------------------------------------------------------
static batch_fn batch_kernel(const pwa_handle* h, int kind, int kb) {
  if (h->variant < 2 || h->lanes_combo < 0 || h->mapped) return nullptr;  // rich handles take single passes
  const LanesCombo& c = kLanesCombos[h->lanes_combo];
  if (c.tile != 32) return nullptr;
  if (c.rho == 5 && kind == BK_HVPQ && kb == 3 && h->n_hel >= 3) return nullptr;  // spills (ptxas -v): batches of 2 there
  switch (h->n_hel) {
    case 1: return batch_kernel_h1(c.rho, c.log_sw, kind, kb);
    case 2: return batch_kernel_h2(c.rho, c.log_sw, kind, kb);
    case 3: return batch_kernel_h3(c.rho, c.log_sw, kind, kb);
    case 4: return batch_kernel_h4(c.rho, c.log_sw, kind, kb);
  }
  return nullptr;
}

// shared-memory plan of a batch launch: the handle's stage geometry, as many stages as fit beside the batch scratch
static bool batch_plan(const pwa_handle* h, int kind, int kb, BatchArgs& b, size_t& smem) {
  const LanesCombo& c = kLanesCombos[h->lanes_combo];
  const int SW = 1 << c.log_sw, RP = c.rho * SW, NW = 8, EW = 32 / SW;
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  const unsigned k_bytes = up((unsigned)RP * lanes::batch_ks(kind, kb) * 8, 128);
  const unsigned red_bytes = up((unsigned)NW * lanes::batch_row_len(kind, kb, h->n_res) * 8, 128);
  const unsigned xch_bytes = up(2u * NW * EW * (lanes::batch_nv(kind, kb, h->n_hel) + 2) * 8, 128);  // x 2: the paired value batch keeps two events per lane
  const unsigned fixed = k_bytes + red_bytes + xch_bytes + 32u * 2 * 8 + 128;
  const long long fit = ((long long)dev_smem - fixed) / h->largs.stage_bytes;
  // tiles consumed at the same time: the paired value batch of the 8-slice shape takes two, the others 8 / passes per tile
  const int group = (kind == BK_NLL && c.log_sw == 3) ? 2 : std::max(1, NW / (32 / EW));
  const int stages = ring_stages((int)std::min<long long>(fit, h->largs.stages), group);
  if (stages < 2) return false;
  b.stages = stages;
  b.off_K = (unsigned)stages * h->largs.stage_bytes;
  b.off_red = b.off_K + k_bytes;
  b.off_xch = b.off_red + red_bytes;
  b.off_bar = b.off_xch + xch_bytes;
  smem = (size_t)stages * h->largs.stage_bytes + fixed;
  return true;
}

bool batch_supported(const pwa_handle* h, int kind, int kb) {
  if (!batch_kernel(h, kind, kb)) return false;
  BatchArgs b;
  size_t smem;
  return batch_plan(h, kind, kb, b, smem);
}

template <int KIND, int KB>
static void launch_reduce_batch(pwa_handle* h, const double* theta, const double* v, double* sums, double* braw, double* out) {
  k_reduce_batch<KIND, KB><<<1, 1024, 0, h->stream>>>(h->d_batch, h->grid, h->n_res, theta, v, (double)h->smp[0].n, sums,
                                                      h->d_pcache, braw, out, h->d_flags);
}

pwa_status batch_launch(pwa_handle* h, int kind, int kb, const double* theta, const double* v, double* out) {
  batch_fn fn = batch_kernel(h, kind, kb);
  BatchArgs b;
  size_t smem = 0;
  if (!fn || !batch_plan(h, kind, kb, b, smem)) return set_error(h, PWA_ERR_INVALID_ARG, "no batch kernel for this shape", cudaSuccess);
  const int row_len = lanes::batch_row_len(kind, kb, h->n_res);
  const size_t need = 2 * (size_t)h->grid * row_len + 2 * (size_t)row_len + 4 + 4 * (size_t)h->n_par;
  if (need > h->batch_doubles) {
    if (h->d_batch) cudaFree(h->d_batch);
    h->d_batch = nullptr;
    h->batch_doubles = 0;
    if (cudaMalloc(&h->d_batch, sizeof(double) * need) != cudaSuccess) {
      cudaGetLastError();
      return set_error(h, PWA_ERR_OOM, "batch scratch allocation failed", cudaSuccess);
    }
    h->batch_doubles = need;
  }
  cudaError_t ce = cudaSuccess;
  const unsigned abit = 1u << (8 + 4 * kind + (kb - 1));
  if (!(h->attr_done & abit)) {
    int dev_smem = 0;  // function-wide attribute: the device limit, whatever this handle needs
    cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
    ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(batch sweep)", ce);
    h->attr_done |= abit;
  }
  b.theta = theta;
  b.v = v;
  b.partial = h->d_batch;
  const bool prof = h->profiling && h->prof_used + 2 <= h->prof_events.size();
  if (prof) cudaEventRecord(h->prof_events[h->prof_used], h->stream);
  LaneArgs la = h->largs;
  la.nprod = producers_for(b.stages);
  fn<<<h->grid, lanes::lanes_threads(8, 2), smem, h->stream>>>(la, b);
  if (prof) {
    cudaEventRecord(h->prof_events[h->prof_used + 1], h->stream);
    h->prof_used += 2;
  }
  h->launches++;
  if ((ce = cudaGetLastError()) != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "launch batch sweep kernel", ce);
  double* sums = h->d_batch + 2 * (size_t)h->grid * row_len;
  double* braw = sums + 2 * (size_t)row_len;
  if (kind == BK_NLL && kb == 2) launch_reduce_batch<BK_NLL, 2>(h, theta, v, sums, braw, out);
  else if (kind == BK_NLL && kb == 4) launch_reduce_batch<BK_NLL, 4>(h, theta, v, sums, braw, out);
  else if (kind == BK_HVPQ && kb == 2) launch_reduce_batch<BK_HVPQ, 2>(h, theta, v, sums, braw, out);
  else if (kind == BK_HVPQ && kb == 3) launch_reduce_batch<BK_HVPQ, 3>(h, theta, v, sums, braw, out);
  else return set_error(h, PWA_ERR_INVALID_ARG, "unsupported batch count", cudaSuccess);
  h->launches++;
  if ((ce = cudaGetLastError()) != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "launch k_reduce_batch", ce);
  return PWA_OK;
}

}  // namespace pwa
