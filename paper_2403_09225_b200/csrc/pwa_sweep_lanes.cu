// pwa_sweep_lanes.cu - host side of the warp-autonomous sweep: kernel table, shared-memory plan, launch.
#include <cstdlib>
#include <cstring>
#include <cstdio>

#include "pwa_internal.h"

namespace pwa {

namespace {
struct Combo {
  int rho, log_sw, nw;
};
// instantiated (RHO, LOG_SW, NW) triples, in order of preference; capacity RHO << LOG_SW resonances
constexpr Combo kCombos[] = {{4, 3, 7}, {4, 3, 11}, {2, 4, 15}, {2, 4, 11}};

template <int H, int RHO, int LOG_SW, int NW>
lanes_fn for_mode(int mode) {
  switch (mode) {
    case MODE_NLL: return lanes::k_sweep_lanes<H, RHO, LOG_SW, NW, MODE_NLL>;
    case MODE_GRAD: return lanes::k_sweep_lanes<H, RHO, LOG_SW, NW, MODE_GRAD>;
    default: return lanes::k_sweep_lanes<H, RHO, LOG_SW, NW, MODE_FULL>;
  }
}

template <int H>
lanes_fn for_combo(int rho, int log_sw, int nw, int mode) {
  if (rho == 4 && log_sw == 3 && nw == 7) return for_mode<H, 4, 3, 7>(mode);
  if (rho == 4 && log_sw == 3 && nw == 11) return for_mode<H, 4, 3, 11>(mode);
  if (rho == 2 && log_sw == 4 && nw == 15) return for_mode<H, 2, 4, 15>(mode);
  if (rho == 2 && log_sw == 4 && nw == 11) return for_mode<H, 2, 4, 11>(mode);
  return nullptr;
}

int env_int(const char* name, int dflt) {
  const char* e = std::getenv(name);
  return (e && *e) ? std::atoi(e) : dflt;
}
inline unsigned up(unsigned x, unsigned m) { return (x + m - 1) / m * m; }
}  // namespace

lanes_fn lanes_kernel(int H, int rho, int log_sw, int nw, int mode) {
  switch (H) {
    case 2: return for_combo<2>(rho, log_sw, nw, mode);
  }
  return nullptr;
}

pwa_status lanes_configure(pwa_handle* h, std::string& why) {
  const int R = h->n_res, H = h->n_hel, C = h->n_chan;
  for (int sidx = 0; sidx < 2; ++sidx) {
    const SampleDev& d = h->smp[sidx];
    if (d.n >= (1LL << 30)) { why = "sample too long for 32-bit TMA coordinates"; return PWA_OK; }
    if ((d.stride & 1) || ((uintptr_t)d.mass & 15) || ((uintptr_t)d.amp & 15) || (d.weight && ((uintptr_t)d.weight & 15))) {
      why = "event store not 16-byte aligned per plane (odd stride or misaligned base)";
      return PWA_OK;
    }
  }
  int rho = env_int("PWA_RHO", 0), log_sw = env_int("PWA_LOGSW", -1), nw = env_int("PWA_NW", 0);
  if (rho == 0 || log_sw < 0 || nw == 0) {  // smallest padded capacity; ties go to the earlier table entry
    int best = -1;
    for (const Combo& c : kCombos) {
      const int cap = c.rho << c.log_sw;
      if (cap < R || !lanes_kernel(H, c.rho, c.log_sw, c.nw, MODE_FULL)) continue;
      if (rho && c.rho != rho) continue;
      if (log_sw >= 0 && c.log_sw != log_sw) continue;
      if (nw && c.nw != nw) continue;
      if (best < 0 || cap < best) { best = cap; rho = c.rho; log_sw = c.log_sw; nw = c.nw; }
    }
    if (best < 0) { why = "no lanes-kernel instance for this (n_res, n_hel)"; return PWA_OK; }
  }
  if (!lanes_kernel(H, rho, log_sw, nw, MODE_FULL) || (rho << log_sw) < R) { why = "no lanes-kernel instance"; return PWA_OK; }
  const int SW = 1 << log_sw, RP = rho * SW, NW = nw;

  // amplitude rows incl. the zero-filled planes of padding resonances, in nbox boxes of rows_box (<= 256, x8) rows
  const int rows_need = up((unsigned)RP * H, 8);
  const int nbox = (rows_need + 255) / 256, rows_box = (int)up((unsigned)((rows_need + nbox - 1) / nbox), 8);
  const unsigned sub_bytes = (unsigned)nbox * rows_box * lanes::SUB * 16;  // multiple of 1024: swizzle atom alignment
  const unsigned off_mass = (lanes::TILE / lanes::SUB) * sub_bytes, off_wgt = off_mass + (unsigned)C * lanes::TILE * 8;
  const unsigned stage_bytes = up(off_wgt + lanes::TILE * 8, 1024);
  const unsigned k_bytes = up((unsigned)RP * lanes::KS * 8, 128);
  const unsigned red_bytes = up((unsigned)NW * (R * 10 + 2) * 8, 128);
  const unsigned fixed = k_bytes + red_bytes + 8u * 2 * 8 + 128;
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  int stages = (int)std::min<long long>(8, ((long long)dev_smem - fixed) / stage_bytes);
  const int st_env = env_int("PWA_STAGES", 0);
  if (st_env >= 2 && st_env <= stages) stages = st_env;
  if (stages < 2) { why = "tile does not fit in shared memory"; return PWA_OK; }
  const size_t smem = (size_t)stages * stage_bytes + fixed;

  for (int mode = 0; mode < 3; ++mode) {
    lanes_fn fn = lanes_kernel(H, rho, log_sw, nw, mode);
    cudaError_t ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(lanes sweep)", ce);
    int occ = 0;
    ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, (NW + 1) * 32, smem);
    if (ce != cudaSuccess || occ < 1) {
      cudaGetLastError();
      why = "lanes kernel cannot be resident (registers / shared memory)";
      return PWA_OK;
    }
  }
  LaneArgs& a = h->largs;
  std::memset(&a, 0, sizeof(a));
  a.weighted = h->smp[1].weight != nullptr;
  for (int sidx = 0; sidx < 2; ++sidx) {
    const SampleDev& d = h->smp[sidx];
    a.n[sidx] = d.n;
    bool ok = encode_2d(&a.tm_amp[sidx], d.amp, 2ull * d.n, (unsigned long long)R * H, (unsigned long long)d.stride * 16,
                        2 * lanes::SUB, rows_box, true) &&
              encode_2d(&a.tm_mass[sidx], d.mass, (unsigned long long)d.n, (unsigned long long)C,
                        (unsigned long long)d.stride * 8, lanes::TILE, C);
    if (ok && d.weight)
      ok = encode_2d(&a.tm_wgt[sidx], d.weight, (unsigned long long)d.n, 1, up((unsigned)((d.n * 8) & 0x7fffffff), 16) + 16,
                     lanes::TILE, 1);
    if (!ok) { why = "cuTensorMapEncodeTiled failed"; return PWA_OK; }
  }
  a.ch = h->d_ch;
  a.R = R; a.C = C; a.stages = stages;
  a.nbox = nbox; a.rows_box = rows_box;
  a.stage_bytes = stage_bytes; a.sub_bytes = sub_bytes; a.off_mass = off_mass; a.off_wgt = off_wgt;
  a.off_K = (unsigned)stages * stage_bytes;
  a.off_red = a.off_K + k_bytes;
  a.off_bar = a.off_red + red_bytes;
  h->lanes_smem = smem;
  h->lanes_rho = rho; h->lanes_log_sw = log_sw; h->lanes_nw = nw;
  h->variant = 2;
  h->block = (NW + 1) * 32;
  h->grid = h->num_sms;
  std::snprintf(h->variant_name, sizeof(h->variant_name), "lanes(rho=%d,sw=%d,nw=%d,stages=%d)", rho, SW, NW, stages);
  return PWA_OK;
}

pwa_status lanes_launch(pwa_handle* h, int mode, const double* theta, const double* v) {
  LaneArgs a = h->largs;
  a.theta = theta;
  a.v = v;
  a.partial = h->d_partial;
  lanes_fn fn = lanes_kernel(h->n_hel, h->lanes_rho, h->lanes_log_sw, h->lanes_nw, mode);
  fn<<<h->grid, h->block, h->lanes_smem, h->stream>>>(a);
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch lanes sweep kernel", ce);
  return PWA_OK;
}

}  // namespace pwa
