// pwa_sweep_lanes.cu - host side of the warp-autonomous sweep: kernel table, shared-memory plan, launch.
#include <cstdlib>
#include <cstring>
#include <cstdio>

#include "pwa_internal.h"

namespace pwa {

namespace {
typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

encode_fn get_encode() {
  static encode_fn fn = nullptr;
  if (fn) return fn;
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<encode_fn>(p);
  return fn;
}

int env_int(const char* name, int dflt) {
  const char* e = std::getenv(name);
  return (e && *e) ? std::atoi(e) : dflt;
}
inline unsigned up(unsigned x, unsigned m) { return (x + m - 1) / m * m; }
}  // namespace

bool encode_2d(CUtensorMap* m, const void* base, unsigned long long cols, unsigned long long rows,
               unsigned long long row_stride_bytes, unsigned box_cols, unsigned box_rows, bool swizzle128) {
  encode_fn fn = get_encode();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {row_stride_bytes};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t es[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), dims, strides, box, es,
            CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

lanes_fn lanes_kernel(int H, int combo, int mode) {
  if (combo < 0 || combo >= kNumLanesCombos) return nullptr;
  switch (H) {
    case 1: return lanes_kernel_h1(combo, mode);
    case 2: return lanes_kernel_h2(combo, mode);
    case 3: return lanes_kernel_h3(combo, mode);
    case 4: return lanes_kernel_h4(combo, mode);
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
  // smallest padded capacity among the instantiated combos (ties: the earlier entry); PWA_COMBO forces one
  int combo = env_int("PWA_COMBO", -1);
  if (combo < 0) {
    int best = -1;
    for (int k = 0; k < kNumLanesCombos; ++k) {
      const int cap = kLanesCombos[k].rho << kLanesCombos[k].log_sw;
      if (cap >= R && (best < 0 || cap < best)) { best = cap; combo = k; }
    }
  }
  if (H > 4 || !lanes_kernel(H, combo, MODE_FULL) || (kLanesCombos[combo].rho << kLanesCombos[combo].log_sw) < R) {
    why = "no lanes-kernel instance for this (n_res, n_hel)";
    return PWA_OK;
  }
  const int rho = kLanesCombos[combo].rho, log_sw = kLanesCombos[combo].log_sw, nw = kLanesCombos[combo].nw;
  const int prod = kLanesCombos[combo].prod, nthreads = lanes::lanes_threads(nw, prod);
  const int SW = 1 << log_sw, RP = rho * SW, NW = nw;

  // amplitude rows incl. the zero-filled planes of padding resonances, in nbox boxes of rows_box (<= 256) rows
  const int rows_need = RP * H;
  const int nbox = (rows_need + 255) / 256, rows_box = (rows_need + nbox - 1) / nbox;
  const unsigned amp_bytes = (unsigned)nbox * rows_box * lanes::TILE * 16;
  const unsigned off_mass = amp_bytes, off_wgt = off_mass + (unsigned)C * lanes::TILE * 8;
  const unsigned stage_bytes = up(off_wgt + lanes::TILE * 8, 128);
  const unsigned k_bytes = up((unsigned)RP * lanes::KS * 8, 128);
  const unsigned red_bytes = up((unsigned)NW * (R * 10 + 2) * 8, 128);
  const unsigned xch_bytes = up((unsigned)NW * (32 / SW) * 4 * H * 8, 128);
  const unsigned fixed = k_bytes + red_bytes + xch_bytes + 8u * 2 * 8 + 128;
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  int stages = (int)std::min<long long>(8, ((long long)dev_smem - fixed) / stage_bytes);
  const int st_env = env_int("PWA_STAGES", 0);
  if (st_env >= 2 && st_env <= stages) stages = st_env;
  if (stages < 2) { why = "tile does not fit in shared memory"; return PWA_OK; }
  const size_t smem = (size_t)stages * stage_bytes + fixed;

  for (int mode = 0; mode < 3; ++mode) {
    lanes_fn fn = lanes_kernel(H, combo, mode);
    cudaError_t ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(lanes sweep)", ce);
    int occ = 0;
    ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, nthreads, smem);
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
                        2 * lanes::TILE, rows_box, false) &&
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
  a.stage_bytes = stage_bytes; a.amp_bytes = amp_bytes; a.off_mass = off_mass; a.off_wgt = off_wgt;
  a.off_K = (unsigned)stages * stage_bytes;
  a.off_red = a.off_K + k_bytes;
  a.off_xch = a.off_red + red_bytes;
  a.off_bar = a.off_xch + xch_bytes;
  h->lanes_smem = smem;
  h->lanes_combo = combo;
  h->variant = 2;
  h->block = nthreads;
  h->grid = h->num_sms;
  std::snprintf(h->variant_name, sizeof(h->variant_name), "lanes(rho=%d,sw=%d,nw=%d%s,stages=%d)", rho, SW, NW, prod == 2 ? "g" : "", stages);
  return PWA_OK;
}

pwa_status lanes_launch(pwa_handle* h, int mode, const double* theta, const double* v) {
  LaneArgs a = h->largs;
  a.theta = theta;
  a.v = v;
  a.partial = h->d_partial;
  lanes_fn fn = lanes_kernel(h->n_hel, h->lanes_combo, mode);
  fn<<<h->grid, h->block, h->lanes_smem, h->stream>>>(a);
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch lanes sweep kernel", ce);
  return PWA_OK;
}

}  // namespace pwa
