// pwa_sweep_lanes.cu - host side of the warp-autonomous sweep: kernel table, shared-memory plan, launch.
#include <algorithm>
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

bool encode_3d_swz128(CUtensorMap* m, const void* base, const unsigned long long dims[3], const unsigned long long strides_bytes[2],
                      const unsigned box[3]) {
  encode_fn fn = get_encode();
  if (!fn) return false;
  cuuint64_t d[3] = {dims[0], dims[1], dims[2]};
  cuuint64_t st[2] = {strides_bytes[0], strides_bytes[1]};
  cuuint32_t bx[3] = {box[0], box[1], box[2]};
  cuuint32_t es[3] = {1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(base), d, st, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
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
  // candidates: every instantiated shape with capacity >= R, smallest capacity first (ties: table order); the first
  // whose stage fits in shared memory at least twice is taken.  PWA_COMBO forces one entry (A/B runs).
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  const int forced = env_int("PWA_COMBO", -1);
  int combo = -1, stages = 0;
  int rho = 0, log_sw = 0, nw = 0, prod = 0, tile = 0, SW = 0, RP = 0, NW = 0, nthreads = 0, nbox = 0, rows_box = 0;
  unsigned amp_bytes = 0, off_mass = 0, off_wgt = 0, stage_bytes = 0, k_bytes = 0, red_bytes = 0, xch_bytes = 0, fixed = 0;
  why = H > 4 ? "no lanes-kernel instance for this n_hel" : "no lanes-kernel instance for this n_res";
  std::vector<int> order;
  for (int k = 0; k < kNumLanesCombos; ++k)
    if (forced < 0 || k == forced) order.push_back(k);
  std::stable_sort(order.begin(), order.end(), [](int x, int y) {
    return (kLanesCombos[x].rho << kLanesCombos[x].log_sw) < (kLanesCombos[y].rho << kLanesCombos[y].log_sw);
  });
  {
    for (size_t oi = 0; oi < order.size() && combo < 0 && H <= 4; ++oi) {
      const int k = order[oi];
      const LanesCombo& c = kLanesCombos[k];
      const int cap = c.rho << c.log_sw;
      if (cap < R || !lanes_kernel(H, k, MODE_FULL)) continue;
      rho = c.rho; log_sw = c.log_sw; nw = c.nw; prod = c.prod; tile = c.tile;
      nthreads = lanes::lanes_threads(nw, prod);
      SW = 1 << log_sw; RP = rho * SW;
      NW = c.alt >= 0 ? std::max(nw, kLanesCombos[c.alt].nw) : nw;  // per-warp scratch sized for the larger of the two shapes
      if (tile == 32) {
        // amplitude rows incl. the zero-filled planes of padding resonances, in nbox boxes of rows_box (<= 256) rows
        const int rows_need = RP * H;
        nbox = (rows_need + 255) / 256; rows_box = (rows_need + nbox - 1) / nbox;
        amp_bytes = (unsigned)nbox * rows_box * tile * 16;
        red_bytes = up((unsigned)nw * (R * 10 + 2) * 8, 128);  // rows for the main shape's warps only
      } else {
        if (RP > 256) continue;  // one 3-D box [H][RP][8 events]
        nbox = 1; rows_box = RP;
        amp_bytes = (unsigned)H * RP * tile * 16;
        red_bytes = up((unsigned)(R * 10 + 2) * 8, 128);  // one row: the warps add into it in turn
      }
      off_mass = amp_bytes; off_wgt = up(off_mass + (unsigned)C * tile * 8, 128);  // TMA destinations: 128-byte aligned
      stage_bytes = up(off_wgt + tile * 8, tile == 32 ? 128 : 1024);
      k_bytes = up((unsigned)RP * lanes::KS * 8, 128);
      xch_bytes = up((unsigned)NW * (32 / SW) * (4 * H + 2) * 8, 128);
      fixed = k_bytes + red_bytes + xch_bytes + 32u * 2 * 8 + 128;
      const int fit = (int)std::min<long long>(32, ((long long)dev_smem - fixed) / stage_bytes);
      stages = std::min(8, fit);  // deeper rings were measured no faster (the kernel is not feed-bound); PWA_STAGES overrides
      const int st_env = env_int("PWA_STAGES", 0);
      if (st_env >= 2 && st_env <= fit) stages = st_env;
      if (stages < 2) { why = "tile does not fit in shared memory"; continue; }
      combo = k;
    }
  }
  if (combo < 0) return PWA_OK;
  why.clear();
  const size_t smem = (size_t)stages * stage_bytes + fixed;

  const int alt = kLanesCombos[combo].alt;
  for (int mode = 0; mode < 5; ++mode) {
    const bool use_alt = alt >= 0 && (mode == MODE_GRAD || mode == MODE_GRAD3 || mode == MODE_HVPQ);
    const int cmb = use_alt ? alt : combo;
    const int nthr = lanes::lanes_threads(kLanesCombos[cmb].nw, kLanesCombos[cmb].prod);
    lanes_fn fn = lanes_kernel(H, cmb, mode);
    cudaError_t ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(lanes sweep)", ce);
    int occ = 0;
    ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, nthr, smem);
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
    bool ok;
    if (tile == 32) {
      ok = encode_2d(&a.tm_amp[sidx], d.amp, 2ull * d.n, (unsigned long long)R * H, (unsigned long long)d.stride * 16,
                     2 * tile, rows_box, false);
    } else {  // (2 doubles x events, resonance [stride H planes], helicity [stride 1 plane]) -> stage [h][slot][8 events]
      const unsigned long long dims[3] = {2ull * d.n, (unsigned long long)R, (unsigned long long)H};
      const unsigned long long strides[2] = {(unsigned long long)H * d.stride * 16, (unsigned long long)d.stride * 16};
      const unsigned box[3] = {2u * tile, (unsigned)RP, (unsigned)H};
      ok = encode_3d_swz128(&a.tm_amp[sidx], d.amp, dims, strides, box);
    }
    ok = ok && encode_2d(&a.tm_mass[sidx], d.mass, (unsigned long long)d.n, (unsigned long long)C,
                         (unsigned long long)d.stride * 8, tile, C);
    if (ok && d.weight)
      ok = encode_2d(&a.tm_wgt[sidx], d.weight, (unsigned long long)d.n, 1, up((unsigned)((d.n * 8) & 0x7fffffff), 16) + 16,
                     tile, 1);
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
  h->lanes_combo_alt = alt;
  if (h->lanes_combo_alt >= 0)
    h->block_alt = lanes::lanes_threads(kLanesCombos[h->lanes_combo_alt].nw, kLanesCombos[h->lanes_combo_alt].prod);
  h->variant = 2;
  h->block = nthreads;
  h->grid = h->num_sms;
  std::snprintf(h->variant_name, sizeof(h->variant_name), "lanes(rho=%d,sw=%d,nw=%d%s,tile=%d,stages=%d)", rho, SW, nw, prod == 2 ? "g" : "", tile, stages);
  return PWA_OK;
}

pwa_status lanes_launch(pwa_handle* h, int mode, const double* theta, const double* v, const double* skip) {
  LaneArgs a = h->largs;
  a.theta = theta;
  a.v = v;
  a.skip = skip;
  a.partial = h->d_partial;
  const bool use_alt = h->lanes_combo_alt >= 0 && (mode == MODE_GRAD || mode == MODE_GRAD3 || mode == MODE_HVPQ);
  lanes_fn fn = lanes_kernel(h->n_hel, use_alt ? h->lanes_combo_alt : h->lanes_combo, mode);
  fn<<<h->grid, use_alt ? h->block_alt : h->block, h->lanes_smem, h->stream>>>(a);
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch lanes sweep kernel", ce);
  return PWA_OK;
}


}  // namespace pwa
