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

int producers_for(int stages) {
  const int cap = std::min(4, std::max(1, env_int("PWA_NPROD", 4)));
  for (int d = cap; d > 1; --d)
    if (stages % d == 0) return d;
  return 1;
}

int ring_stages(int fit, int group) {
  if (group < 1) group = 1;
  const int lo = std::max(2, group);
  int best = fit - fit % group;
  if (best < lo) return 0;
  const int less = best - group;
  if (less >= lo && less >= 3 && producers_for(less) > producers_for(best)) best = less;
  return best;
}

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

namespace {
// shared-memory plan of one entry of kLanesCombos for a model shape
struct Plan {
  int combo = -1, stages = 0;
  int rho = 0, log_sw = 0, nw = 0, prod = 0, tile = 0, SW = 0, RP = 0, NW = 0, nthreads = 0, nbox = 0, rows_box = 0;
  unsigned amp_bytes = 0, off_mass = 0, off_wgt = 0, stage_bytes = 0, k_bytes = 0, red_bytes = 0, xch_bytes = 0, fixed = 0;
};

// candidates: every instantiated shape with capacity >= R, smallest capacity first (ties: table order); the first
// whose stage fits in shared memory at least twice is taken.  PWA_COMBO forces one entry (A/B runs).  tiled: only the
// entries fed from a tiled store (PROD 4) / only the others.
bool pick_plan(int R, int H, int C, int dev_smem, bool tiled, Plan& p, std::string& why) {
  const int forced = env_int("PWA_COMBO", -1);
  why = H > 4 ? "no lanes-kernel instance for this n_hel" : "no lanes-kernel instance for this n_res";
  std::vector<int> order;
  for (int k = 0; k < kNumLanesCombos; ++k)
    if (forced < 0 || k == forced) order.push_back(k);
  std::stable_sort(order.begin(), order.end(), [](int x, int y) {
    return (kLanesCombos[x].rho << kLanesCombos[x].log_sw) < (kLanesCombos[y].rho << kLanesCombos[y].log_sw);
  });
  for (size_t oi = 0; oi < order.size() && p.combo < 0 && H <= 4; ++oi) {
    const int k = order[oi];
    const LanesCombo& c = kLanesCombos[k];
    const int cap = c.rho << c.log_sw;
    if ((c.prod == 4) != tiled) continue;
    if (cap < R || !lanes_kernel(H, k, MODE_FULL)) continue;
    if (forced < 0) {  // measured preference (profiles/r02_shapes.md); a forced entry is taken as it is
      // beyond 32 resonances a 32-event stage fits only a few times: the 8-event tiles (8 stages, one column per warp)
      // were faster in every shape measured (R = 33 .. 128, H = 1 .. 4), also at a larger padded capacity
      if (R > 32 && c.tile == 32) continue;
    }
    p.rho = c.rho; p.log_sw = c.log_sw; p.nw = c.nw; p.prod = c.prod; p.tile = c.tile;
    p.nthreads = lanes::lanes_threads(c.nw, c.prod);
    p.SW = 1 << c.log_sw; p.RP = c.rho * p.SW;
    p.NW = c.alt >= 0 ? std::max(c.nw, kLanesCombos[c.alt].nw) : c.nw;  // per-warp scratch sized for the larger of the two shapes
    if (c.prod == 4) {
      // the stage is the tile's image in the store: R*H amplitude rows of 128 bytes (no padding rows), masses, weights
      p.nbox = 1; p.rows_box = R * H;
      p.amp_bytes = (unsigned)R * H * c.tile * 16;
      p.red_bytes = up((unsigned)(R * 10 + 2) * 8, 128);
      p.off_mass = p.amp_bytes; p.off_wgt = p.off_mass + (unsigned)C * c.tile * 8;
      p.stage_bytes = up(p.off_wgt + c.tile * 8, 128);
    } else {
      if (c.tile == 32) {
        // amplitude rows incl. the zero-filled planes of padding resonances, in nbox boxes of rows_box (<= 256) rows
        const int rows_need = p.RP * H;
        p.nbox = (rows_need + 255) / 256; p.rows_box = (rows_need + p.nbox - 1) / p.nbox;
        p.amp_bytes = (unsigned)p.nbox * p.rows_box * c.tile * 16;
        p.red_bytes = up((unsigned)c.nw * (R * 10 + 2) * 8, 128);  // rows for the main shape's warps only
      } else {
        if (p.RP > 256) continue;  // one 3-D box [H][RP][8 events]
        p.nbox = 1; p.rows_box = p.RP;
        p.amp_bytes = (unsigned)H * p.RP * c.tile * 16;
        p.red_bytes = up((unsigned)(R * 10 + 2) * 8, 128);  // one row: the warps add into it in turn
      }
      p.off_mass = p.amp_bytes; p.off_wgt = up(p.off_mass + (unsigned)C * c.tile * 8, 128);  // TMA destinations: 128-byte aligned
      p.stage_bytes = up(p.off_wgt + c.tile * 8, c.tile == 32 ? 128 : 1024);
    }
    p.k_bytes = up((unsigned)p.RP * lanes::KS * 8, 128);
    p.xch_bytes = up((unsigned)p.NW * (32 / p.SW) * (4 * H + 2) * 8, 128);
    p.fixed = p.k_bytes + p.red_bytes + p.xch_bytes + 32u * 2 * 8 + 128;
    const int fit = (int)std::min<long long>(32, ((long long)dev_smem - p.fixed) / p.stage_bytes);
    // warps that keep their column (NW a multiple of the passes per tile) consume NW / NP tiles at the same time
    const int NP = c.tile / (32 / p.SW), group = (c.nw % NP == 0) ? c.nw / NP : 1;
    p.stages = ring_stages(std::min(8, fit), group);  // deeper rings were measured no faster; PWA_STAGES overrides
    const int st_env = env_int("PWA_STAGES", 0);
    if (st_env >= 2 && st_env <= fit && st_env % group == 0) p.stages = st_env;
    if (p.stages < 2) { why = "tile does not fit in shared memory"; continue; }
    p.combo = k;
  }
  return p.combo >= 0;
}
}  // namespace

bool lanes_wants_tiled(int device, int R, int H, int C, int* phase_mul, unsigned* tile_bytes, unsigned* off_mass, unsigned* off_wgt) {
  const char* e = std::getenv("PWA_TILED");
  if (e && e[0] == '0') return false;
  int dev_smem = 0;
  if (cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) != cudaSuccess) return false;
  std::string why;
  Plan plain, tiled;
  if (pick_plan(R, H, C, dev_smem, false, plain, why) && plain.tile != 8) return false;  // a 32-event tile fits: planes
  if (!pick_plan(R, H, C, dev_smem, true, tiled, why)) return false;
  *phase_mul = 32 / tiled.SW;
  *tile_bytes = tiled.stage_bytes;
  *off_mass = tiled.off_mass;
  *off_wgt = tiled.off_wgt;
  return true;
}

pwa_status lanes_configure(pwa_handle* h, std::string& why) {
  const int R = h->n_res, H = h->n_hel, C = h->n_chan;
  for (int sidx = 0; sidx < 2; ++sidx) {
    if (h->tiled) {
      if (h->tstore[sidx].n >= (1LL << 30)) return set_error(h, PWA_ERR_INVALID_ARG, "sample too long for the tiled store's 32-bit event index", cudaSuccess);
      continue;
    }
    const SampleDev& d = h->smp[sidx];
    if (d.n >= (1LL << 30)) { why = "sample too long for 32-bit TMA coordinates"; return PWA_OK; }
    if ((d.stride & 1) || ((uintptr_t)d.mass & 15) || ((uintptr_t)d.amp & 15) || (d.weight && ((uintptr_t)d.weight & 15))) {
      why = "event store not 16-byte aligned per plane (odd stride or misaligned base)";
      return PWA_OK;
    }
  }
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  Plan p;
  if (!pick_plan(R, H, C, dev_smem, h->tiled, p, why)) {
    if (h->tiled) return set_error(h, PWA_ERR_CUDA, "no kernel for the tiled store (internal)", cudaSuccess);
    return PWA_OK;
  }
  const int combo = p.combo, stages = p.stages, rho = p.rho, nw = p.nw, prod = p.prod, tile = p.tile, SW = p.SW, RP = p.RP,
            nthreads = p.nthreads, nbox = p.nbox, rows_box = p.rows_box;
  const unsigned amp_bytes = p.amp_bytes, off_mass = p.off_mass, off_wgt = p.off_wgt, stage_bytes = p.stage_bytes, k_bytes = p.k_bytes,
                 red_bytes = p.red_bytes, xch_bytes = p.xch_bytes, fixed = p.fixed;
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
      if (h->tiled) return set_error(h, PWA_ERR_CUDA, "the tiled-store kernel cannot be resident (internal)", ce);
      why = "lanes kernel cannot be resident (registers / shared memory)";
      return PWA_OK;
    }
  }
  LaneArgs& a = h->largs;
  std::memset(&a, 0, sizeof(a));
  a.weighted = h->weighted;
  for (int sidx = 0; sidx < 2; ++sidx) {
    if (h->tiled) {  // no tensor maps: the producer copies whole tiles
      a.n[sidx] = h->tstore[sidx].n;
      a.tiled[sidx] = h->tstore[sidx].base;
      continue;
    }
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
  a.nprod = producers_for(stages);
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
  std::snprintf(h->variant_name, sizeof(h->variant_name), "lanes(rho=%d,sw=%d,nw=%d%s,tile=%d%s,stages=%d)", rho, SW, nw, prod >= 2 && prod != 3 ? "g" : "", tile,
                prod == 4 ? "t" : "", stages);
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
