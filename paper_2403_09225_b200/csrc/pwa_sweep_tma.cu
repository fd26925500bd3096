// pwa_sweep_tma.cu - host side of the tiled TMA sweep: kernel table, tensor maps, launch configuration.
#include <cstdlib>
#include <cstring>

#include "pwa_internal.h"

namespace pwa {

// ---- kernel table: H in 1..4, RHO in 1..4; the thread cap follows from RHO (register budget) --------------
int tma_maxw(int rho) {
  switch (rho) {
    case 1: return 16;
    case 2: return 16;
    case 3: return 12;
    case 4: return 12;
  }
  return 0;
}

template <int H, int RHO>
static tma_fn tma_for_mode(int mode) {
  constexpr int MAXW = RHO <= 2 ? 16 : 12;  // compute warps + the producer warp
  switch (mode) {
    case MODE_NLL: return k_sweep_tma<H, RHO, MODE_NLL, MAXW>;
    case MODE_GRAD: return k_sweep_tma<H, RHO, MODE_GRAD, MAXW>;
    default: return k_sweep_tma<H, RHO, MODE_FULL, MAXW>;
  }
}

template <int H>
static tma_fn tma_for_rho(int rho, int mode) {
  switch (rho) {
    case 1: return tma_for_mode<H, 1>(mode);
    case 2: return tma_for_mode<H, 2>(mode);
    case 3: return tma_for_mode<H, 3>(mode);
    case 4: return tma_for_mode<H, 4>(mode);
  }
  return nullptr;
}

tma_fn tma_kernel(int H, int rho, int mode) {
  switch (H) {
    case 1: return tma_for_rho<1>(rho, mode);
    case 2: return tma_for_rho<2>(rho, mode);
    case 3: return tma_for_rho<3>(rho, mode);
    case 4: return tma_for_rho<4>(rho, mode);
  }
  return nullptr;
}

// ---- tensor maps --------------------------------------------------------------------------------------------
typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static encode_fn get_encode() {
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

// fp64 matrix [rows][row_stride_bytes / 8], valid extent (cols, rows), box (box_cols, box_rows); OOB reads give 0
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
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

static int env_int(const char* name, int dflt) {
  const char* e = std::getenv(name);
  return (e && *e) ? std::atoi(e) : dflt;
}

static inline unsigned up(unsigned x, unsigned m) { return (x + m - 1) / m * m; }

// ---- configuration at handle creation ----------------------------------------------------------------------
pwa_status tma_configure(pwa_handle* h, std::string& why) {
  const int R = h->n_res, H = h->n_hel, C = h->n_chan;
  const char* force = std::getenv("PWA_VARIANT");
  if (force && std::strcmp(force, "generic") == 0) { why = "PWA_VARIANT=generic"; return PWA_OK; }
  if (H > 4) { why = "n_hel > 4"; return PWA_OK; }
  for (int sidx = 0; sidx < 2; ++sidx) {
    const SampleDev& d = h->smp[sidx];
    if (d.n >= (1LL << 30)) { why = "sample too long for 32-bit TMA coordinates"; return PWA_OK; }
    if ((d.stride & 1) || ((uintptr_t)d.mass & 15) || ((uintptr_t)d.amp & 15) || (d.weight && ((uintptr_t)d.weight & 15))) {
      why = "event store not 16-byte aligned per plane (odd stride or misaligned base)";
      return PWA_OK;
    }
  }
  // resonances per thread: the register budget caps the slice count per RHO (tma_maxw)
  int rho = env_int("PWA_RHO", 0);
  if (rho == 0) {
    if (R <= 10) rho = 1;
    else if (R <= 20) rho = 2;
    else if (R <= 30) rho = 3;
    else rho = 4;
  }
  if (rho < 1 || rho > 4) { why = "bad PWA_RHO"; return PWA_OK; }
  const int S = (R + rho - 1) / rho;
  if (S + 1 > tma_maxw(rho)) { why = "too many resonances for the tiled kernel"; return PWA_OK; }

  const int RH = R * H;
  const int nbox = (RH + 255) / 256, rows_box = (RH + nbox - 1) / nbox;
  const unsigned amp_bytes = (unsigned)nbox * rows_box * TILE * 16, mass_bytes = (unsigned)C * TILE * 8;
  const unsigned stage_bytes = up(amp_bytes + mass_bytes + TILE * 8, 128);
  auto fixed_bytes = [&](int mode, unsigned* off) {
    const int NQ = mode == MODE_FULL ? 2 * H : H;
    unsigned o = 0;
    off[0] = o; o += 2u * S * NQ * TILE * 16;   // part
    off[1] = o; o += 2u * NQ * TILE * 16;       // tot
    off[2] = o; o += (unsigned)R * KS * 8;       // K
    off[3] = o;
    off[4] = o; o += 8u * (2 * 8 + 4);           // mbarriers: full, empty (<= 8 stages each), pf[2], tf[2]
    return up(o, 128);
  };
  unsigned off_full[5];
  const unsigned fixed_full = fixed_bytes(MODE_FULL, off_full);
  int dev_smem = 0;
  cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  int sm_smem = 0;
  cudaDeviceGetAttribute(&sm_smem, cudaDevAttrMaxSharedMemoryPerMultiprocessor, h->device);
  int bps = env_int("PWA_BPS", 0);
  if (bps <= 0) bps = std::max(1, std::min(8, 20 / (S + 1)));
  int stages = 0;
  for (; bps >= 1; --bps) {
    const long long budget = std::min<long long>(dev_smem, sm_smem / bps - 1024);
    stages = (int)std::min<long long>(8, (budget - (long long)fixed_full) / stage_bytes);
    if (stages >= 3 || (bps == 1 && stages >= 2)) break;
  }
  if (bps < 1 || stages < 2) { why = "tile does not fit in shared memory"; return PWA_OK; }
  const int st_env = env_int("PWA_STAGES", 0);
  if (st_env >= 2 && st_env <= stages) stages = st_env;

  int occ_min = 1 << 30;
  for (int mode = 0; mode < 3; ++mode) {
    tma_fn fn = tma_kernel(H, rho, mode);
    if (!fn) { why = "no kernel instance"; return PWA_OK; }
    unsigned off[5];
    const unsigned fixed = fixed_bytes(mode, off);
    const size_t smem = (size_t)stages * stage_bytes + fixed;
    cudaError_t ce = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_smem);
    if (ce != cudaSuccess) return set_error(h, PWA_ERR_CUDA, "cudaFuncSetAttribute(tma sweep)", ce);
    int occ = 0;
    ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, (S + 1) * 32, smem);
    if (ce != cudaSuccess || occ < 1) {
      cudaGetLastError();
      why = "tiled kernel cannot be resident (registers / shared memory)";
      return PWA_OK;
    }
    occ_min = std::min(occ_min, occ);
    TmaArgs& a = h->targs[mode];
    std::memset(&a, 0, sizeof(a));
    a.R = R; a.C = C; a.S = S; a.stages = stages; a.nbox = nbox; a.rows_box = rows_box;
    a.weighted = h->smp[1].weight != nullptr;
    a.stage_bytes = stage_bytes; a.amp_bytes = amp_bytes; a.mass_bytes = mass_bytes;
    const unsigned base = (unsigned)stages * stage_bytes;
    a.off_part = base + off[0]; a.off_tot = base + off[1]; a.off_K = base + off[2];
    a.off_bar = base + off[4];
    a.ch = h->d_ch;
    for (int sidx = 0; sidx < 2; ++sidx) {
      const SampleDev& d = h->smp[sidx];
      a.n[sidx] = d.n;
      bool ok = encode_2d(&a.amp[sidx], d.amp, 2ull * d.n, (unsigned long long)RH, (unsigned long long)d.stride * 16, 2 * TILE, rows_box) &&
                encode_2d(&a.mass[sidx], d.mass, (unsigned long long)d.n, (unsigned long long)C, (unsigned long long)d.stride * 8, TILE, C);
      if (ok && d.weight)
        ok = encode_2d(&a.wgt[sidx], d.weight, (unsigned long long)d.n, 1, up((unsigned)((d.n * 8) & 0x7fffffff), 16) + 16, TILE, 1);
      if (!ok) { why = "cuTensorMapEncodeTiled failed"; return PWA_OK; }
    }
    h->tma_smem[mode] = smem;
  }
  const int bps_env = env_int("PWA_BPS", 0);
  const int use_bps = bps_env > 0 ? std::min(bps_env, occ_min) : std::min(bps, occ_min);
  h->variant = 1;
  h->tma_rho = rho;
  h->block = (S + 1) * 32;
  h->grid = h->num_sms * use_bps;
  std::snprintf(h->variant_name, sizeof(h->variant_name), "tma(rho=%d,S=%d,stages=%d,bps=%d)", rho, S, stages, use_bps);
  return PWA_OK;
}

pwa_status tma_launch(pwa_handle* h, int mode, const double* theta, const double* v) {
  TmaArgs a = h->targs[mode];
  a.theta = theta;
  a.v = v;
  a.partial = h->d_partial;
  tma_fn fn = tma_kernel(h->n_hel, h->tma_rho, mode);
  fn<<<h->grid, h->block, h->tma_smem[mode], h->stream>>>(a);
  if (cudaError_t ce = cudaGetLastError()) return set_error(h, PWA_ERR_CUDA, "launch tma sweep kernel", ce);
  return PWA_OK;
}

}  // namespace pwa
