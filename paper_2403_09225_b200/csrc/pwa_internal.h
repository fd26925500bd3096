// pwa_internal.h - host-side handle layout shared by pwa_api.cu and pwa_fit.cu (not installed).
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/pwa.h"
#include "pwa_common.cuh"
#include "pwa_sweep_lanes.cuh"

struct pwa_handle {
  int device = 0;
  cudaStream_t stream = nullptr;
  int n_res = 0, n_hel = 0, n_chan = 0, n_par = 0;
  int num_sms = 0;
  bool weighted = false;

  // event store (a-0): device pointers, owned unless borrowed
  pwa::SampleDev smp[2];  // 0 = MC, 1 = data
  void* owned[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  int* d_ch = nullptr;
  // copy-mode handles whose shape needs 8-event tiles keep the events TILED (TiledDev, pwa_common.cuh) instead of as
  // planes: smp[].amp / mass / weight are then null and only the tiled-aware kernels (lanes sweep PROD 4, fit fractions)
  // may run; decided before the store is built (lanes_wants_tiled)
  bool tiled = false;
  pwa::TiledDev tstore[2];  // 0 = MC, 1 = data; base is owned

  // richer model (readings S21, S22; pwa_create_rich): the kernels work in the EXPANDED parameter space [n_res][4]
  // (every wave with its own a, phi, M, Gamma); user vectors are expanded before and contracted after a sweep
  bool mapped = false;          // user parameter layout [a, phi per wave | M, Gamma per resonance]
  bool rich_kernel = false;     // some resonance is not constant-width: k_sweep_rich (pwa_rich.cuh)
  int n_full = 0;               // 4 * n_res
  int n_ls = 0;                 // resonances (lineshapes)
  int* d_map = nullptr;         // [n_full] expanded index -> user index
  int* d_csr_off = nullptr;     // [n_par + 1] user parameter -> range in d_csr_idx
  int* d_csr_idx = nullptr;     // [n_full] expanded indices, ascending within a user parameter
  int* d_wres = nullptr;        // [n_res] resonance of each wave
  int* d_lch = nullptr;         // [n_ls] channel of each resonance
  int* d_lkind = nullptr;       // [n_ls]
  double* d_lshape = nullptr;   // [n_ls][6]
  int* d_wl_off = nullptr;      // [n_ls + 1] resonance -> range in d_wl_idx
  int* d_wl_idx = nullptr;      // [n_res] waves of each resonance, ascending
  double* d_full = nullptr;     // theta_full [n_full] | v_full [n_full] | raw_full [4 + 4 n_full] | K [n_res][16]

  // scratch
  double* d_K = nullptr;        // per-resonance constants
  double* d_partial = nullptr;  // per-block partial sums
  double* d_sums = nullptr;     // block-summed compact sums
  double* d_raw = nullptr;      // public raw vector (4 + 4P)
  unsigned* d_flags = nullptr;  // [0] non-finite flag of the last evaluation, [1] ticket counter of the reduction kernel
  size_t partial_doubles = 0;
  double* d_pcache = nullptr;      // [2][6 R + 2] compact sums P1..P3 + scalars of the last pwa_nll_grad_for_hvp
  double* d_theta_keep = nullptr;  // theta of that call
  bool keep_valid = false;

  // sweep launch configuration (fixed at creation -> deterministic event -> thread map)
  int grid = 0, block = 0;
  int variant = 0;  // 0 = generic (pwa_kernels.cuh), 2 = lanes (pwa_sweep_lanes.cuh)
  char variant_name[64] = "generic";
  // lanes variant (pwa_sweep_lanes.cuh)
  pwa::LaneArgs largs;
  size_t lanes_smem = 0;
  int lanes_combo = -1;
  int lanes_combo_alt = -1, block_alt = 0;  // shape of the lighter modes (MODE_GRAD, MODE_GRAD3, MODE_HVPQ), if another one
  bool weight_padded = false;  // the data weights are library-owned and padded to an even length

  // device staging for the *_host entry point and the fit driver
  double* d_io = nullptr;   // theta | v | nll | grad | hv   (1 + 4P doubles, padded)
  double* h_pin = nullptr;  // pinned host mirror of d_io
  double* d_fit = nullptr;  // fit vectors
  unsigned attr_done = 0;          // bit per kernel whose shared-memory attribute this handle has already set (pair modes 0..5, batch 8..)
  double* d_batch = nullptr;       // batch sweeps: per-block partial rows, column sums, one raw vector
  size_t batch_doubles = 0;
  double* h_fit = nullptr;  // pinned scalars of the fit driver

  long long launches = 0;
  bool profiling = false;
  std::vector<cudaEvent_t> prof_events;  // pairs (start, stop)
  size_t prof_used = 0;
  std::string err;
};

namespace pwa {
// fp64 matrix [rows][row_stride_bytes / 8], valid extent (cols, rows), box (box_cols, box_rows); out-of-bounds reads give 0
bool encode_3d_swz128(CUtensorMap* m, const void* base, const unsigned long long dims[3], const unsigned long long strides_bytes[2],
                      const unsigned box[3]);
bool encode_2d(CUtensorMap* m, const void* base, unsigned long long cols, unsigned long long rows,
               unsigned long long row_stride_bytes, unsigned box_cols, unsigned box_rows, bool swizzle128 = false);
// pwa_sweep_lanes.cu
typedef void (*lanes_fn)(const LaneArgs);
struct LanesCombo {
  int rho, log_sw, nw, prod, tile, alt;  // resonances per lane, log2(slices per warp), compute warps per block, producer kind
                                    // (0 warp, 2 warpgroup, 4 warpgroup + tiled store), events per tile (32, or 8 with the swizzled layout), and the
                                    // entry (same rho, slices, tile) used for the modes with fewer accumulators, whose registers allow a
                                    // third compute warp per scheduler (-1: none; no entry uses one since warps keep their columns:
                                    // the 8-warp warpgroup shape then measured faster in every mode)
};
// instantiated shapes (pwa_sweep_lanes_inst.cu); capacity RHO << LOG_SW resonances; the handle takes the first entry of
// the smallest capacity >= R whose stages fit in shared memory at least twice
constexpr LanesCombo kLanesCombos[] = {
    {1, 2, 15, 0, 32, -1}, {2, 3, 15, 0, 32, -1}, {3, 2, 11, 0, 32, -1}, {3, 2, 8, 2, 32, -1}, {4, 3, 8, 2, 32, -1}, {4, 3, 7, 0, 32, -1},
    {4, 4, 8, 2, 32, -1},  {4, 4, 7, 0, 32, -1},  {4, 5, 8, 2, 32, -1},  {4, 5, 7, 0, 32, -1}, {4, 4, 8, 2, 8, -1},  {4, 5, 8, 2, 8, -1},
    {4, 3, 11, 3, 32, -1}, {5, 1, 8, 2, 32, -1}, {4, 4, 8, 4, 8, -1},  {4, 5, 8, 4, 8, -1},
    // finer capacities (6, 8, 20, 48): fewer padding slots for model sizes between the shapes above
    {3, 1, 8, 2, 32, -1},  {4, 1, 8, 2, 32, -1},  {5, 2, 8, 2, 32, -1},  {3, 4, 8, 2, 32, -1}, {6, 0, 8, 2, 32, -1},
    {3, 3, 8, 2, 32, -1},  {3, 4, 8, 2, 8, -1},   {3, 4, 8, 4, 8, -1},   {3, 5, 8, 2, 8, -1},  {3, 5, 8, 4, 8, -1}};
constexpr int kNumLanesCombos = sizeof(kLanesCombos) / sizeof(kLanesCombos[0]);
lanes_fn lanes_kernel_h1(int combo, int mode);
lanes_fn lanes_kernel_h2(int combo, int mode);
lanes_fn lanes_kernel_h3(int combo, int mode);
lanes_fn lanes_kernel_h4(int combo, int mode);
lanes_fn lanes_kernel(int H, int combo, int mode);
// the fused sweep with two events per lane (pwa_sweep_pair.cuh); nullptr where it is not instantiated
struct PairArgs;
typedef void (*pair_fn)(const LaneArgs, const PairArgs);
pair_fn pair_kernel_h1(int mode);
pair_fn pair_kernel_h2(int mode);
pair_fn pair_kernel_h3(int mode);
pair_fn pair_kernel_h4(int mode);
// the handle's shape has a two-event kernel for this mode (MODE_FULLP, MODE_GRAD3, MODE_HVPQ); PWA_PAIR=0 switches it off
bool pair_available(const pwa_handle* h, int mode);
pwa_status pair_launch(pwa_handle* h, int mode, const double* theta, const double* v, const double* skip);
// batch kernels (pwa_batch.cuh): kind 0 = K parameter sets (value only), 1 = K directions at the kept theta
struct BatchArgs;
typedef void (*batch_fn)(const LaneArgs, const BatchArgs);
batch_fn batch_kernel_h1(int rho, int log_sw, int kind, int kb);
batch_fn batch_kernel_h2(int rho, int log_sw, int kind, int kb);
batch_fn batch_kernel_h3(int rho, int log_sw, int kind, int kb);
batch_fn batch_kernel_h4(int rho, int log_sw, int kind, int kb);
// one batch pass of kb (a supported count) sets / directions: sweep + reduction; false if this handle's shape has no batch kernel
bool batch_supported(const pwa_handle* h, int kind, int kb);
pwa_status batch_launch(pwa_handle* h, int kind, int kb, const double* theta, const double* v, double* out);
// Warps of a producer warpgroup that issue copies (pwa_sweep_lanes.cuh): the largest count <= 4 (PWA_NPROD lowers the
// cap) that DIVIDES the ring's stage count, so that a stage is always refilled by the same thread - the parity wait on a
// stage's empty barrier can only tell neighbouring phases apart, which is safe only in one thread's program order.
int producers_for(int stages);
// A ring of `fit` stages at most.  `group` = tiles that DIFFERENT warps consume at the same time (shapes whose warps keep
// their column: compute warps / passes per tile): the stage count must be a multiple of it, so that the tiles t and
// t + stages, which share a stage, are consumed by the same warps one after the other - a consumer that starts to wait
// for a stage's next phase before the current one has completed would be let through by the parity wait.  Among the
// admissible counts: `fit` rounded down, or one step less where that admits more producers (5 -> 4, 7 -> 6).
// Returns 0 if no admissible count >= 2 exists.
int ring_stages(int fit, int group);
pwa_status lanes_configure(pwa_handle* h, std::string& why);  // sets variant = 2 on success; PWA_OK + why if unsuitable
// Would a copy-mode handle of this shape run on 8-event tiles?  Then its store is built tiled (PROD 4 entries) and
// *phase_mul / *tile_bytes / *off_mass / *off_wgt describe the layout (TiledDev).  PWA_TILED=0 switches it off.
bool lanes_wants_tiled(int device, int R, int H, int C, int* phase_mul, unsigned* tile_bytes, unsigned* off_mass, unsigned* off_wgt);
pwa_status lanes_launch(pwa_handle* h, int mode, const double* theta, const double* v, const double* skip = nullptr);
// internal entry points used by the fit driver (enqueue only)
pwa_status eval(pwa_handle* h, int mode, const double* theta, const double* v, double* nll, double* grad,
                double* hv);
pwa_status eval_grad_keep(pwa_handle* h, const double* theta, double* nll, double* grad);
struct CgTail;  // pwa_kernels.cuh: a CG iteration run in the tail of the HVP's reduction launch (lanes variant, plain handles)
pwa_status eval_hvp_kept(pwa_handle* h, const double* v, double* hv, const double* skip = nullptr,  // skip: LaneArgs::skip
                         const CgTail* cg = nullptr);
pwa_status set_error(pwa_handle* h, pwa_status st, const char* what, cudaError_t ce);
pwa_status expand_theta(pwa_handle* h, const double* theta);  // rich handles: h->d_full[0 .. n_full) <- theta expanded
}  // namespace pwa

namespace pwa {
// Binds the calling thread to a handle's device for the duration of one C-ABI call and restores the caller's current
// device afterwards ("one handle = one device", include/pwa.h): a handle may be used from a thread whose current
// device is another one (one host thread per GPU).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; }
    if (prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched && prev >= 0) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};
}  // namespace pwa

#define PWA_CUDA_CHECK(h, call)                                              \
  do {                                                                       \
    cudaError_t ce__ = (call);                                               \
    if (ce__ != cudaSuccess) return pwa::set_error((h), PWA_ERR_CUDA, #call, ce__); \
  } while (0)
