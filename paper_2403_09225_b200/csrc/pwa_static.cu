// pwa_static.cu - pwa_nll_grad_hvp_static (include/pwa.h): the fused evaluation without a handle and without any
// allocation.  Prologue + generic sweep + reduction / unpack / combine (pwa_kernels.cuh, SURVEY 8(a) rows a-1 .. a-7)
// with every piece of scratch in ONE file-scope device array instead of the handle's cudaMalloc'ed buffers.
//
// The array's name is a host-side stand-in in host code, not a device address: the host gets the address once per
// device from cudaGetSymbolAddress (device_state below) and hands pointers into it to the kernels; the prologue
// variant of this file names the array directly, which device code may.
#include <cstdio>
#include <mutex>

#include "pwa_internal.h"
#include "pwa_kernels.cuh"

namespace {
using namespace pwa;

constexpr int kMaxRes = PWA_STATIC_MAX_RES;
constexpr size_t kScratchDoubles = PWA_STATIC_SCRATCH_BYTES / sizeof(double);
constexpr int kBlock = 256;
constexpr int kReduceBlocks = 8;

constexpr size_t round32(size_t x) { return (x + 31) / 32 * 32; }
constexpr int nb_of(int R, int mode) { return mode == MODE_NLL ? 0 : (R + rpb_of(mode) - 1) / rpb_of(mode); }

// layout of the array, in doubles (every region starts on a 256-byte boundary)
constexpr size_t kRowMax = (size_t)nb_of(kMaxRes, MODE_FULL) * 32 + 2;  // longest partial row (MODE_FULL at kMaxRes)
constexpr size_t OFF_FLAGS = 0;                                         // unsigned[2]: non-finite flag, reduction ticket
constexpr size_t OFF_CH = 32;                                           // int[kMaxRes]: mass channel of each resonance
constexpr size_t OFF_K = OFF_CH + round32(kMaxRes / 2);                 // [kMaxRes][KSTRIDE] per-resonance constants
constexpr size_t OFF_SUMS = OFF_K + round32((size_t)kMaxRes * KSTRIDE);  // [2][row] column sums of the partials
constexpr size_t OFF_RAW = OFF_SUMS + round32(2 * kRowMax);             // raw vector, 4 + 4P
constexpr size_t OFF_PARTIAL = OFF_RAW + round32(4 + 16 * (size_t)kMaxRes);  // [2][grid][row] per-block partial rows
static_assert(nb_of(kMaxRes, MODE_GRAD) * 32 + 2 <= (int)kRowMax, "MODE_FULL has the longest rows");
static_assert(OFF_PARTIAL + 2 * 148 * kRowMax <= kScratchDoubles, "one block per SM of a B200 must fit at PWA_STATIC_MAX_RES");
static_assert((size_t)(kBlock / 32) * kRowMax * sizeof(double) <= 48 * 1024, "the sweep stays under the default shared-memory limit");

static __device__ __align__(256) double g_scratch[kScratchDoubles];

struct ChanList {
  int ch[kMaxRes];
};

// Variant of k_prologue (pwa_kernels.cuh) that writes into the static array: the per-resonance constants of theta and
// v, the channel list (a kernel argument: no host -> device copy), and zeroes of what a call must find at zero.
__global__ void k_prologue_static(const double* __restrict__ theta, const double* __restrict__ v, int R, const ChanList cl) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0) {
    unsigned* f = reinterpret_cast<unsigned*>(g_scratch + OFF_FLAGS);
    f[0] = 0u;  // non-finite flag
    f[1] = 0u;  // ticket of k_reduce_unpack (a call cut short by an error could have left it mid-count)
  }
  if (r >= R) return;
  reinterpret_cast<int*>(g_scratch + OFF_CH)[r] = cl.ch[r];
  const double a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
  double s, c;
  sincos(phi, &s, &c);
  const cplx e = {c, s};
  const cplx cc = {a * c, a * s};
  double* k = g_scratch + OFF_K + (size_t)r * KSTRIDE;
  k[K_M2] = M * M;
  k[K_Y] = M * G;
  k[K_Y2] = (M * G) * (M * G);
  k[3] = 0.0;
  k[K_CR] = cc.re;
  k[K_CI] = cc.im;
  cplx al = {0.0, 0.0}, be = {0.0, 0.0};
  if (v) {
    // alpha = e v_a + i c v_phi ;  beta = c lambda,  lambda = -(2M - i Gamma) v_M + i M v_Gamma  (pwa_common.cuh)
    const double va = v[4 * r], vp = v[4 * r + 1], vM = v[4 * r + 2], vG = v[4 * r + 3];
    al = cadd(cscale(e, va), cscale(cmuli(cc), vp));
    const cplx lam = {-2.0 * M * vM, G * vM + M * vG};
    be = cmul(cc, lam);
  }
  k[K_AR] = al.re;
  k[K_AI] = al.im;
  k[K_BR] = be.re;
  k[K_BI] = be.im;
  k[10] = 0.0;
  k[11] = 0.0;
}

typedef void (*sweep_fn)(const SweepArgs);

template <int MODE>
sweep_fn sweep_for_h(int H) {
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

sweep_fn sweep_kernel(int H, int mode) {
  return mode == MODE_NLL ? sweep_for_h<MODE_NLL>(H) : mode == MODE_GRAD ? sweep_for_h<MODE_GRAD>(H) : sweep_for_h<MODE_FULL>(H);
}

// ---- per-device set-up: the array's device address, the SM count, blocks per SM of every (mode, H) at kMaxRes ------
constexpr int kMaxDevices = 64;
struct DeviceState {
  bool ready = false;
  double* scratch = nullptr;  // device address of g_scratch ON THIS DEVICE
  int num_sms = 0;
  int occ[3][PWA_MAX_HEL + 1] = {};
};
DeviceState g_dev[kMaxDevices];
std::mutex g_dev_mutex;

// the caller has made `device` current
pwa_status device_state(int device, const DeviceState** out) {
  std::lock_guard<std::mutex> lk(g_dev_mutex);
  DeviceState& d = g_dev[device];
  if (!d.ready) {
    void* p = nullptr;
    cudaError_t ce = cudaGetSymbolAddress(&p, g_scratch);
    if (ce != cudaSuccess || p == nullptr) return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: cudaGetSymbolAddress(g_scratch)", ce);
    if ((ce = cudaDeviceGetAttribute(&d.num_sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess || d.num_sms < 1)
      return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: cudaDeviceGetAttribute", ce);
    // blocks per SM at the largest shared-memory footprint a mode can ask for: the grid then depends on (device, mode,
    // n_hel, n_res) only, so that repeated calls use the same event -> thread map
    for (int mode = 0; mode < 3; ++mode)
      for (int H = 1; H <= PWA_MAX_HEL; ++H) {
        int occ = 0;
        const size_t smem = (size_t)(kBlock / 32) * ((size_t)nb_of(kMaxRes, mode) * 32 + 2) * sizeof(double);
        ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sweep_kernel(H, mode), kBlock, smem);
        if (ce != cudaSuccess) return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: occupancy query", ce);
        d.occ[mode][H] = occ < 1 ? 1 : occ;
      }
    d.scratch = static_cast<double*>(p);
    d.ready = true;
  }
  *out = &d;
  return PWA_OK;
}

pwa_status bad(const char* what) {
  char msg[320];
  std::snprintf(msg, sizeof(msg), "pwa_nll_grad_hvp_static: %s", what);
  return set_error(nullptr, PWA_ERR_INVALID_ARG, msg, cudaSuccess);
}

bool sample_ok(const pwa_sample& s) {
  return s.n_events >= 1 && (s.stride == 0 || s.stride >= s.n_events) && s.mass && s.amp && !((uintptr_t)s.amp & 15) &&
         !((uintptr_t)s.mass & 7) && !((uintptr_t)s.weight & 7);
}

SampleDev sample_dev(const pwa_sample& s) {
  SampleDev d;
  d.mass = s.mass;
  d.amp = reinterpret_cast<const double2*>(s.amp);
  d.weight = s.weight;
  d.n = s.n_events;
  d.stride = s.stride ? s.stride : s.n_events;
  return d;
}
}  // namespace

extern "C" pwa_status pwa_nll_grad_hvp_static(const pwa_model_desc* m, const double* theta, const double* v, double* nll,
                                              double* grad, double* hv) {
  if (!m || !theta) return bad("null descriptor or theta");
  if (!nll && !grad && !hv) return bad("no output wanted");
  if (hv && !v) return bad("hv needs v");
  if (m->n_res < 1) return bad("n_res < 1");
  if (m->n_res > kMaxRes) {
    char msg[256];
    std::snprintf(msg, sizeof(msg), "n_res = %d exceeds PWA_STATIC_MAX_RES = %d: the fixed %u-byte scratch array cannot hold its partial sums (use a handle)",
                  m->n_res, kMaxRes, (unsigned)PWA_STATIC_SCRATCH_BYTES);
    return bad(msg);
  }
  if (m->n_hel < 1 || m->n_hel > PWA_MAX_HEL) return bad("n_hel out of range");
  if (m->n_chan < 1 || m->n_chan > PWA_MAX_CHAN) return bad("n_chan out of range");
  if (m->mem != PWA_MEM_DEVICE) return bad("the event buffers must be device memory (mem = PWA_MEM_DEVICE): nothing is copied");
  if (!m->res_chan) return bad("null res_chan");
  if (!sample_ok(m->data) || !sample_ok(m->mc)) return bad("bad sample (n_events < 1, stride < n_events, null or misaligned buffer)");
  if (m->mc.weight) return bad("mc.weight must be NULL (unweighted phase space)");
  const int R = m->n_res, H = m->n_hel;
  ChanList cl;
  for (int r = 0; r < kMaxRes; ++r) {
    cl.ch[r] = r < R ? m->res_chan[r] : 0;
    if (cl.ch[r] < 0 || cl.ch[r] >= m->n_chan) return bad("res_chan value out of range");
  }
  if (m->device < 0 || m->device >= kMaxDevices) return bad("device ordinal out of range");
  DeviceGuard guard(m->device);
  {
    int cur = -1;
    cudaError_t ce = cudaGetDevice(&cur);
    if (ce != cudaSuccess || cur != m->device) return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: cudaSetDevice", ce);
  }
  const DeviceState* ds = nullptr;
  if (pwa_status st = device_state(m->device, &ds)) return st;

  const int mode = hv ? MODE_FULL : grad ? MODE_GRAD : MODE_NLL;
  const double* vv = mode == MODE_FULL ? v : nullptr;
  const int nb = nb_of(R, mode);
  const size_t row = (size_t)nb * 32 + 2;
  // blocks: whole multiples of the SM count, as many per SM as the kernel's occupancy allows and the array holds
  int per_sm = ds->occ[mode][H];
  while (per_sm > 1 && OFF_PARTIAL + 2 * (size_t)per_sm * ds->num_sms * row > kScratchDoubles) --per_sm;
  const int grid = per_sm * ds->num_sms;
  if (OFF_PARTIAL + 2 * (size_t)grid * row > kScratchDoubles) return bad("this device has too many SMs for the fixed scratch array");

  cudaStream_t stream = static_cast<cudaStream_t>(m->stream);
  double* S = ds->scratch;
  unsigned* flags = reinterpret_cast<unsigned*>(S + OFF_FLAGS);

  k_prologue_static<<<(R + 127) / 128, 128, 0, stream>>>(theta, vv, R, cl);
  if (cudaError_t ce = cudaGetLastError()) return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: launch k_prologue_static", ce);

  SweepArgs a;
  a.s[0] = sample_dev(m->mc);
  a.s[1] = sample_dev(m->data);
  a.K = S + OFF_K;
  a.ch = reinterpret_cast<const int*>(S + OFF_CH);
  a.R = R;
  a.C = m->n_chan;
  a.nb = nb;
  a.partial = S + OFF_PARTIAL;
  sweep_kernel(H, mode)<<<grid, kBlock, (size_t)(kBlock / 32) * row * sizeof(double), stream>>>(a);
  if (cudaError_t ce = cudaGetLastError()) return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: launch sweep kernel", ce);

  const double n_mc = (double)m->mc.n_events;
  const CgTail none = {};
#define PWA_REDUCE(M)                                                                                                      \
  k_reduce_unpack<M><<<kReduceBlocks, 1024, 0, stream>>>(S + OFF_PARTIAL, grid, nb, R, 0, theta, vv, n_mc, S + OFF_SUMS,  \
                                                          S + OFF_RAW, 1, nll, grad, hv, flags, flags + 1, nullptr, nullptr, none)
  switch (mode) {
    case MODE_NLL: PWA_REDUCE(MODE_NLL); break;
    case MODE_GRAD: PWA_REDUCE(MODE_GRAD); break;
    default: PWA_REDUCE(MODE_FULL); break;
  }
#undef PWA_REDUCE
  if (cudaError_t ce = cudaGetLastError()) return set_error(nullptr, PWA_ERR_CUDA, "pwa_nll_grad_hvp_static: launch k_reduce_unpack", ce);
  return PWA_OK;
}
