/*
 * pwa.h - C ABI of the B200-native partial-wave-analysis likelihood library (libpwa_b200.so).
 *
 * What the library computes (all arithmetic fp64, on one CUDA device, in hand-written sm_100a kernels):
 *
 *   intensity   I_i = sum_h | sum_r z_r(i) F_rh(i) |^2                      PAPER.md:57-60 (Eq. 1, 1/2 dropped:
 *                                                                            DESIGN.md reading S1)
 *   z_r(i) = a_r e^{i phi_r} / (M_r^2 - m_{ch(r)}(i)^2 - i M_r Gamma_r)      BASELINE.json configs[0] (S4)
 *   NLL(theta) = - sum_data w_i ln I_i + W ln( sum_mc I_j / N_mc ),  W = sum_data w_i
 *                                                                            PAPER.md:67 (Eq. 3), S2, S3
 *   grad NLL, and (Hessian of NLL) . v for a given direction v               PAPER.md:90 (Eq. 6), :95 (Eq. 7, S9)
 *   a projected, truncated line-search Newton-CG minimisation of NLL         PAPER.md:27, :43, :119; S15', S19
 *   K values / K Hessian-vector products in one pass over the events, the Hessian matrix (pwa_nll_batch ...)
 *   additive raw sums of an event shard and their combination (Eqs. 4-7), fit fractions (S20)
 *   optionally (pwa_create_rich): partial waves sharing a resonance's lineshape, mass-dependent width, Flatte (S21, S22)
 *
 * Parameters: theta[4r..4r+3] = (a_r, phi_r, M_r, Gamma_r), r = 0..n_res-1 (S6); P = 4*n_res doubles
 * (pwa_create_rich handles: [a, phi per wave | M, Gamma per resonance], P = 2 n_res + 2 n_lineshape).
 * F_rh(i) ("amp") is the parameter-free projection of PAPER.md:70, an input computed once by the caller.
 *
 * Conventions
 *   - Every call returns a pwa_status; nothing throws across this boundary; no global state (one exception: the scratch
 *     array of pwa_nll_grad_hvp_static).  One handle = one device
 *     + one stream; a handle is not thread-safe, different handles are independent.  Every call binds the calling
 *     thread to the handle's device for its duration and restores the caller's current device before it returns, so
 *     a handle may be used from any host thread (one thread per GPU).
 *   - There is no CPU path.  If no CUDA device is usable, pwa_create fails with PWA_ERR_CUDA.
 *   - Evaluation calls (pwa_nll ... pwa_raw_sums, pwa_combine) only ENQUEUE work on the handle's stream
 *     and return; they never synchronise.  Their theta / v / output pointers are DEVICE pointers that
 *     must stay valid until the stream has run the work.  Outputs may not alias inputs.
 *   - pwa_fit_newton_cg, pwa_status_flags and the *_host convenience calls synchronise the stream.
 *   - Results are bit-identical between repeated calls with identical inputs on the same device
 *     (fixed grid, fixed event -> thread map, fixed-order reductions, no floating-point atomics).
 */
#ifndef PWA_B200_H
#define PWA_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PWA_MAX_RES 512   /* n_res  <= 512 */
#define PWA_MAX_HEL 8     /* n_hel  <= 8   */
#define PWA_MAX_CHAN 16   /* n_chan <= 16  */

typedef struct pwa_handle pwa_handle; /* opaque, owned by the library */

typedef enum {
  PWA_OK = 0,
  PWA_ERR_INVALID_ARG = 1,   /* null pointer, size out of range, misaligned buffer, bad res_chan ... */
  PWA_ERR_CUDA = 2,          /* a CUDA runtime call failed (see pwa_last_error) or no device */
  PWA_ERR_OOM = 3,           /* device (or pinned host) allocation failed */
  PWA_ERR_NONFINITE = 4,     /* fit: NLL or gradient not finite at the start point */
  PWA_ERR_NOT_CONVERGED = 5  /* fit: stopped without meeting the convergence classification (S19) */
} pwa_status;

typedef enum { PWA_MEM_HOST = 0, PWA_MEM_DEVICE = 1 } pwa_memkind;

/* One event sample (data or phase-space MC).  Layouts (event index fastest):
 *   mass  [n_chan][stride]            fp64, invariant mass m_c(i) in GeV of channel c
 *   amp   [n_res][n_hel][stride][2]   fp64, (Re, Im) of F_rh(i), amplitude-major, interleaved complex
 *   weight[n_events] or NULL          fp64, NULL = unit weights
 * `stride` is the distance in EVENTS between consecutive planes (>= n_events; 0 means n_events). */
typedef struct {
  int64_t n_events;
  int64_t stride;
  const double* mass;
  const double* amp;
  const double* weight;
} pwa_sample;

typedef struct {
  int32_t n_res, n_hel, n_chan;
  const int32_t* res_chan; /* [n_res] HOST pointer, channel of each resonance, values in [0, n_chan) */
  pwa_sample data, mc;     /* mc.weight must be NULL (unweighted phase space, S10) */
  pwa_memkind mem;         /* where data/mc mass, amp, weight live */
  int32_t borrow;          /* PWA_MEM_DEVICE only. 1: adopt the device pointers (zero copy; the caller
                              keeps them alive and unchanged for the life of the handle; amp must be
                              16-byte aligned, mass/weight 8-byte aligned).  0: the library copies and
                              the caller may free its buffers when pwa_create returns.  The copy is laid out
                              for the kernel the handle selects: planes as above, or - for shapes whose
                              32-event tile does not fit twice in shared memory, e.g. n_res = 100, n_hel = 4 -
                              8-event tiles that one bulk copy moves into shared memory (about 20 % faster
                              there than the same kernel over borrowed planes; same results bit for bit;
                              pwa_kernel_variant then says "tile=8t"; while pwa_create runs the copy exists
                              beside the caller's buffers; PWA_TILED=0 in the environment keeps planes). */
  int32_t device;          /* CUDA device ordinal */
  void* stream;            /* cudaStream_t, or NULL for the legacy default stream */
} pwa_model_desc;

/* Creates a handle: validates the descriptor (PWA_ERR_INVALID_ARG on: null desc/out/res_chan/mass/amp,
 * n_res not in [1,PWA_MAX_RES], n_hel not in [1,PWA_MAX_HEL], n_chan not in [1,PWA_MAX_CHAN],
 * res_chan out of range, n_events < 1, stride < n_events, mc.weight != NULL, misaligned borrowed
 * buffers), uploads or adopts the event store, allocates scratch.  *out is NULL on failure. */
pwa_status pwa_create(const pwa_model_desc* model, pwa_handle** out);
pwa_status pwa_destroy(pwa_handle* h); /* NULL is allowed */
int32_t pwa_n_params(const pwa_handle* h); /* P: 4*n_res (2*n_res + 2*n_lineshape for a pwa_create_rich handle); -1 for NULL */

/* ---- richer model: partial waves sharing resonance lineshapes, lineshape kinds (readings S21, S22) -------
 * Eq. 1 sums partial-wave amplitudes Lambda_m U_m; a resonance contributes several partial waves
 * ("phase angles and couplings of individual partial wave amplitudes") that share its mass and width
 * (Table 1).  With a pwa_rich_desc the n_res plane groups of the model descriptor are PARTIAL WAVES m (coupling
 * a_m e^{i phi_m}, planes F_mh); wave m takes its lineshape 1/D_l from resonance l = wave_res[m]:
 *     A_h(i) = sum_m a_m e^{i phi_m} F_mh(i) / D_{wave_res[m]}(i)
 * Lineshape kinds, m = mass[ls_chan[l]][i], parameters (M, Gamma) per resonance:
 *   PWA_LS_CONST    D = M^2 - m^2 - i M Gamma                                                  (S4)
 *   PWA_LS_MASSDEP  D = M^2 - m^2 - i M Gamma(m), Gamma(m) = Gamma (q(m)/q(M))^(2L+1) M/m, q = break-up momentum of
 *                   (m1, m2); no barrier factors; shape = (m1, m2, L, -, -, -); needs M and every m above m1 + m2
 *                   (else the result is NaN and the non-finite flag is raised)
 *   PWA_LS_FLATTE   D = M^2 - m^2 - i Gamma (rho_1(m) + Rg rho_2(m)), rho_k = 2 q_k(m)/m for the channels (m1, m2) and
 *                   (m3, m4), continued analytically below a threshold; "Gamma" is the coupling g_1, Rg = g_2/g_1
 *                   fixed; shape = (m1, m2, m3, m4, Rg, -)
 * Parameter layout of such a handle: theta = [a_0, phi_0, ..., a_{W-1}, phi_{W-1}, M_0, Gamma_0, ..., M_{L-1},
 * Gamma_{L-1}], P = 2 n_res + 2 n_lineshape; every entry point (evaluation, raw sums, fit and its box, Hessian) uses
 * it.  model->res_chan is ignored (channels come from ls_chan).  All arrays are HOST pointers, copied.
 * Cost: models whose resonances are all PWA_LS_CONST run on the fast kernels (two extra tiny launches per evaluation
 * expand theta, v and contract the sums: exact by the chain rule); a model with any other kind runs on the general-
 * lineshape kernel (csrc/pwa_rich.cuh), which reads F twice per gradient / HVP evaluation.  pwa_fit_fractions returns
 * one fraction per RESONANCE (n_lineshape doubles): the coherent sum of its partial waves, any lineshape kind.  PWA_ERR_INVALID_ARG: n_lineshape not in [1, n_res], null
 * arrays, wave_res / ls_chan / ls_kind out of range.  rich == NULL: same as pwa_create. */
typedef enum { PWA_LS_CONST = 0, PWA_LS_MASSDEP = 1, PWA_LS_FLATTE = 2 } pwa_lineshape;
typedef struct {
  int32_t n_lineshape;      /* L resonances */
  const int32_t* wave_res;  /* [n_res]       resonance of each partial wave, values in [0, L) */
  const int32_t* ls_chan;   /* [L]           mass channel of each resonance */
  const int32_t* ls_kind;   /* [L]           pwa_lineshape; NULL = all PWA_LS_CONST */
  const double* ls_shape;   /* [L][6]        shape parameters per kind (above); may be NULL if every kind is CONST */
} pwa_rich_desc;
pwa_status pwa_create_rich(const pwa_model_desc* model, const pwa_rich_desc* rich, pwa_handle** out);

/* ---- evaluation: device pointers, enqueue only ------------------------------------------------
 * theta, v, grad, hv: P doubles; nll: 1 double.  PAPER.md:67 (Eq. 3), :90 (Eq. 6), :95 (Eq. 7). */
pwa_status pwa_nll(pwa_handle* h, const double* theta, double* nll);
pwa_status pwa_nll_grad(pwa_handle* h, const double* theta, double* nll, double* grad);
pwa_status pwa_hvp(pwa_handle* h, const double* theta, const double* v, double* hv);
/* the fused sweep: one streaming pass over all data and MC events gives all three */
pwa_status pwa_nll_grad_hvp(pwa_handle* h, const double* theta, const double* v, double* nll,
                            double* grad, double* hv);

/* ---- split evaluation for Newton-CG (the optimiser asks for many HVPs at one theta) -------------
 * pwa_nll_grad_for_hvp = pwa_nll_grad that also keeps, inside the handle, a copy of theta and the direction-
 * independent sums of the HVP (the compact sums P1, P2, P3 of DESIGN.md section 5.1).  pwa_hvp_cached(v) then gives
 * H(theta) v for the theta of the LAST pwa_nll_grad_for_hvp call with a lighter sweep (only the v-dependent sums:
 * 49 instead of 69 FP64 instructions per event and resonance).  Results equal pwa_hvp(theta, v) to rounding.
 * Other calls (pwa_nll, pwa_nll_grad, pwa_hvp, pwa_raw_sums ...) may come in between: they do not touch what is kept.
 * pwa_hvp_cached before any pwa_nll_grad_for_hvp: PWA_ERR_INVALID_ARG.  Device pointers, enqueue only. */
pwa_status pwa_nll_grad_for_hvp(pwa_handle* h, const double* theta, double* nll, double* grad);
pwa_status pwa_hvp_cached(pwa_handle* h, const double* v, double* hv);

/* ---- K evaluations in one pass over the event store (multi-start batching; 300 fits on the same events,
 * :133: 11+ starts per analysis; Table 1's parameter errors, :102-113, need the Hessian at the fitted point) ----------
 * pwa_nll_batch: nll[k] = NLL(theta[k]), k < K.  theta: DEVICE pointer, K x P doubles, row k = parameter set k; nll:
 * DEVICE pointer, K doubles.  The K sets share every read of the event store (HBM and shared memory): the value-only
 * sweep is bound by that feed, so K values cost little more than one.
 * pwa_hvp_cached_batch: hv[k] = H(theta) v[k], k < K, at the theta of the last pwa_nll_grad_for_hvp call (as
 * pwa_hvp_cached).  v, hv: DEVICE pointers, K x P doubles.  The K directions share the propagators, B F and A_h.
 * pwa_hessian: H[i][j] = d2 NLL / dtheta_i dtheta_j at theta, P x P doubles (DEVICE, row-major), through
 * pwa_nll_grad_for_hvp(theta) and pwa_hvp_cached_batch on the unit vectors; replaces the kept state.  Its inverse on
 * the free parameters is the covariance estimate behind Table 1's errors.
 * All three enqueue on the handle's stream and do not synchronise; each result equals the corresponding single call to
 * rounding (another summation tree).  K is split into the batch sizes the kernels are built for (values: 4 and 2,
 * directions: 3 and 2); shapes served by the generic or the 8-event-tile kernel, and remainders of one, take one pass
 * per evaluation.  The non-finite flag of pwa_status_flags refers to the last pass only.
 * PWA_ERR_INVALID_ARG: K < 1, null pointers, pwa_hvp_cached_batch before any pwa_nll_grad_for_hvp. */
pwa_status pwa_nll_batch(pwa_handle* h, int32_t K, const double* theta, double* nll);
pwa_status pwa_hvp_cached_batch(pwa_handle* h, int32_t K, const double* v, double* hv);
pwa_status pwa_hessian(pwa_handle* h, const double* theta, double* hess);

/* ---- shard interface (Eqs. 4-7) -----------------------------------------------
 * pwa_raw_sums runs the same streaming pass but stops before the logarithm / division of Eqs. 4, 6, 7
 * and writes the ADDITIVE raw sums of this handle's events:  raw[pwa_raw_size(h)] doubles (device)
 *   raw[0] = sum_data w ln I   raw[1] = W = sum_data w   raw[2] = G = sum_mc I   raw[3] = N_mc
 *   raw[4      .. 4+P)   gd = sum_data w g_i / I_i
 *   raw[4+P    .. 4+2P)  gG = sum_mc g_j
 *   raw[4+2P   .. 4+3P)  hd = sum_data w [ g_i (g_i.v)/I_i^2 - (H_i v)/I_i ]
 *   raw[4+3P   .. 4+4P)  hG = sum_mc H_j v
 * (g_i = grad_theta I_i, H_i = Hessian of I_i).  v may be NULL: the hd, hG blocks are then zero.
 * Raw sums of disjoint shards add element-wise (that sum is the one all-reduce of a multi-GPU run);
 * pwa_combine applies Eqs. 4, 6, 7 to the (summed) raw vector:
 *   NLL = -raw[0] + W ln(G/N_mc);  grad = -gd + W gG/G;  Hv = hd + W [ hG/G - gG (gG.v)/G^2 ].
 * nll, grad, hv may each be NULL (not wanted); hv requires v. */
int32_t pwa_raw_size(const pwa_handle* h); /* 4 + 4P */
pwa_status pwa_raw_sums(pwa_handle* h, const double* theta, const double* v, double* raw);
pwa_status pwa_combine(pwa_handle* h, const double* raw, const double* v, double* nll, double* grad,
                       double* hv);

/* ---- fit ---------------------------------------------------------------------------------------
 * Projected, truncated line-search Newton-CG (Nocedal & Wright Alg. 7.1 for the inner CG; bound constraints by
 * projection, readings S15' and S19; the paper names SciPy's Newton-CG, mentions undefined
 * "constraint conditions", and gives no settings).  The start point is projected into the box; a
 * variable on a bound whose gradient pushes outward is frozen for the inner solve; trial points are projected, not
 * rejected.  gP below is the gradient with the frozen entries set to zero.  All vectors stay on the device; the
 * host reads back a few scalars per iteration for control flow.  The call replaces the state kept by
 * pwa_nll_grad_for_hvp (a pwa_hvp_cached after the fit refers to the fit's last gradient point). */
typedef struct {
  int32_t max_outer;      /* 500   outer Newton iterations */
  int32_t max_cg;         /* 50    CG iterations per outer step (BASELINE.json configs[4]) */
  double gtol;            /* 1e-5  stop when |gP|_inf <= gtol */
  double xtol;            /* 1e-8  stop when the accepted step |theta_new - theta|_inf <= xtol */
  double ftol;            /* 1e-12 stop when |f_new - f| <= ftol max(1,|f|) */
  double armijo_c1;       /* 1e-4 */
  double backtrack;       /* 0.5   step shrink factor rho */
  int32_t max_backtrack;  /* 40 */
  double max_seconds;     /* 0 = off; wall-time cap ("early stopping") */
  double gamma_min, gamma_max, mass_min, mass_max; /* bounds of the FIT only (S19): Gamma_r in [5e-3, 2], M_r in
                                                      [0.1, 4]; a pair (0,0) switches that box off */
  double gconv;           /* 1.0   a stopped fit counts as converged iff |gP|_inf <= gconv */
} pwa_fit_opts;

typedef struct {
  double nll;             /* NLL at the returned theta */
  double grad_inf_norm;   /* |gP|_inf there (projected gradient: entries frozen on a bound do not count) */
  int32_t outer_iters, cg_iters;
  int32_t n_nll, n_grad, n_hvp; /* sweeps of each kind */
  int32_t stop_reason;    /* 1 gtol, 2 xtol, 3 ftol, 4 max_outer, 5 max_seconds, 6 line search failed */
  int32_t status;         /* PWA_OK (converged), PWA_ERR_NOT_CONVERGED or PWA_ERR_NONFINITE */
  double seconds;         /* wall time of the call */
  int32_t n_active;       /* variables frozen on a bound at the returned theta */
} pwa_fit_result;

void pwa_fit_opts_default(pwa_fit_opts* opts);
/* theta_inout: DEVICE pointer, P doubles, start point in, final point out.  opts NULL = defaults.
 * Returns result->status (or PWA_ERR_INVALID_ARG / PWA_ERR_CUDA).  Synchronises the stream.
 * PWA_ERR_NONFINITE: the NLL or gradient at the (projected) start point, or the gradient at an accepted point, is not
 * finite; theta_inout then holds the last accepted point (the projected start point if no step was taken). */
pwa_status pwa_fit_newton_cg(pwa_handle* h, double* theta_inout, const pwa_fit_opts* opts,
                             pwa_fit_result* result);

/* ---- host-buffer convenience (the end-to-end path: copies in and out, synchronises) -------------
 * theta_host, v_host: P doubles in HOST memory (v_host may be NULL: then grad_host only);
 * nll_host 1 double, grad_host / hv_host P doubles in HOST memory (each may be NULL). */
pwa_status pwa_nll_grad_hvp_host(pwa_handle* h, const double* theta_host, const double* v_host,
                                 double* nll_host, double* grad_host, double* hv_host);

/* ---- allocation-free evaluation (no handle) ------------------------------------------------------
 * For callers that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc.  pwa_create allocates a handle's scratch; this ONE entry point needs no handle and calls no
 * cudaMalloc, cudaFree or allocating library routine: its scratch (per-resonance constants, per-block partial sums of
 * Eqs. 4-7, their column sums, the raw vector, the reduction's ticket) lives in a fixed
 * PWA_STATIC_SCRATCH_BYTES array in the library's device image, which every GPU that loads the library holds until
 * the process exits.  Same result as pwa_nll_grad_hvp on a handle created from the same descriptor (Eq. 3,
 * :90 Eq. 6, :95 Eq. 7) to rounding: the sweep is the event-per-thread kernel of csrc/pwa_kernels.cuh (the generic
 * variant), another summation tree than the tiled kernels; bit-identical between repeated calls on one device.
 *   model   as for pwa_create with mem = PWA_MEM_DEVICE: the event buffers are DEVICE pointers, read in place (borrow
 *           is ignored; amp 16-byte aligned, mass / weight 8-byte aligned); res_chan is a HOST pointer read during the
 *           call (passed to the kernels by value); model->stream is the stream the work is enqueued on.
 *   theta, v, nll, grad, hv   DEVICE pointers as for pwa_nll_grad_hvp, P = 4 n_res.  v may be NULL (then hv must be
 *           NULL); each of nll, grad, hv may be NULL (not wanted), not all three.  Outputs may not alias inputs.
 * Limits: n_res <= PWA_STATIC_MAX_RES (the partial rows of more resonances do not fit the fixed array), n_hel and
 * n_chan as for pwa_create, any number of events.  Beyond them: PWA_ERR_INVALID_ARG, message in pwa_last_error(NULL).
 * Enqueues three kernels and returns without synchronising.  The first call on each device also looks up the array's
 * device address and the launch configuration (host-side queries, no allocation by this library; the CUDA runtime
 * loads the kernels on their first launch): under graph capture make one call with the same n_res / n_hel before the
 * capture starts.
 * EVERY call on a device shares the one array, which keeps the previous call's contents (what must start at zero -
 * the reduction's ticket, the non-finite flag - is cleared by the call's first kernel).  Calls that overlap on the
 * GPU - two streams, or two host threads on different streams - race on it and give wrong results: order them on one
 * stream or with events.  The array holds no result a later call reads. */
#define PWA_STATIC_MAX_RES 64
#define PWA_STATIC_SCRATCH_BYTES (4u << 20) /* 4 MiB per device */
pwa_status pwa_nll_grad_hvp_static(const pwa_model_desc* model, const double* theta, const double* v, double* nll,
                                   double* grad, double* hv);

/* ---- fit fractions (Table 1 of the paper lists a "fraction" F_i per resonance; S20) ----
 * frac[r] = sum_mc sum_h |c_r B_r(j) F_rh(j)|^2 / sum_mc I_j  over the handle's phase-space MC sample.
 * pwa_create_rich handles: frac[l] = sum_mc sum_h |sum_{m in l} z_m(j) F_mh(j)|^2 / sum_mc I_j per resonance l.
 * theta: DEVICE pointer, P doubles; frac: DEVICE pointer, n_res (rich handles: n_lineshape) doubles.  Enqueues on the handle's stream (one pass
 * over the MC event store), does not synchronise.  PWA_ERR_INVALID_ARG on null pointers. */
pwa_status pwa_fit_fractions(pwa_handle* h, const double* theta, double* frac);

/* ---- diagnostics -------------------------------------------------------------------------------*/
/* Synchronises; *flags_host bit0 = the last evaluation produced a non-finite NLL, gradient or HVP. */
pwa_status pwa_status_flags(pwa_handle* h, uint32_t* flags_host);
/* Sweep-kernel timing for roofline reports: while enabled, the library brackets every sweep-kernel launch
 * with a pair of CUDA events on the handle's stream (at most 4096 pairs are kept; later launches are not
 * recorded).  pwa_profile_read synchronises the stream, returns the summed device time of the recorded
 * sweep launches in milliseconds and their count, and clears the record.  Either output may be NULL. */
pwa_status pwa_profile_enable(pwa_handle* h, int32_t on);
pwa_status pwa_profile_read(pwa_handle* h, double* total_ms, int64_t* n_launches);
/* Number of kernels this handle has launched since creation (never synchronises). */
int64_t pwa_kernel_launches(const pwa_handle* h);
/* Algorithmic HBM bytes one full evaluation reads: N_mc (16 R H + 8 C) + N_data (16 R H + 8 C [+8]). */
int64_t pwa_bytes_per_eval(const pwa_handle* h);
/* Name of the sweep-kernel variant the handle selected ("generic", ...), library-owned string. */
const char* pwa_kernel_variant(const pwa_handle* h);
/* Last error message of this handle (or of the last failed pwa_create if h is NULL). Library-owned. */
const char* pwa_last_error(const pwa_handle* h);
const char* pwa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PWA_B200_H */
