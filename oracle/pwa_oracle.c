/*
 * pwa_oracle.c - plain, slow, CPU reference ("oracle") for the PWA likelihood hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may build, load or call it.  It shares no code
 * with the CUDA path (paper_2403_09225_b200/csrc) and neither includes the other.
 *
 * What it computes, one event at a time, straight from the definitions:
 *   intensity   I_i = sum_h | sum_r z_r(i) F_rh(i) |^2                PAPER.md:57-60 (Eq. 1; the 1/2 is
 *                                                                     dropped, reading S1)
 *   z_r(i) = a_r e^{i phi_r} / (M_r^2 - m_{ch(r)}(i)^2 - i M_r Gamma_r)   BASELINE.json configs[0] (BW form)
 *   NLL = - sum_data w_i ln I_i + W ln( sum_mc I_j / N_mc ),  W = sum_data w_i
 *                                                                     PAPER.md:67 (Eq. 3), sign flipped (S2),
 *                                                                     N_Data := W for weighted events (S3)
 *   gradient and Hessian-vector product of NLL by the chain rule written out by hand
 *                                                                     PAPER.md:90 (Eq. 6), :95 (Eq. 7, S9)
 * The per-shard raw sums (F_m, G_m and their derivatives) and the combination of
 * Eqs. 4, 6, 7 are separate entry points so that shard additivity can be tested.
 *
 * Parameters: theta[4r..4r+3] = (a_r, phi_r, M_r, Gamma_r)  (reading S6).  Parameters,
 *             directions and results cross this interface as REAL (so the finite-difference pins can
 *             work in 80-bit arithmetic); event data is fp64.
 * Layouts:    mass[c*stride + i], amp[((r*H + h)*stride + i)*2 + {0:re,1:im}], weight[i] or NULL.
 *
 * Compiled twice: -DORACLE_LD gives REAL = long double (x87 80-bit; the parity reference), the
 * default gives REAL = double with Neumaier-compensated sums (the timed CPU baseline).  Events are
 * taken in storage order; with OpenMP each thread sums a contiguous block and the blocks are added
 * in thread order.
 *
 * Pins (tests/test_oracle_pins.py): Richardson central finite differences of the NLL and of the
 * gradient in 80-bit arithmetic, global-phase and common-scale invariance, the closed-form |BW|^2
 * integral, a Hermitian-form evaluation of the MC term through a library matmul, special cases,
 * weight linearity and shard additivity.  Parity against a value printed in the paper: unpinned
 * (the paper's only printed likelihood value, -lnL = -4110 at PAPER.md:131, needs its own sample).
 */
#include <complex.h>
#undef I /* the intensity is called I below; the imaginary unit is IU */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORACLE_LD
#define REAL long double
#define FN(name) name##_ld
#define R_LOG logl
#define R_COS cosl
#define R_SIN sinl
#define R_FABS fabsl
#define C_RE creall
#define C_IM cimagl
#define C_CONJ conjl
#else
#define REAL double
#define FN(name) name##_d
#define R_LOG log
#define R_COS cos
#define R_SIN sin
#define R_FABS fabs
#define C_RE creal
#define C_IM cimag
#define C_CONJ conj
#endif
typedef REAL _Complex CPLX;
#define MKC(re, im) ((CPLX)((REAL)(re) + (REAL)(im) * (CPLX)_Complex_I))
#define IU MKC(0, 1)

#define ORACLE_MAX_RES 512
#define ORACLE_MAX_HEL 16

/* running sum: plain in long double, Neumaier-compensated in double */
typedef struct { REAL s, c; } acc_t;
static inline void acc_add(acc_t *a, REAL x) {
#ifdef ORACLE_LD
  a->s += x;
#else
  REAL t = a->s + x;
  if (R_FABS(a->s) >= R_FABS(x)) a->c += (a->s - t) + x; else a->c += (x - t) + a->s;
  a->s = t;
#endif
}
static inline REAL acc_get(const acc_t *a) { return a->s + a->c; }

typedef struct {
  int R, H, C;
  const int32_t *res_chan;
  int64_t stride;              /* events between consecutive planes of mass / amp */
  const double *mass, *amp, *weight;
} sample_t;

/* Everything the likelihood needs from one event.  g and hv have 4R entries; hv only if v != NULL. */
typedef struct { REAL I, Idot; } event_scalars;

static event_scalars event_terms(const sample_t *s, int64_t i, const REAL *theta, const REAL *v,
                                 REAL *g, REAL *hv) {
  const int R = s->R, H = s->H;
  CPLX z[ORACLE_MAX_RES], dz[ORACLE_MAX_RES][4], A[ORACLE_MAX_HEL], S[ORACLE_MAX_RES];
  CPLX Bv[ORACLE_MAX_RES], ev[ORACLE_MAX_RES];
  event_scalars out = {0, 0};

  /* propagators and the four first derivatives of z_r */
  for (int r = 0; r < R; ++r) {
    REAL a = theta[4 * r], phi = theta[4 * r + 1], M = theta[4 * r + 2], G = theta[4 * r + 3];
    REAL m = s->mass[(int64_t)s->res_chan[r] * s->stride + i];
    CPLX D = MKC(M * M - m * m, -M * G);
    CPLX B = (REAL)1 / D;
    CPLX e = MKC(R_COS(phi), R_SIN(phi));
    CPLX DM = MKC(2 * M, -G);                  /* dD/dM;  dD/dGamma = -iM */
    z[r] = a * e * B;
    dz[r][0] = e * B;                          /* dz/da     */
    dz[r][1] = IU * z[r];                      /* dz/dphi   */
    dz[r][2] = -z[r] * B * DM;                 /* dz/dM     */
    dz[r][3] = IU * M * z[r] * B;              /* dz/dGamma */
    Bv[r] = B; ev[r] = e;
  }
#define F(r, h) MKC(s->amp[(((int64_t)(r) * H + (h)) * s->stride + i) * 2], \
                    s->amp[(((int64_t)(r) * H + (h)) * s->stride + i) * 2 + 1])
  /* coherent sum over resonances, incoherent sum over helicities (Eq. 1) */
  for (int h = 0; h < H; ++h) {
    A[h] = 0;
    for (int r = 0; r < R; ++r) A[h] += z[r] * F(r, h);
    out.I += C_RE(A[h]) * C_RE(A[h]) + C_IM(A[h]) * C_IM(A[h]);
  }
  /* g_(r,k) = dI/dtheta_(r,k) = 2 Re( dz_r/dtheta_k * S_r ),  S_r = sum_h conj(A_h) F_rh */
  for (int r = 0; r < R; ++r) {
    S[r] = 0;
    for (int h = 0; h < H; ++h) S[r] += C_CONJ(A[h]) * F(r, h);
    for (int k = 0; k < 4; ++k) g[4 * r + k] = 2 * C_RE(dz[r][k] * S[r]);
  }
  if (!v) return out;

  /* directional derivative along v: zdot_r, Adot_h, Idot = g.v, Sdot_r */
  CPLX Adot[ORACLE_MAX_HEL];
  for (int h = 0; h < H; ++h) Adot[h] = 0;
  for (int r = 0; r < R; ++r) {
    CPLX zdot = 0;
    for (int k = 0; k < 4; ++k) zdot += (REAL)v[4 * r + k] * dz[r][k];
    for (int h = 0; h < H; ++h) Adot[h] += zdot * F(r, h);
  }
  for (int h = 0; h < H; ++h) out.Idot += 2 * C_RE(C_CONJ(A[h]) * Adot[h]);
  for (int r = 0; r < R; ++r) {
    REAL M = theta[4 * r + 2], G = theta[4 * r + 3];
    CPLX B = Bv[r], e = ev[r], zz = z[r], DM = MKC(2 * M, -G);
    /* the ten second derivatives of z = a e^{i phi} B */
    CPLX z_aa = 0, z_ap = IU * e * B, z_aM = -e * B * B * DM, z_aG = IU * M * e * B * B;
    CPLX z_pp = -zz, z_pM = -IU * zz * B * DM, z_pG = -M * zz * B;
    CPLX z_MM = zz * (2 * B * B * DM * DM - 2 * B);
    CPLX z_MG = zz * (-2 * IU * M * B * B * DM + IU * B);
    CPLX z_GG = -2 * M * M * zz * B * B;
    REAL va = v[4 * r], vp = v[4 * r + 1], vM = v[4 * r + 2], vG = v[4 * r + 3];
    CPLX w[4];
    w[0] = z_aa * va + z_ap * vp + z_aM * vM + z_aG * vG;
    w[1] = z_ap * va + z_pp * vp + z_pM * vM + z_pG * vG;
    w[2] = z_aM * va + z_pM * vp + z_MM * vM + z_MG * vG;
    w[3] = z_aG * va + z_pG * vp + z_MG * vM + z_GG * vG;
    CPLX Sdot = 0;
    for (int h = 0; h < H; ++h) Sdot += C_CONJ(Adot[h]) * F(r, h);
    for (int k = 0; k < 4; ++k) hv[4 * r + k] = 2 * C_RE(dz[r][k] * Sdot) + 2 * C_RE(w[k] * S[r]);
  }
#undef F
  return out;
}

/*
 * Raw sums of one shard of one sample (F_m, G_m, their first derivatives and HVPs).
 *   is_data = 1:  scal[0] = sum w ln I   scal[1] = sum w      gsum = sum w g/I    hsum = sum w [ g Idot/I^2 - (H v)/I ]
 *   is_data = 0:  scal[0] = sum I        scal[1] = count      gsum = sum g        hsum = sum H v
 * Events first..first+count-1.  v may be NULL (then hsum is not written).  Returns 0, or 1 on bad sizes.
 */
int FN(oracle_raw_sums)(int n_res, int n_hel, int n_chan, const int32_t *res_chan, int64_t stride,
                        const double *mass, const double *amp, const double *weight, int64_t first,
                        int64_t count, int is_data, const REAL *theta, const REAL *v, REAL *scal,
                        REAL *gsum, REAL *hsum, int n_threads) {
  if (n_res < 1 || n_res > ORACLE_MAX_RES || n_hel < 1 || n_hel > ORACLE_MAX_HEL || n_chan < 1) return 1;
  const int P = 4 * n_res;
  sample_t s = {n_res, n_hel, n_chan, res_chan, stride, mass, amp, weight};
  if (n_threads < 1) n_threads = 1;
#ifndef _OPENMP
  n_threads = 1;
#endif
  const int NA = 2 + 2 * P;
  acc_t *acc = (acc_t *)calloc((size_t)n_threads * NA, sizeof(acc_t));
  if (!acc) return 1;
#pragma omp parallel num_threads(n_threads)
  {
    int t = 0, nt = 1;
#ifdef _OPENMP
    t = omp_get_thread_num(); nt = omp_get_num_threads();
#endif
    acc_t *a = acc + (size_t)t * NA;
    REAL *g = (REAL *)malloc(sizeof(REAL) * 2 * P), *hv = g + P;
    int64_t lo = first + count * t / nt, hi = first + count * (t + 1) / nt;
    for (int64_t i = lo; i < hi; ++i) {
      event_scalars e = event_terms(&s, i, theta, v, g, hv);
      if (is_data) {
        REAL w = weight ? (REAL)weight[i] : (REAL)1;
        acc_add(&a[0], w * R_LOG(e.I));
        acc_add(&a[1], w);
        for (int k = 0; k < P; ++k) acc_add(&a[2 + k], w * g[k] / e.I);
        if (v) for (int k = 0; k < P; ++k) acc_add(&a[2 + P + k], w * (g[k] * e.Idot / (e.I * e.I) - hv[k] / e.I));
      } else {
        acc_add(&a[0], e.I);
        acc_add(&a[1], 1);
        for (int k = 0; k < P; ++k) acc_add(&a[2 + k], g[k]);
        if (v) for (int k = 0; k < P; ++k) acc_add(&a[2 + P + k], hv[k]);
      }
    }
    free(g);
  }
  for (int j = 0; j < NA; ++j) {
    acc_t tot = {0, 0};
    for (int t = 0; t < n_threads; ++t) acc_add(&tot, acc_get(&acc[(size_t)t * NA + j]));
    REAL val = acc_get(&tot);
    if (j < 2) scal[j] = val;
    else if (j < 2 + P) gsum[j - 2] = val;
    else if (v) hsum[j - 2 - P] = val;
  }
  free(acc);
  return 0;
}

/*
 * Eqs. 4, 6, 7 with the sign of NLL = -lnL:
 *   NLL  = -Ld + W ln(G / N_mc)
 *   grad = -gd + W gG / G
 *   Hv   =  hd + W [ hG / G - gG (gG . v) / G^2 ]          (middle term of Eq. 7 read as in S9)
 * Inputs are the raw sums added over all shards (scal_data = {Ld, W}, scal_mc = {G, N_mc}).
 * v, hd, hG, hv may be NULL together.
 */
void FN(oracle_combine)(int n_par, const REAL *scal_data, const REAL *scal_mc, const REAL *gd,
                        const REAL *gG, const REAL *hd, const REAL *hG, const REAL *v,
                        REAL *nll, REAL *grad, REAL *hv) {
  const REAL Ld = scal_data[0], W = scal_data[1], G = scal_mc[0], n_mc = scal_mc[1];
  *nll = -Ld + W * R_LOG(G / n_mc);
  for (int k = 0; k < n_par; ++k) grad[k] = -gd[k] + W * gG[k] / G;
  if (!v) return;
  REAL dot = 0;
  for (int k = 0; k < n_par; ++k) dot += gG[k] * v[k];
  for (int k = 0; k < n_par; ++k) hv[k] = hd[k] + W * (hG[k] / G - gG[k] * dot / (G * G));
}

/* I_i for events first..first+count-1 (used for sampled-output checks at sizes the sums cannot cover) */
int FN(oracle_intensity)(int n_res, int n_hel, int n_chan, const int32_t *res_chan, int64_t stride,
                         const double *mass, const double *amp, int64_t first, int64_t count,
                         const REAL *theta, double *out) {
  if (n_res < 1 || n_res > ORACLE_MAX_RES || n_hel < 1 || n_hel > ORACLE_MAX_HEL || n_chan < 1) return 1;
  sample_t s = {n_res, n_hel, n_chan, res_chan, stride, mass, amp, NULL};
  REAL *g = (REAL *)malloc(sizeof(REAL) * 8 * n_res);
  for (int64_t i = 0; i < count; ++i) out[i] = (double)event_terms(&s, first + i, theta, NULL, g, g).I;
  free(g);
  return 0;
}

/* I_i, g_i . v, g_i (4R) and H_i v (4R) of ONE event - the per-event quantities of SURVEY.md §8(c) */
int FN(oracle_event)(int n_res, int n_hel, int n_chan, const int32_t *res_chan, int64_t stride,
                     const double *mass, const double *amp, int64_t i, const REAL *theta,
                     const REAL *v, REAL *I, REAL *Idot, REAL *g, REAL *hv) {
  if (n_res < 1 || n_res > ORACLE_MAX_RES || n_hel < 1 || n_hel > ORACLE_MAX_HEL || n_chan < 1) return 1;
  sample_t s = {n_res, n_hel, n_chan, res_chan, stride, mass, amp, NULL};
  REAL *gg = (REAL *)malloc(sizeof(REAL) * 8 * n_res), *hh = gg + 4 * n_res;
  event_scalars e = event_terms(&s, i, theta, v, gg, hh);
  *I = e.I; *Idot = e.Idot;
  for (int k = 0; k < 4 * n_res; ++k) { g[k] = gg[k]; if (v) hv[k] = hh[k]; }
  free(gg);
  return 0;
}

int FN(oracle_max_threads)(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
