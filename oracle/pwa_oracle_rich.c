/*
 * pwa_oracle_rich.c - plain, slow CPU reference for the RICHER amplitude model.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as pwa_oracle.c, which stays as it is and keeps pinning the
 * base model).  It shares no code with the CUDA path and neither includes the other.
 *
 * The model (readings S21, S22; the paper prints Eq. 1 and no lineshape formula):
 *   partial waves m = 0 .. W-1, each with its own complex coupling Lambda_m = a_m e^{i phi_m} and pre-computed
 *   projections U_m^mu = F_mh(i) (PAPER.md:57-60, Eq. 1: A^mu = sum_m Lambda_m U_m^mu; :70 U pre-computed);
 *   every wave belongs to one RESONANCE l = ls[m] whose lineshape BW_l(m_i) = 1 / D_l(m_i) it shares with the other
 *   partial waves of that resonance ("one [template] for calculating the amplitude of a single
 *   intermediate resonance"; :102 "phase angles and couplings of individual partial wave amplitudes" against one
 *   mass and width per resonance in Table 1):
 *       A_h(i) = sum_m a_m e^{i phi_m} F_mh(i) / D_{ls[m]}(i),      I_i = sum_h |A_h(i)|^2.
 *   Lineshape kinds (S22), m = mass[ch[l]][i], parameters (M, Gamma) per resonance:
 *     0  constant width          D = M^2 - m^2 - i M Gamma                                  (BASELINE.json configs[0])
 *     1  mass-dependent width    D = M^2 - m^2 - i M Gamma(m),  Gamma(m) = Gamma (q(m)/q(M))^(2L+1) M/m,
 *                                q(m) = sqrt((m^2 - (m1+m2)^2)(m^2 - (m1-m2)^2)) / (2m)   two-body break-up momentum,
 *                                sp = (m1, m2, L); no barrier factors; needs M, m > m1 + m2
 *     2  Flatte (refs [28], [29], quoted for the f0(980))
 *                                D = M^2 - m^2 - i Gamma (rho_1(m) + Rg rho_2(m)),  rho_k = 2 q_k(m)/m for the two
 *                                channels (m1, m2) and (m3, m4); below a threshold q_k -> i |q_k| (analytic
 *                                continuation); "Gamma" is the coupling g_1, Rg = g_2/g_1 is fixed; sp = (m1, m2, m3, m4, Rg)
 * Parameters (S21): theta = [a_0, phi_0, ..., a_{W-1}, phi_{W-1}, M_0, Gamma_0, ..., M_{L-1}, Gamma_{L-1}],  P = 2W + 2L.
 * NLL, gradient and Hessian-vector product exactly as in pwa_oracle.c (PAPER.md:67 Eq. 3, :90 Eq. 6, :95 Eq. 7),
 * with the chain rule written out for shared lineshape parameters.
 *
 * Pins (tests/test_oracle_rich.py): one wave per resonance with kind 0 IS the base model (pwa_oracle.c, pinned by its
 * own closed forms); Richardson finite differences in 80-bit arithmetic for every kind and for shared resonances;
 * per-event equivalence of kinds 1 and 2 with a constant-width propagator at event-wise (M', Gamma') computed in the
 * test from the textbook q, rho formulas; phase / scale invariance; waves with identical projections add coherently.
 */
#include <complex.h>
#undef I
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
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
#define R_SQRT sqrtl
#define R_POW powl
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
#define R_SQRT sqrt
#define R_POW pow
#define C_RE creal
#define C_IM cimag
#define C_CONJ conj
#endif
typedef REAL _Complex CPLX;
#define MKC(re, im) ((CPLX)((REAL)(re) + (REAL)(im) * (CPLX)_Complex_I))
#define IU MKC(0, 1)
#define RICH_MAX_WAVE 512
#define RICH_MAX_HEL 16
#define RICH_SP 6 /* shape parameters per resonance */

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
  int W, L, H, C;
  const int32_t *ls;      /* [W] resonance of each wave */
  const int32_t *ch;      /* [L] mass channel of each resonance */
  const int32_t *kind;    /* [L] */
  const double *sp;       /* [L][RICH_SP] */
  int64_t stride;
  const double *mass, *amp, *weight;
} rsample_t;

/* squared break-up momentum q^2(s) of a two-body channel (m1, m2) at invariant mass squared s (may be negative) */
static REAL q2_of(REAL s, REAL m1, REAL m2) {
  return (s - (m1 + m2) * (m1 + m2)) * (s - (m1 - m2) * (m1 - m2)) / (4 * s);
}

/* D_l(m) and its derivatives with respect to (M, Gamma): D, D_M, D_G, D_MM, D_MG  (D_GG = 0 for every kind) */
static void lineshape(int kind, const double *sp, REAL M, REAL G, REAL m, CPLX d[5]) {
  if (kind == 0) {
    d[0] = MKC(M * M - m * m, -M * G);
    d[1] = MKC(2 * M, -G);
    d[2] = MKC(0, -M);
    d[3] = MKC(2, 0);
    d[4] = MKC(0, -1);
  } else if (kind == 1) {
    /* M Gamma(m) = Gamma chi(M) psi(m),  chi(M) = M^2 / q(M)^n,  psi(m) = q(m)^n / m,  n = 2L + 1 */
    const REAL m1 = sp[0], m2 = sp[1], n = 2 * (REAL)sp[2] + 1;
    const REAL psi = R_POW(R_SQRT(q2_of(m * m, m1, m2)), n) / m;
    const REAL u = M * M, sp_ = (m1 + m2) * (m1 + m2), sm_ = (m1 - m2) * (m1 - m2);
    const REAL p = q2_of(u, m1, m2);
    const REAL p1 = (REAL)0.25 - sp_ * sm_ / (4 * u * u);  /* d q^2 / du   */
    const REAL p2 = sp_ * sm_ / (2 * u * u * u);           /* d2 q^2 / du2 */
    const REAL pn = R_POW(p, -n / 2);
    const REAL f = u * pn;                                                    /* chi           */
    const REAL f1 = pn - (n / 2) * u * pn / p * p1;                           /* d chi / du    */
    const REAL f2 = -n * pn / p * p1 + (n / 2) * (n / 2 + 1) * u * pn / (p * p) * p1 * p1 - (n / 2) * u * pn / p * p2;
    const REAL chi = f, chi1 = 2 * M * f1, chi2 = 2 * f1 + 4 * u * f2;        /* d/dM, d2/dM2  */
    d[0] = MKC(M * M - m * m, -G * chi * psi);
    d[1] = MKC(2 * M, -G * chi1 * psi);
    d[2] = MKC(0, -chi * psi);
    d[3] = MKC(2, -G * chi2 * psi);
    d[4] = MKC(0, -chi1 * psi);
  } else {
    const REAL s = m * m;
    const REAL qa = q2_of(s, sp[0], sp[1]), qb = q2_of(s, sp[2], sp[3]), Rg = sp[4];
    const CPLX rho1 = qa >= 0 ? MKC(2 * R_SQRT(qa) / m, 0) : MKC(0, 2 * R_SQRT(-qa) / m);
    const CPLX rho2 = qb >= 0 ? MKC(2 * R_SQRT(qb) / m, 0) : MKC(0, 2 * R_SQRT(-qb) / m);
    const CPLX psi = rho1 + Rg * rho2;
    d[0] = MKC(M * M - m * m, 0) - IU * G * psi;
    d[1] = MKC(2 * M, 0);
    d[2] = -IU * psi;
    d[3] = MKC(2, 0);
    d[4] = 0;
  }
}

typedef struct { REAL I, Idot; } event_scalars;

/* Everything the likelihood needs from one event.  g and hv have P = 2W + 2L entries (zeroed here); hv only if v. */
static event_scalars event_terms(const rsample_t *s, int64_t i, const REAL *theta, const REAL *v, REAL *g, REAL *hv) {
  const int W = s->W, L = s->L, H = s->H, P = 2 * W + 2 * L;
  CPLX z[RICH_MAX_WAVE], dz[RICH_MAX_WAVE][4], A[RICH_MAX_HEL], S[RICH_MAX_WAVE];
  CPLX Bv[RICH_MAX_WAVE], ev[RICH_MAX_WAVE], dD[RICH_MAX_WAVE][5];
  int pidx[RICH_MAX_WAVE][4];
  event_scalars out = {0, 0};
  for (int k = 0; k < P; ++k) { g[k] = 0; if (v) hv[k] = 0; }

  /* propagators and the four first derivatives of z_m = a_m e^{i phi_m} / D_l,  l = ls[m] */
  for (int m = 0; m < W; ++m) {
    const int l = s->ls[m];
    pidx[m][0] = 2 * m; pidx[m][1] = 2 * m + 1; pidx[m][2] = 2 * W + 2 * l; pidx[m][3] = 2 * W + 2 * l + 1;
    REAL a = theta[pidx[m][0]], phi = theta[pidx[m][1]], M = theta[pidx[m][2]], G = theta[pidx[m][3]];
    REAL mass = s->mass[(int64_t)s->ch[l] * s->stride + i];
    lineshape(s->kind[l], s->sp + (size_t)l * RICH_SP, M, G, mass, dD[m]);
    CPLX B = (REAL)1 / dD[m][0];
    CPLX e = MKC(R_COS(phi), R_SIN(phi));
    z[m] = a * e * B;
    dz[m][0] = e * B;                    /* dz/da     */
    dz[m][1] = IU * z[m];                /* dz/dphi   */
    dz[m][2] = -z[m] * B * dD[m][1];     /* dz/dM     */
    dz[m][3] = -z[m] * B * dD[m][2];     /* dz/dGamma */
    Bv[m] = B; ev[m] = e;
  }
#define F(m, h) MKC(s->amp[(((int64_t)(m) * H + (h)) * s->stride + i) * 2], \
                    s->amp[(((int64_t)(m) * H + (h)) * s->stride + i) * 2 + 1])
  for (int h = 0; h < H; ++h) {
    A[h] = 0;
    for (int m = 0; m < W; ++m) A[h] += z[m] * F(m, h);
    out.I += C_RE(A[h]) * C_RE(A[h]) + C_IM(A[h]) * C_IM(A[h]);
  }
  /* dI/dtheta_p = sum over the waves that depend on p of 2 Re( dz_m/dtheta_p * S_m ),  S_m = sum_h conj(A_h) F_mh */
  for (int m = 0; m < W; ++m) {
    S[m] = 0;
    for (int h = 0; h < H; ++h) S[m] += C_CONJ(A[h]) * F(m, h);
    for (int k = 0; k < 4; ++k) g[pidx[m][k]] += 2 * C_RE(dz[m][k] * S[m]);
  }
  if (!v) return out;

  CPLX Adot[RICH_MAX_HEL];
  for (int h = 0; h < H; ++h) Adot[h] = 0;
  for (int m = 0; m < W; ++m) {
    CPLX zdot = 0;
    for (int k = 0; k < 4; ++k) zdot += (REAL)v[pidx[m][k]] * dz[m][k];
    for (int h = 0; h < H; ++h) Adot[h] += zdot * F(m, h);
  }
  for (int h = 0; h < H; ++h) out.Idot += 2 * C_RE(C_CONJ(A[h]) * Adot[h]);
  for (int m = 0; m < W; ++m) {
    CPLX B = Bv[m], e = ev[m], zz = z[m];
    CPLX DM = dD[m][1], DG = dD[m][2], DMM = dD[m][3], DMG = dD[m][4];
    /* the ten second derivatives of z = a e^{i phi} / D(M, Gamma) */
    CPLX z_aa = 0, z_ap = IU * e * B, z_aM = -e * B * B * DM, z_aG = -e * B * B * DG;
    CPLX z_pp = -zz, z_pM = -IU * zz * B * DM, z_pG = -IU * zz * B * DG;
    CPLX z_MM = zz * (2 * B * B * DM * DM - B * DMM);
    CPLX z_MG = zz * (2 * B * B * DM * DG - B * DMG);
    CPLX z_GG = zz * (2 * B * B * DG * DG);
    REAL va = v[pidx[m][0]], vp = v[pidx[m][1]], vM = v[pidx[m][2]], vG = v[pidx[m][3]];
    CPLX w[4];
    w[0] = z_aa * va + z_ap * vp + z_aM * vM + z_aG * vG;
    w[1] = z_ap * va + z_pp * vp + z_pM * vM + z_pG * vG;
    w[2] = z_aM * va + z_pM * vp + z_MM * vM + z_MG * vG;
    w[3] = z_aG * va + z_pG * vp + z_MG * vM + z_GG * vG;
    CPLX Sdot = 0;
    for (int h = 0; h < H; ++h) Sdot += C_CONJ(Adot[h]) * F(m, h);
    for (int k = 0; k < 4; ++k) hv[pidx[m][k]] += 2 * C_RE(dz[m][k] * Sdot) + 2 * C_RE(w[k] * S[m]);
  }
#undef F
  return out;
}

/* Raw sums of events first..first+count-1 of one sample; same meaning and layout as oracle_raw_sums (pwa_oracle.c). */
int FN(rich_raw_sums)(int n_wave, int n_ls, int n_hel, int n_chan, const int32_t *ls, const int32_t *ch,
                      const int32_t *kind, const double *sp, int64_t stride, const double *mass, const double *amp,
                      const double *weight, int64_t first, int64_t count, int is_data, const REAL *theta,
                      const REAL *v, REAL *scal, REAL *gsum, REAL *hsum, int n_threads) {
  if (n_wave < 1 || n_wave > RICH_MAX_WAVE || n_ls < 1 || n_ls > n_wave || n_hel < 1 || n_hel > RICH_MAX_HEL || n_chan < 1) return 1;
  const int P = 2 * n_wave + 2 * n_ls;
  rsample_t s = {n_wave, n_ls, n_hel, n_chan, ls, ch, kind, sp, stride, mass, amp, weight};
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

/* I_i for events first..first+count-1 */
int FN(rich_intensity)(int n_wave, int n_ls, int n_hel, int n_chan, const int32_t *ls, const int32_t *ch,
                       const int32_t *kind, const double *sp, int64_t stride, const double *mass, const double *amp,
                       int64_t first, int64_t count, const REAL *theta, double *out) {
  if (n_wave < 1 || n_wave > RICH_MAX_WAVE || n_ls < 1 || n_ls > n_wave || n_hel < 1 || n_hel > RICH_MAX_HEL || n_chan < 1) return 1;
  rsample_t s = {n_wave, n_ls, n_hel, n_chan, ls, ch, kind, sp, stride, mass, amp, NULL};
  REAL *g = (REAL *)malloc(sizeof(REAL) * 2 * (2 * n_wave + 2 * n_ls));
  for (int64_t i = 0; i < count; ++i) out[i] = (double)event_terms(&s, first + i, theta, NULL, g, g).I;
  free(g);
  return 0;
}
