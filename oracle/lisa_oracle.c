/*
 * oracle/lisa_oracle.c -- CPU ORACLE. TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, obviously-correct evaluation of the per-likelihood hot path of
 * arXiv:2501.08261 ("GPU-accelerated LISA parameter estimation with full time
 * domain response"), written from the paper's equations and from the
 * readings A1..A22 listed in DESIGN.md / SURVEY.md section 8(c).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or constant generator with the CUDA library under
 * paper_2501_08261_b200/csrc, and neither side includes the other.
 *
 * Precision: compiled twice from this one source,
 *     -DORC_REAL_LD  : REAL = long double (x86 80-bit) -> the parity truth
 *     (default)      : REAL = double                   -> the timed CPU baseline
 * Array arguments at the ABI are always double; all arithmetic is in REAL.
 *
 * No blocking, fusion or reordering beyond what the equations state: every
 * stage is a loop over samples that evaluates the printed formula.  OpenMP is
 * used only to spread independent output samples over host cores.
 *
 * Parity pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   S1  orc_modes_to_pol   : l=2 closed-form spin-weighted harmonics, orthonormality
 *                            by quadrature, beta=0 twist, per-l norm, and an
 *                            independent numpy restatement of Eq. 2.4-2.6
 *   O-I orc_delay_read     : exact on polynomials of degree <= p, partition of unity
 *   S2  orc_link_response  : analytic transfer function on a static triangle (C1)
 *   S3  orc_tdi            : exact laser-noise cancellation on integer delays (C2),
 *                            X2 = X1.5 - delayed X1.5 (C3), cyclic symmetry (C4),
 *                            monochromatic closed form (C5), brute-force term tables
 *                            read from tests/golden/
 *   S4  orc_fft_r2c        : naive DFT, numpy.fft, Parseval (C9)
 *   S5  orc_loglike        : closed forms log L(h=d), log L(lambda d), log L(0) (C10)
 *   orbit                  : arm-length and Kepler invariants, independent numpy forms
 *   PSD orc_psd_weights    : Eq. 2.15 = the transfer of uncorrelated link / test-mass noises through
 *                            orc_tdi on static equal arms (sums of squared responses, both
 *                            generations), Eq. 2.14 at its printed knees and in its power-law limits,
 *                            zeros of the generation-2 factor (tests/test_oracle_psd_transfer.py)
 *   C12 second path        : S2 and S3 re-evaluated with absolute-time delays and Neville's recursion
 *                            in numpy long double, agreement 2e-15 (tests/test_oracle_second_path.py)
 *   C11 laser residual     : first-order residual sum_terms s Ldot_l D pdot(t - D - L_l) of un-nested
 *                            TDI on breathing arms, its low-frequency limit and the X2/X1.5 ratio
 *                            2 omega (L2+L-2+L3+L-3) (tests/test_oracle_laser_residual.py)
 *   orc_laser_links        : identical to orc_laser_links3 with one laser, and the definition read by
 *                            orc_delay_read (same file)
 *   orbit TABLE (A21)      : exact on polynomial trajectories, KEPLER1 table vs KEPLER1 closed form
 *   UP  orc_upsample2      : exact on linear series, identity on even samples, closed-form
 *                            midpoint error of a quadratic
 *   F1  orc_fisher         : linear-model closed form via Parseval (time-domain Gram matrix),
 *                            symmetry, step independence, Hessian of orc_loglike
 *   A22 tt_order / nested  : velocity = d/dt position, first-order travel time vs the fixed point of
 *                            c L = |r_r(t) - r_s(t - L)|, chained delay vs the light path traced
 *                            leg by leg, nested == summed on a static constellation, and
 *                            three-laser cancellation on flexing arms (chained X2 at the 1e-13
 *                            floor, chained X1.5 and summed X2 at 1e-8)
 * No function is "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <tgmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORC_REAL_LD
typedef long double REAL;
#define RC(x) x##L
#else
typedef double REAL;
#define RC(x) x
#endif

#define ORC_PI RC(3.14159265358979323846264338327950288419716939937510)
#define ORC_C_LIGHT RC(299792458.0) /* m/s */

typedef struct {
  REAL re, im;
} cplx;

static cplx c_make(REAL re, REAL im) {
  cplx z = {re, im};
  return z;
}
static cplx c_add(cplx a, cplx b) { return c_make(a.re + b.re, a.im + b.im); }
static cplx c_mul(cplx a, cplx b) {
  return c_make(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
static cplx c_conj(cplx a) { return c_make(a.re, -a.im); }
static cplx c_scale(cplx a, REAL s) { return c_make(a.re * s, a.im * s); }
static cplx c_expi(REAL x) { return c_make(cos(x), sin(x)); }

/* Orbit description.  Declared independently of include/lisa_td.h on purpose. */
typedef struct {
  int kind; /* 0 = STATIC, 1 = KEPLER1 (reading A8), 2 = TABLE (reading A21) */
  double L_m, a_m, year_s, phase0, t_ref;
  double r_static[3][3]; /* metres, [spacecraft][xyz] */
  double L_static[6];    /* seconds, link order [1,2,3,-1,-2,-3] */
  /* TABLE: positions tabulated at t_tab0 + j dt_tab, j = 0..n_tab-1 */
  int n_tab, tab_order;  /* tab_order odd: tab_order + 1 interpolation nodes */
  double t_tab0, dt_tab;
  const double* r_tab;   /* [n_tab][3][3] metres */
  /* Delay model (reading A22 of DESIGN.md).
   * tt_order 0: L_l(t) = |r_r(t) - r_s(t)| / c (reading A8).
   * tt_order 1: first order in v/c of  c L = |r_r(t) - r_s(t - L)|:
   *             L_l(t) = (d/c) (1 + n.v_s/c),  d = |r_r - r_s|, n = (r_r - r_s)/d, v_s = sender
   *             velocity, all at the reception time t (so L_l != L_{-l}).  STATIC ignores it.
   * nested 0: TDI delays are sums of L_l(t), all at the output time (reading A10).
   * nested 1: TDI delays are chained along the light path traced back from the output time:
   *           tau_0 = 0, tau_{i+1} = tau_i + L_{l_i}(t - tau_i). */
  int tt_order, nested;
} orc_orbit;

/* Link order l = [1,2,3,-1,-2,-3]; (sender, receiver) spacecraft, 1-based
 * (PAPER.md:132 notation y_{slr}; labels of Eq. 2.9 at PAPER.md:165). */
static const int LINK_S[6] = {3, 1, 2, 2, 3, 1};
static const int LINK_R[6] = {2, 3, 1, 3, 1, 2};

int orc_sizeof_real(void) { return (int)sizeof(REAL); }
int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------ S1 -- */

static REAL factorial(int n) {
  REAL f = 1;
  for (int i = 2; i <= n; ++i) f *= (REAL)i;
  return f;
}

/* Wigner small-d, z-y-z convention, Wigner's factorial sum:
 * d^l_{m'm}(b) = sum_k (-1)^{k-m+m'} sqrt((l+m)!(l-m)!(l+m')!(l-m')!)
 *   / ((l+m-k)! k! (l-k-m')! (k-m+m')!) cos(b/2)^{2l-2k+m-m'} sin(b/2)^{2k-m+m'} */
static REAL wigner_small_d(int l, int mp, int m, REAL beta) {
  REAL cb = cos(beta / 2), sb = sin(beta / 2);
  REAL pref = sqrt(factorial(l + m) * factorial(l - m) * factorial(l + mp) * factorial(l - mp));
  REAL sum = 0;
  for (int k = 0; k <= 2 * l; ++k) {
    int a = l + m - k, b = l - k - mp, c = k - m + mp;
    if (a < 0 || b < 0 || c < 0) continue;
    REAL term = pref / (factorial(a) * factorial(k) * factorial(b) * factorial(c));
    term *= pow(cb, (REAL)(2 * l - 2 * k + m - mp)) * pow(sb, (REAL)(2 * k - m + mp));
    if ((k - m + mp) & 1) term = -term;
    sum += term;
  }
  return sum;
}

/* Reading A2: frakD^l_{m'm}(a,b,g) = e^{+i m' a} d^l_{m'm}(b) e^{+i m g}. */
static cplx wigner_D(int l, int mp, int m, REAL a, REAL b, REAL g) {
  return c_scale(c_expi((REAL)mp * a + (REAL)m * g), wigner_small_d(l, mp, m, b));
}

void orc_wigner_small_d(int l, int mp, int m, double beta, double* out) {
  *out = (double)wigner_small_d(l, mp, m, (REAL)beta);
}

/* _{-2}Y_{lm}(iota,phi) = sqrt((2l+1)/4pi) d^l_{m,2}(iota) e^{i m phi}  (A2; PAPER.md:74 fn.1) */
static cplx swsh_m2(int l, int m, REAL iota, REAL phi) {
  REAL norm = sqrt((REAL)(2 * l + 1) / (4 * ORC_PI));
  return c_scale(c_expi((REAL)m * phi), norm * wigner_small_d(l, m, 2, iota));
}

void orc_swsh(int l, int m, double iota, double phi, double* re, double* im) {
  cplx y = swsh_m2(l, m, (REAL)iota, (REAL)phi);
  *re = (double)y.re;
  *im = (double)y.im;
}

#define ORC_LMAX 8
#define ORC_NM (2 * ORC_LMAX + 1)

/* One sample of Eq. 2.1-2.3 with readings A1, A2, A6.
 * amp/phase: the n_modes listed co-precessing modes at this sample. */
static void s1_sample(int n_modes, const int* l, const int* m, const REAL* amp, const REAL* phase,
                      int twisted, REAL alpha, REAL beta, REAL gamma, int have_e0, REAL a0,
                      REAL b0, REAL g0, REAL iota, REAL phi, REAL psi, REAL* hplus, REAL* hcross) {
  cplx H = c_make(0, 0);
  for (int ll = 2; ll <= ORC_LMAX; ++ll) {
    /* co-precessing modes of this l, index m + ll */
    cplx hcp[ORC_NM], hj[ORC_NM], hl0[ORC_NM];
    int any = 0;
    for (int i = 0; i < ORC_NM; ++i) hcp[i] = c_make(0, 0);
    for (int k = 0; k < n_modes; ++k) {
      if (l[k] != ll) continue;
      any = 1;
      /* A6: h_lm = amp e^{-i phase};  h_{l,-m} = (-1)^l conj(h_lm) */
      cplx h = c_scale(c_expi(-phase[k]), amp[k]);
      hcp[m[k] + ll] = c_add(hcp[m[k] + ll], h);
      if (m[k] != 0) {
        cplx hm = c_conj(h);
        if (ll & 1) hm = c_scale(hm, -1);
        hcp[-m[k] + ll] = c_add(hcp[-m[k] + ll], hm);
      }
    }
    if (!any) continue;
    /* Eq. 2.1 (A1: sum over the first index): h^J_{lm} = sum_{m'} frakD^l_{m'm}(a,b,g) h^CP_{lm'} */
    for (int mm = -ll; mm <= ll; ++mm) {
      if (twisted) {
        cplx s = c_make(0, 0);
        for (int mp = -ll; mp <= ll; ++mp)
          s = c_add(s, c_mul(wigner_D(ll, mp, mm, alpha, beta, gamma), hcp[mp + ll]));
        hj[mm + ll] = s;
      } else {
        hj[mm + ll] = hcp[mm + ll];
      }
    }
    /* Eq. 2.2: constant rotation J -> L0 */
    for (int mm = -ll; mm <= ll; ++mm) {
      if (have_e0) {
        cplx s = c_make(0, 0);
        for (int mp = -ll; mp <= ll; ++mp)
          s = c_add(s, c_mul(wigner_D(ll, mp, mm, a0, b0, g0), hj[mp + ll]));
        hl0[mm + ll] = s;
      } else {
        hl0[mm + ll] = hj[mm + ll];
      }
    }
    /* Eq. 2.3 */
    for (int mm = -ll; mm <= ll; ++mm) H = c_add(H, c_mul(hl0[mm + ll], swsh_m2(ll, mm, iota, phi)));
  }
  /* multiply h+ - i hx by e^{i 2 psi} */
  H = c_mul(H, c_expi(2 * psi));
  *hplus = H.re;
  *hcross = -H.im;
}

/* REAL-array core: writes hp/hc[b*N + n] for n in [n_lo, n_hi). */
static void s1_core(int B, long N, int n_modes, const int* l, const int* m, const double* amp,
                    const double* phase, const double* alpha, const double* beta,
                    const double* gamma, const double* iota, const double* phi, const double* psi,
                    const double* euler0, long n_lo, long n_hi, REAL* hp, REAL* hc) {
  int twisted = (alpha != NULL);
  for (int b = 0; b < B; ++b) {
#pragma omp parallel for schedule(static)
    for (long n = n_lo; n < n_hi; ++n) {
      REAL a[32], p[32];
      for (int k = 0; k < n_modes; ++k) {
        a[k] = (REAL)amp[((size_t)b * n_modes + k) * N + n];
        p[k] = (REAL)phase[((size_t)b * n_modes + k) * N + n];
      }
      REAL al = 0, be = 0, ga = 0;
      if (twisted) {
        al = (REAL)alpha[(size_t)b * N + n];
        be = (REAL)beta[(size_t)b * N + n];
        ga = (REAL)gamma[(size_t)b * N + n];
      }
      REAL a0 = 0, b0 = 0, g0 = 0;
      if (euler0) {
        a0 = (REAL)euler0[3 * b + 0];
        b0 = (REAL)euler0[3 * b + 1];
        g0 = (REAL)euler0[3 * b + 2];
      }
      s1_sample(n_modes, l, m, a, p, twisted, al, be, ga, euler0 != NULL, a0, b0, g0,
                (REAL)iota[b], (REAL)phi[b], (REAL)psi[b], &hp[(size_t)b * N + n],
                &hc[(size_t)b * N + n]);
    }
  }
}

static int s1_args_ok(int B, long N, int n_modes, const int* l, const int* m) {
  if (B <= 0 || N <= 0 || n_modes <= 0 || n_modes > 32) return 0;
  for (int k = 0; k < n_modes; ++k)
    if (l[k] < 2 || l[k] > ORC_LMAX || m[k] < -l[k] || m[k] > l[k]) return 0;
  return 1;
}

int orc_modes_to_pol(int B, long N, int n_modes, const int* l, const int* m, const double* amp,
                     const double* phase, const double* alpha, const double* beta,
                     const double* gamma, const double* iota, const double* phi,
                     const double* psi, const double* euler0, long n_lo, long n_hi,
                     double* hplus, double* hcross) {
  if (!s1_args_ok(B, N, n_modes, l, m) || n_lo < 0 || n_hi > N) return -1;
  REAL* hp = (REAL*)calloc((size_t)B * N, sizeof(REAL));
  REAL* hc = (REAL*)calloc((size_t)B * N, sizeof(REAL));
  if (!hp || !hc) return -3;
  s1_core(B, N, n_modes, l, m, amp, phase, alpha, beta, gamma, iota, phi, psi, euler0, n_lo, n_hi,
          hp, hc);
  for (int b = 0; b < B; ++b)
    for (long n = n_lo; n < n_hi; ++n) {
      hplus[(size_t)b * N + n] = (double)hp[(size_t)b * N + n];
      hcross[(size_t)b * N + n] = (double)hc[(size_t)b * N + n];
    }
  free(hp);
  free(hc);
  return 0;
}

/* --------------------------------------------------------------- orbits -- */

/* Positions r[3][3] (metres) and velocities v[3][3] (m/s) at time t.
 * STATIC: as given, at rest.  KEPLER1: reading A8 (first-order solution of Kepler's equation)
 * and its time derivative.  TABLE: reading A21 and the derivative of the interpolant. */
static void orbit_state(const orc_orbit* o, REAL t, REAL r[3][3], REAL v[3][3]) {
  if (o->kind == 0) {
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        r[i][j] = (REAL)o->r_static[i][j];
        v[i][j] = 0;
      }
    return;
  }
  if (o->kind == 2) {
    /* TABLE (orbits "tracked over the whole observation period", ESA-style file;
     * reading A21): Lagrange interpolation of degree q = tab_order on the q+1 nodes
     * j0 .. j0+q,  j0 = floor(u) - (q-1)/2 clamped to [0, n_tab-q-1],  u = (t - t_tab0)/dt_tab.
     * Velocity = d/dt of the same polynomial:  c_i'(x) = sum_{k != i} [prod_{m != i,k} (x - m)] /
     * prod_{m != i} (i - m), divided by dt_tab. */
    int q = o->tab_order;
    REAL u = (t - (REAL)o->t_tab0) / (REAL)o->dt_tab;
    long j0 = (long)floor(u) - (q - 1) / 2;
    if (j0 < 0) j0 = 0;
    if (j0 > o->n_tab - q - 1) j0 = o->n_tab - q - 1;
    REAL x = u - (REAL)j0;
    for (int k = 0; k < 3; ++k)
      for (int j = 0; j < 3; ++j) r[k][j] = v[k][j] = 0;
    for (int i = 0; i <= q; ++i) {
      REAL c = 1, den = 1, dc = 0;
      for (int m = 0; m <= q; ++m)
        if (m != i) {
          c *= (x - (REAL)m) / (REAL)(i - m);
          den *= (REAL)(i - m);
        }
      for (int k = 0; k <= q; ++k) {
        if (k == i) continue;
        REAL pr = 1;
        for (int m = 0; m <= q; ++m)
          if (m != i && m != k) pr *= x - (REAL)m;
        dc += pr;
      }
      dc /= den * (REAL)o->dt_tab;
      for (int k = 0; k < 3; ++k)
        for (int j = 0; j < 3; ++j) {
          REAL rij = (REAL)o->r_tab[((size_t)(j0 + i) * 3 + k) * 3 + j];
          r[k][j] += c * rij;
          v[k][j] += dc * rij;
        }
    }
    return;
  }
  REAL a = (REAL)o->a_m;
  REAL delta = (REAL)o->L_m / (2 * a);
  REAL sq3 = sqrt((REAL)3);
  REAL e = sqrt(1 + 2 * delta / sq3 + 4 * delta * delta / 3) - 1;
  REAL inc = atan(delta / (1 + delta / sq3));
  REAL ci = cos(inc), si = sin(inc);
  REAL w = 2 * ORC_PI / (REAL)o->year_s; /* dM/dt */
  for (int k = 0; k < 3; ++k) {
    REAL sigma = 2 * ORC_PI * (REAL)k / 3;
    REAL M = 2 * ORC_PI * (t - (REAL)o->t_ref) / (REAL)o->year_s - sigma - (REAL)o->phase0;
    REAL psi = M + e * sin(M);
    REAL dpsi = w * (1 + e * cos(M)); /* d psi / dt */
    REAL x = a * (cos(psi) - e) * ci;
    REAL y = a * sqrt(1 - e * e) * sin(psi);
    REAL z = a * (cos(psi) - e) * si;
    REAL vx = -a * sin(psi) * dpsi * ci;
    REAL vy = a * sqrt(1 - e * e) * cos(psi) * dpsi;
    REAL vz = -a * sin(psi) * dpsi * si;
    REAL cs = cos(sigma), ss = sin(sigma);
    r[k][0] = cs * x - ss * y;
    r[k][1] = ss * x + cs * y;
    r[k][2] = z;
    v[k][0] = cs * vx - ss * vy;
    v[k][1] = ss * vx + cs * vy;
    v[k][2] = vz;
  }
}

/* Positions r[3][3] (metres) and light travel times L[6] (seconds, link order) at time t.
 * STATIC: as given.  Otherwise L_l = d/c (tt_order 0, reading A8) or (d/c)(1 + n.v_s/c)
 * (tt_order 1, reading A22), d = |r_r - r_s|, n from sender to receiver. */
static void orbit_eval(const orc_orbit* o, REAL t, REAL r[3][3], REAL L[6]) {
  REAL v[3][3];
  orbit_state(o, t, r, v);
  if (o->kind == 0) {
    for (int k = 0; k < 6; ++k) L[k] = (REAL)o->L_static[k];
    return;
  }
  for (int k = 0; k < 6; ++k) {
    const REAL* rs = r[LINK_S[k] - 1];
    const REAL* rr = r[LINK_R[k] - 1];
    const REAL* vs = v[LINK_S[k] - 1];
    REAL d0 = rr[0] - rs[0], d1 = rr[1] - rs[1], d2 = rr[2] - rs[2];
    REAL d = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
    L[k] = d / ORC_C_LIGHT;
    if (o->tt_order == 1) {
      REAL nv = (d0 * vs[0] + d1 * vs[1] + d2 * vs[2]) / d;
      L[k] = (d / ORC_C_LIGHT) * (1 + nv / ORC_C_LIGHT);
    }
  }
}

void orc_orbit_state(const orc_orbit* o, double t, double* r9, double* v9) {
  REAL r[3][3], v[3][3];
  orbit_state(o, (REAL)t, r, v);
  for (int i = 0; i < 9; ++i) {
    r9[i] = (double)r[i / 3][i % 3];
    v9[i] = (double)v[i / 3][i % 3];
  }
}

/* Chained delay (seconds) of the signed link labels lab[0..n) applied in this order, starting
 * at time t (reading A22):  tau_0 = 0,  tau_{i+1} = tau_i + L_{lab_i}(t - tau_i). */
static int link_index(int link);
static REAL nested_delay(const orc_orbit* o, REAL t, const int* lab, int n) {
  REAL tau = 0;
  for (int i = 0; i < n; ++i) {
    REAL r[3][3], L[6];
    orbit_eval(o, t - tau, r, L);
    tau += L[link_index(lab[i])];
  }
  return tau;
}
double orc_nested_delay(const orc_orbit* o, double t, const int* lab, int n) {
  return (double)nested_delay(o, (REAL)t, lab, n);
}

void orc_orbit_eval(const orc_orbit* o, double t, double* r9, double* L6) {
  REAL r[3][3], L[6];
  orbit_eval(o, (REAL)t, r, L);
  for (int i = 0; i < 9; ++i) r9[i] = (double)r[i / 3][i % 3];
  for (int k = 0; k < 6; ++k) L6[k] = (double)L[k];
}

/* ------------------------------------------------------------------ O-I -- */

/* Lagrange coefficients, literal O(p^2) product:
 * taps j = -h+1 .. h, h = (p+1)/2,  c_j(eps) = prod_{i != j} (eps - i)/(j - i).  out[j + h - 1]. */
static void lagrange_coeffs(int order, REAL eps, REAL* c) {
  int h = (order + 1) / 2;
  for (int j = -h + 1; j <= h; ++j) {
    REAL v = 1;
    for (int i = -h + 1; i <= h; ++i)
      if (i != j) v *= (eps - (REAL)i) / (REAL)(j - i);
    c[j + h - 1] = v;
  }
}

void orc_lagrange_coeffs(int order, double eps, double* c) {
  REAL cc[64];
  lagrange_coeffs(order, (REAL)eps, cc);
  for (int i = 0; i <= order; ++i) c[i] = (double)cc[i];
}

/* Fractional-delay read x(n - D): K = ceil(D), eps = K - D in [0,1), base b = n - K,
 * value = sum_j c_j(eps) x[b + j], x = 0 outside [0,N).  D = 0 returns x[n] itself. */
static REAL delay_read(const REAL* x, long N, long n, REAL D, int order) {
  REAL Kf = ceil(D);
  REAL eps = Kf - D;
  long b = n - (long)Kf;
  if (eps == 0) return (b >= 0 && b < N) ? x[b] : 0;
  int h = (order + 1) / 2;
  REAL c[64];
  lagrange_coeffs(order, eps, c);
  REAL s = 0;
  for (int j = -h + 1; j <= h; ++j) {
    long idx = b + j;
    if (idx >= 0 && idx < N) s += c[j + h - 1] * x[idx];
  }
  return s;
}

double orc_delay_read(const double* x, long N, long n, double D, int order) {
  REAL* xr = (REAL*)malloc((size_t)N * sizeof(REAL));
  for (long i = 0; i < N; ++i) xr[i] = (REAL)x[i];
  REAL v = delay_read(xr, N, n, (REAL)D, order);
  free(xr);
  return (double)v;
}

/* ------------------------------------------------------------------ S2 -- */

/* 10 s -> 5 s (the waveforms are sampled "every Delta t = 10 s and then linearly
 * interpolate[d] ... to generate the arm and TDI responses with a sampling time of 5 s"; reading
 * A20 of DESIGN.md).  Coarse series c[0..Nc), Nc = N/2 + 1, on t0 + i (2 dt); fine series on
 * t0 + n dt:  x[2i] = c[i],  x[2i+1] = (c[i] + c[i+1]) / 2. */
int orc_upsample2(int B, long N, const double* coarse, double* fine) {
  if (B <= 0 || N < 2 || (N & 1)) return -1;
  long Nc = N / 2 + 1;
  for (int b = 0; b < B; ++b)
    for (long n = 0; n < N; ++n) {
      const double* c = coarse + (size_t)b * Nc;
      REAL v = (n & 1) ? ((REAL)c[n / 2] + (REAL)c[n / 2 + 1]) / 2 : (REAL)c[n / 2];
      fine[(size_t)b * N + n] = (double)v;
    }
  return 0;
}

static REAL dot3(const REAL* a, const REAL* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* Eq. 2.7-2.8 with readings A7, A11 and P3 (delays in samples).
 * hp/hc: [B][N] REAL; y: [B][6][N] REAL; writes n in [n_lo,n_hi); zero outside [margin, N-margin). */
static void s2_core(int B, long N, REAL t0, REAL dt, int order, long margin, const REAL* hp,
                    const REAL* hc, const double* lambda, const double* beta_sky,
                    const orc_orbit* orbit, long n_lo, long n_hi, REAL* y) {
  for (int b = 0; b < B; ++b) {
    REAL lam = (REAL)lambda[b], bet = (REAL)beta_sky[b];
    /* Eq. 2.7 */
    REAL k[3] = {-cos(bet) * cos(lam), -cos(bet) * sin(lam), -sin(bet)};
    REAL v[3] = {-sin(bet) * cos(lam), -sin(bet) * sin(lam), cos(bet)};
    REAL u[3] = {sin(lam), -cos(lam), 0};
    const REAL* hpb = hp + (size_t)b * N;
    const REAL* hcb = hc + (size_t)b * N;
#pragma omp parallel for schedule(static)
    for (long n = n_lo; n < n_hi; ++n) {
      REAL* yb = y + (size_t)b * 6 * N;
      if (n < margin || n >= N - margin) {
        for (int l = 0; l < 6; ++l) yb[(size_t)l * N + n] = 0;
        continue;
      }
      REAL t = t0 + (REAL)n * dt;
      REAL r[3][3], L[6];
      orbit_eval(orbit, t, r, L);
      for (int l = 0; l < 6; ++l) {
        const REAL* rs = r[LINK_S[l] - 1];
        const REAL* rr = r[LINK_R[l] - 1];
        REAL d[3] = {rr[0] - rs[0], rr[1] - rs[1], rr[2] - rs[2]};
        REAL dn = sqrt(dot3(d, d));
        REAL nh[3] = {d[0] / dn, d[1] / dn, d[2] / dn};
        REAL un = dot3(u, nh), vn = dot3(v, nh), kn = dot3(k, nh);
        REAL xp = un * un - vn * vn;
        REAL xc = un * vn;
        /* t_s = t - L_l - k.r_s/c ; t_r = t - k.r_r/c, expressed as delays in samples */
        REAL Ds = (L[l] + dot3(k, rs) / ORC_C_LIGHT) / dt;
        REAL Dr = (dot3(k, rr) / ORC_C_LIGHT) / dt;
        REAL dhp = delay_read(hpb, N, n, Ds, order) - delay_read(hpb, N, n, Dr, order);
        REAL dhc = delay_read(hcb, N, n, Ds, order) - delay_read(hcb, N, n, Dr, order);
        /* A11: standard projection (1/2) n.h.n */
        yb[(size_t)l * N + n] = (xp * dhp + 2 * xc * dhc) / (2 * (1 - kn));
      }
    }
  }
}

int orc_link_response(int B, long N, double t0, double dt, int order, long margin,
                      const double* hplus, const double* hcross, const double* lambda,
                      const double* beta_sky, const orc_orbit* orbit, long n_lo, long n_hi,
                      double* y) {
  if (B <= 0 || N <= 0 || order < 1 || order > 63 || !(order & 1) || n_lo < 0 || n_hi > N)
    return -1;
  size_t tot = (size_t)B * N;
  REAL* hp = (REAL*)malloc(tot * sizeof(REAL));
  REAL* hc = (REAL*)malloc(tot * sizeof(REAL));
  REAL* yy = (REAL*)calloc(tot * 6, sizeof(REAL));
  if (!hp || !hc || !yy) return -3;
  for (size_t i = 0; i < tot; ++i) {
    hp[i] = (REAL)hplus[i];
    hc[i] = (REAL)hcross[i];
  }
  s2_core(B, N, (REAL)t0, (REAL)dt, order, margin, hp, hc, lambda, beta_sky, orbit, n_lo, n_hi, yy);
  for (int b = 0; b < B; ++b)
    for (int l = 0; l < 6; ++l)
      for (long n = n_lo; n < n_hi; ++n) {
        size_t i = ((size_t)b * 6 + l) * N + n;
        y[i] = (double)yy[i];
      }
  free(hp);
  free(hc);
  free(yy);
  return 0;
}

/* Reading A12: common laser noise injected at link level,
 * y_l[n] = p(n - L_l(t_n)/dt) - p[n]; zero outside [margin, N-margin). y: [6][N]. */
int orc_laser_links(long N, double t0, double dt, int order, long margin, const double* p,
                    const orc_orbit* orbit, double* y) {
  REAL* pr = (REAL*)malloc((size_t)N * sizeof(REAL));
  if (!pr) return -3;
  for (long i = 0; i < N; ++i) pr[i] = (REAL)p[i];
#pragma omp parallel for schedule(static)
  for (long n = 0; n < N; ++n) {
    if (n < margin || n >= N - margin) {
      for (int l = 0; l < 6; ++l) y[(size_t)l * N + n] = 0;
      continue;
    }
    REAL r[3][3], L[6];
    orbit_eval(orbit, (REAL)t0 + (REAL)n * (REAL)dt, r, L);
    for (int l = 0; l < 6; ++l)
      y[(size_t)l * N + n] = (double)(delay_read(pr, N, n, L[l] / (REAL)dt, order) - pr[n]);
  }
  free(pr);
  return 0;
}

/* Three independent lasers, one per spacecraft (used to pin the chaining order of A22):
 * y_{slr}[n] = p_s(n - L_l(t_n)/dt) - p_r[n]; p: [3][N]; zero outside [margin, N-margin). */
int orc_laser_links3(long N, double t0, double dt, int order, long margin, const double* p,
                     const orc_orbit* orbit, double* y) {
  REAL* pr = (REAL*)malloc((size_t)3 * N * sizeof(REAL));
  if (!pr) return -3;
  for (long i = 0; i < 3 * N; ++i) pr[i] = (REAL)p[i];
#pragma omp parallel for schedule(static)
  for (long n = 0; n < N; ++n) {
    if (n < margin || n >= N - margin) {
      for (int l = 0; l < 6; ++l) y[(size_t)l * N + n] = 0;
      continue;
    }
    REAL r[3][3], L[6];
    orbit_eval(orbit, (REAL)t0 + (REAL)n * (REAL)dt, r, L);
    for (int l = 0; l < 6; ++l)
      y[(size_t)l * N + n] = (double)(delay_read(pr + (size_t)(LINK_S[l] - 1) * N, N, n, L[l] / (REAL)dt, order) -
                                      pr[(size_t)(LINK_R[l] - 1) * N + n]);
  }
  free(pr);
  return 0;
}

/* ------------------------------------------------------------------ S3 -- */

/* Term tables for the Michelson X.  Links are signed labels
 * +-1..3; delays are multisets of signed link labels, terminated by 0.
 * X1.5: Eq. 2.9 as printed.
 * X2  : Eq. 2.10 with the y123 block corrected (reading A9). */
typedef struct {
  int sign, link;
  int delays[8];
} tdi_term;

static const tdi_term X15_TERMS[8] = {
    {+1, -3, {3, 2, -2, 0}}, {-1, -3, {3, 0}},          {+1, 3, {2, -2, 0}}, {-1, 3, {0}},
    {+1, 2, {-2, 0}},        {-1, 2, {-2, -3, 3, 0}},   {+1, -2, {0}},       {-1, -2, {-3, 3, 0}},
};

static const tdi_term X20_TERMS[16] = {
    {+1, -3, {3, 2, -2, 0}},
    {-1, -3, {3, 0}},
    {+1, -3, {-2, 2, 3, 3, -3, 0}},
    {-1, -3, {3, 3, -3, -2, -2, 2, 2, 0}},
    {+1, 3, {2, -2, 0}},
    {-1, 3, {0}},
    {+1, 3, {-2, 2, 3, -3, 0}},
    {-1, 3, {3, -3, -2, -2, 2, 2, 0}},
    {+1, 2, {-2, 0}},
    {-1, 2, {-2, -3, 3, 0}},
    {+1, 2, {-2, -2, 2, 3, 3, -3, -3, 0}},
    {-1, 2, {3, -3, -2, -2, 2, 0}},
    {+1, -2, {0}},
    {-1, -2, {-3, 3, 0}},
    {+1, -2, {-2, 2, 3, 3, -3, -3, 0}},
    {-1, -2, {3, -3, -2, 2, 0}},
};

/* The same terms with the delay labels in CHAINING order (reading A22): the label nearest to the
 * output time first.  X compares the two light paths that leave spacecraft 1, visit 2 and 3 in
 * opposite orders (twice each for generation 2) and return to 1.  Traced BACK from the output time
 * t at spacecraft 1, link by link (link l is received at LINK_R[l], so stepping back along it
 * lands on LINK_S[l]), the two paths are
 *     path A: 3, -3, -2, 2, -2, 2, 3, -3      (1 <- 2 <- 1 <- 3 <- 1 <- 3 <- 1 <- 2 <- 1)
 *     path B: -2, 2, 3, -3, 3, -3, -2, 2      (1 <- 3 <- 1 <- 2 <- 1 <- 2 <- 1 <- 3 <- 1)
 * and every delay of Eq. 2.9 / 2.10 is, as a multiset, a leading piece of one of them, applied to
 * the link measured at the spacecraft that piece ends on.  Written out term by term: */
static const tdi_term X15_NESTED[8] = {
    {+1, -3, {-2, 2, 3, 0}}, {-1, -3, {3, 0}},          {+1, 3, {-2, 2, 0}}, {-1, 3, {0}},
    {+1, 2, {-2, 0}},        {-1, 2, {3, -3, -2, 0}},   {+1, -2, {0}},       {-1, -2, {3, -3, 0}},
};
static const tdi_term X20_NESTED[16] = {
    {+1, -3, {-2, 2, 3, 0}},
    {-1, -3, {3, 0}},
    {+1, -3, {-2, 2, 3, -3, 3, 0}},
    {-1, -3, {3, -3, -2, 2, -2, 2, 3, 0}},
    {+1, 3, {-2, 2, 0}},
    {-1, 3, {0}},
    {+1, 3, {-2, 2, 3, -3, 0}},
    {-1, 3, {3, -3, -2, 2, -2, 2, 0}},
    {+1, 2, {-2, 0}},
    {-1, 2, {3, -3, -2, 0}},
    {+1, 2, {-2, 2, 3, -3, 3, -3, -2, 0}},
    {-1, 2, {3, -3, -2, 2, -2, 0}},
    {+1, -2, {0}},
    {-1, -2, {3, -3, 0}},
    {+1, -2, {-2, 2, 3, -3, 3, -3, 0}},
    {-1, -2, {3, -3, -2, 2, 0}},
};

/* cyclic relabelling 1->2->3->1 of |link|, sign kept */
static int cyc(int link, int times) {
  int s = link < 0 ? -1 : 1, a = link < 0 ? -link : link;
  for (int i = 0; i < times; ++i) a = a % 3 + 1;
  return s * a;
}
static int link_index(int link) { return link > 0 ? link - 1 : -link + 2; }

/* y: [B][6][N] REAL -> tdi: [B][3][N] REAL, XYZ (out_kind 0) or AET (1).
 * generation 15 or 20.  All L at the output time t, delays summed not nested (A10), unless
 * orbit->nested (A22).
 * Outputs are zero outside [margin_lo, N - margin_hi). */
static void s3_core(int B, long N, REAL t0, REAL dt, int order, int generation, int out_kind,
                    long margin_lo, long margin_hi, const REAL* y, const orc_orbit* orbit,
                    long n_lo, long n_hi, REAL* tdi) {
  const tdi_term* terms = generation == 15 ? X15_TERMS : X20_TERMS;
  if (orbit->nested) terms = generation == 15 ? X15_NESTED : X20_NESTED;
  int n_terms = generation == 15 ? 8 : 16;
  for (int b = 0; b < B; ++b) {
    const REAL* yb = y + (size_t)b * 6 * N;
    REAL* ob = tdi + (size_t)b * 3 * N;
#pragma omp parallel for schedule(static)
    for (long n = n_lo; n < n_hi; ++n) {
      if (n < margin_lo || n >= N - margin_hi) {
        for (int c = 0; c < 3; ++c) ob[(size_t)c * N + n] = 0;
        continue;
      }
      REAL r[3][3], L[6];
      orbit_eval(orbit, t0 + (REAL)n * dt, r, L);
      REAL xyz[3];
      for (int c = 0; c < 3; ++c) { /* X, Y, Z by 0, 1, 2 cyclic permutations */
        REAL acc = 0;
        for (int k = 0; k < n_terms; ++k) {
          REAL D = 0;
          if (orbit->nested) { /* A22: chained along the light path */
            int lab[8], nl = 0;
            for (int q = 0; terms[k].delays[q] != 0; ++q) lab[nl++] = cyc(terms[k].delays[q], c);
            D = nested_delay(orbit, t0 + (REAL)n * dt, lab, nl);
          } else { /* A10: summed, every L at the output time */
            for (int q = 0; terms[k].delays[q] != 0; ++q)
              D += L[link_index(cyc(terms[k].delays[q], c))];
          }
          D /= dt;
          const REAL* series = yb + (size_t)link_index(cyc(terms[k].link, c)) * N;
          acc += (REAL)terms[k].sign * delay_read(series, N, n, D, order);
        }
        xyz[c] = acc;
      }
      if (out_kind == 0) {
        for (int c = 0; c < 3; ++c) ob[(size_t)c * N + n] = xyz[c];
      } else { /* Eq. 2.11 */
        ob[(size_t)0 * N + n] = (xyz[2] - xyz[0]) / sqrt((REAL)2);
        ob[(size_t)1 * N + n] = (xyz[0] - 2 * xyz[1] + xyz[2]) / sqrt((REAL)6);
        ob[(size_t)2 * N + n] = (xyz[0] + xyz[1] + xyz[2]) / sqrt((REAL)3);
      }
    }
  }
}

int orc_tdi(int B, long N, double t0, double dt, int order, int generation, int out_kind,
            long margin_lo, long margin_hi, const double* y, const orc_orbit* orbit, long n_lo,
            long n_hi, double* tdi) {
  if (B <= 0 || N <= 0 || order < 1 || order > 63 || !(order & 1) ||
      (generation != 15 && generation != 20) || n_lo < 0 || n_hi > N)
    return -1;
  size_t tot = (size_t)B * 6 * N;
  REAL* yy = (REAL*)malloc(tot * sizeof(REAL));
  REAL* tt = (REAL*)calloc((size_t)B * 3 * N, sizeof(REAL));
  if (!yy || !tt) return -3;
  for (size_t i = 0; i < tot; ++i) yy[i] = (REAL)y[i];
  s3_core(B, N, (REAL)t0, (REAL)dt, order, generation, out_kind, margin_lo, margin_hi, yy, orbit,
          n_lo, n_hi, tt);
  for (int b = 0; b < B; ++b)
    for (int c = 0; c < 3; ++c)
      for (long n = n_lo; n < n_hi; ++n) {
        size_t i = ((size_t)b * 3 + c) * N + n;
        tdi[i] = (double)tt[i];
      }
  free(yy);
  free(tt);
  return 0;
}

/* ------------------------------------------------------------- S4 / S5 -- */

/* Radix-2 decimation-in-time FFT, in place, forward sign e^{-2 pi i k n / N}. */
static int fft_pow2(cplx* a, long N) {
  if (N <= 0 || (N & (N - 1))) return -1;
  for (long i = 1, j = 0; i < N; ++i) {
    long bit = N >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) {
      cplx t = a[i];
      a[i] = a[j];
      a[j] = t;
    }
  }
  for (long len = 2; len <= N; len <<= 1) {
    long half = len >> 1;
#pragma omp parallel for schedule(static) if (N >= 65536)
    for (long i = 0; i < N / 2; ++i) { /* butterfly i of this stage */
      long blk = i / half, k = i % half;
      cplx* p = a + blk * len;
      cplx w = c_expi(-2 * ORC_PI * (REAL)k / (REAL)len);
      cplx x = p[k], z = c_mul(w, p[k + half]);
      p[k] = c_add(x, z);
      p[k + half] = c_make(x.re - z.re, x.im - z.im);
    }
  }
  return 0;
}

/* H[k] = sum_n x[n] e^{-2 pi i k n / N}, k = 0..N/2.  spec: REAL cplx [N/2+1]. */
static int fft_r2c_core(long N, const REAL* x, cplx* spec) {
  cplx* a = (cplx*)malloc((size_t)N * sizeof(cplx));
  if (!a) return -3;
  for (long i = 0; i < N; ++i) a[i] = c_make(x[i], 0);
  int rc = fft_pow2(a, N);
  if (rc == 0)
    for (long k = 0; k <= N / 2; ++k) spec[k] = a[k];
  free(a);
  return rc;
}

int orc_fft_r2c(long N, const double* x, double* spec /* [N/2+1][2] */) {
  REAL* xr = (REAL*)malloc((size_t)N * sizeof(REAL));
  cplx* s = (cplx*)malloc((size_t)(N / 2 + 1) * sizeof(cplx));
  if (!xr || !s) return -3;
  for (long i = 0; i < N; ++i) xr[i] = (REAL)x[i];
  int rc = fft_r2c_core(N, xr, s);
  if (rc == 0)
    for (long k = 0; k <= N / 2; ++k) {
      spec[2 * k] = (double)s[k].re;
      spec[2 * k + 1] = (double)s[k].im;
    }
  free(xr);
  free(s);
  return rc;
}

/* The definition itself, O(N^2); cross-check of the FFT at small N (C9). */
int orc_dft_naive(long N, const double* x, double* spec) {
  for (long k = 0; k <= N / 2; ++k) {
    cplx s = c_make(0, 0);
    for (long n = 0; n < N; ++n) {
      /* reduce k*n mod N in integers so the phase stays accurate */
      long kn = (long)(((unsigned long long)k * (unsigned long long)n) % (unsigned long long)N);
      s = c_add(s, c_scale(c_expi(-2 * ORC_PI * (REAL)kn / (REAL)N), (REAL)x[n]));
    }
    spec[2 * k] = (double)s.re;
    spec[2 * k + 1] = (double)s.im;
  }
  return 0;
}

/* Eq. 2.12-2.13 with readings A13, A17:
 * log L = sum_c sum_{k=kmin}^{kmax} w_c[k] ( Re(D_c[k] conj(H_c[k])) - |H_c[k]|^2 / 2 ).
 * spec: [3][N/2+1] REAL cplx for one walker.  Also returns (d|h) and (h|h). */
static void loglike_core(long nf, const cplx* spec, const double* data_spec, const double* weight,
                         long kmin, long kmax, REAL* ll, REAL* dh, REAL* hh) {
  REAL sdh = 0, shh = 0;
  for (int c = 0; c < 3; ++c)
    for (long k = kmin; k <= kmax; ++k) {
      cplx H = spec[(size_t)c * nf + k];
      REAL dre = (REAL)data_spec[2 * ((size_t)c * nf + k)];
      REAL dim = (REAL)data_spec[2 * ((size_t)c * nf + k) + 1];
      REAL w = (REAL)weight[(size_t)c * nf + k];
      sdh += w * (dre * H.re + dim * H.im);
      shh += w * (H.re * H.re + H.im * H.im);
    }
  *dh = sdh;
  *hh = shh;
  *ll = sdh - shh / 2;
}

/* tdi: [B][3][N] (A,E,T) -> loglike[B] (+ optional dh[B], hh[B]); N a power of two. */
int orc_loglike(int B, long N, const double* tdi, const double* data_spec, const double* weight,
                long kmin, long kmax, double* loglike, double* dh, double* hh) {
  long nf = N / 2 + 1;
  if (B <= 0 || kmin < 0 || kmin > kmax || kmax > N / 2) return -1;
  REAL* x = (REAL*)malloc((size_t)N * sizeof(REAL));
  cplx* spec = (cplx*)malloc((size_t)3 * nf * sizeof(cplx));
  if (!x || !spec) return -3;
  int rc = 0;
  for (int b = 0; b < B && rc == 0; ++b) {
    for (int c = 0; c < 3 && rc == 0; ++c) {
      for (long n = 0; n < N; ++n) x[n] = (REAL)tdi[((size_t)b * 3 + c) * N + n];
      rc = fft_r2c_core(N, x, spec + (size_t)c * nf);
    }
    if (rc) break;
    REAL ll, sdh, shh;
    loglike_core(nf, spec, data_spec, weight, kmin, kmax, &ll, &sdh, &shh);
    loglike[b] = (double)ll;
    if (dh) dh[b] = (double)sdh;
    if (hh) hh[b] = (double)shh;
  }
  free(x);
  free(spec);
  return rc;
}

/* Fisher matrix by first-order finite differences ("The Fisher matrix is computed
 * from the derivatives of the likelihood function, using first-order finite differences";
 * reading A19 of DESIGN.md).  Walker 0 is the centre theta, walker i = 1..D is
 * theta + delta_i e_i.  With the forward difference  d_i h = (h_i - h_0) / delta_i  taken on the
 * Fourier transforms of the three channels,
 *   Gamma_ij = (d_i h | d_j h) = sum_c sum_{k=kmin}^{kmax} w_c[k] Re( d_i H_c[k] conj(d_j H_c[k]) ),
 * the same inner product as Eq. 2.13 (weights of A17).  tdi: [D+1][3][N]; fisher: [D][D]. */
int orc_fisher(int D, long N, const double* tdi, const double* delta, const double* weight, long kmin,
               long kmax, double* fisher) {
  long nf = N / 2 + 1;
  if (D <= 0 || kmin < 0 || kmin > kmax || kmax > N / 2) return -1;
  for (int i = 0; i < D; ++i)
    if (delta[i] == 0.0) return -1;
  REAL* x = (REAL*)malloc((size_t)N * sizeof(REAL));
  cplx* spec = (cplx*)malloc((size_t)(D + 1) * 3 * nf * sizeof(cplx));
  if (!x || !spec) return -3;
  int rc = 0;
  for (int b = 0; b <= D && rc == 0; ++b)
    for (int c = 0; c < 3 && rc == 0; ++c) {
      for (long n = 0; n < N; ++n) x[n] = (REAL)tdi[((size_t)b * 3 + c) * N + n];
      rc = fft_r2c_core(N, x, spec + ((size_t)b * 3 + c) * nf);
    }
  for (int i = 0; i < D && rc == 0; ++i)
    for (int j = 0; j < D; ++j) {
      REAL sum = 0;
      for (int c = 0; c < 3; ++c)
        for (long k = kmin; k <= kmax; ++k) {
          cplx h0 = spec[(size_t)c * nf + k];
          cplx hi = spec[((size_t)(i + 1) * 3 + c) * nf + k];
          cplx hj = spec[((size_t)(j + 1) * 3 + c) * nf + k];
          REAL dire = (hi.re - h0.re) / (REAL)delta[i], diim = (hi.im - h0.im) / (REAL)delta[i];
          REAL djre = (hj.re - h0.re) / (REAL)delta[j], djim = (hj.im - h0.im) / (REAL)delta[j];
          sum += (REAL)weight[(size_t)c * nf + k] * (dire * djre + diim * djim);
        }
      fisher[(size_t)i * D + j] = (double)sum;
    }
  free(x);
  free(spec);
  return rc;
}

/* Eq. 2.14-2.15 with readings A14, A15, A17:
 * w_c[k] = 4 df dt^2 / S_c(k df), df = 1/(N dt); w = 0 at k = 0.
 * generation 20 multiplies S by 4 sin^2(2x), x = 2 pi f L/c.  weight: [3][N/2+1] (A,E,T). */
int orc_psd_weights(long N, double dt, double acc_noise, double oms_noise, double arm_s,
                    int generation, double* weight) {
  long nf = N / 2 + 1;
  REAL df = 1 / ((REAL)N * (REAL)dt);
  for (long k = 0; k < nf; ++k) {
    if (k == 0) {
      for (int c = 0; c < 3; ++c) weight[(size_t)c * nf] = 0;
      continue;
    }
    REAL f = (REAL)k * df;
    REAL w2 = 2 * ORC_PI * f;
    REAL s_acc = (REAL)acc_noise * (REAL)acc_noise * (1 + (RC(4e-4) / f) * (RC(4e-4) / f)) *
                 (1 + pow(f / RC(0.008), (REAL)4)) / (w2 * w2 * w2 * w2) * (w2 / ORC_C_LIGHT) *
                 (w2 / ORC_C_LIGHT);
    REAL s_op = (REAL)oms_noise * (REAL)oms_noise * (1 + pow(RC(0.002) / f, (REAL)4)) *
                (w2 / ORC_C_LIGHT) * (w2 / ORC_C_LIGHT);
    REAL x = w2 * (REAL)arm_s;
    REAL sx = sin(x), cx = cos(x);
    REAL s_ae = 8 * sx * sx * (2 * s_acc * (3 + 2 * cx + cos(2 * x)) + s_op * (2 + cx));
    REAL sh = sin(x / 2);
    REAL s_t = 16 * s_op * (1 - cx) * sx * sx + 128 * s_acc * sx * sx * sh * sh * sh * sh;
    if (generation == 20) {
      REAL g = 4 * sin(2 * x) * sin(2 * x);
      s_ae *= g;
      s_t *= g;
    }
    REAL num = 4 * df * (REAL)dt * (REAL)dt;
    weight[(size_t)0 * nf + k] = (double)(num / s_ae);
    weight[(size_t)1 * nf + k] = (double)(num / s_ae);
    weight[(size_t)2 * nf + k] = (double)(num / s_t);
  }
  return 0;
}

/* ---------------------------------------------------------------- chain -- */

/* S1 -> S2 -> S3 (-> S4/S5) for walkers one at a time, REAL carried between
 * stages (no rounding to double in between).  TDI is produced for n in
 * [n_lo, n_hi) only; the link responses and polarisations are evaluated on the
 * index ranges those outputs can reach (the margins bound the stencil reach).
 * tdi_out: [B][3][N] or NULL.  If loglike != NULL the range must be [0,N) and
 * N a power of two.  y_out ([B][6][N]) and hp_out/hc_out ([B][N]) optional. */
int orc_chain(int B, long N, int n_modes, const int* l, const int* m, const double* amp,
              const double* phase, const double* alpha, const double* beta, const double* gamma,
              const double* iota, const double* phi, const double* psi, const double* euler0,
              double t0, double dt, int order, const double* lambda, const double* beta_sky,
              const orc_orbit* orbit, long margin_y, int generation, int out_kind,
              long margin_lo, long margin_hi, long n_lo, long n_hi, double* hp_out,
              double* hc_out, double* y_out, double* tdi_out, const double* data_spec,
              const double* weight, long kmin, long kmax, double* loglike, double* dh, double* hh) {
  if (!s1_args_ok(B, N, n_modes, l, m) || n_lo < 0 || n_hi > N || n_lo > n_hi) return -1;
  if (order < 1 || order > 63 || !(order & 1)) return -1;
  if (generation != 15 && generation != 20) return -1;
  if (loglike && (n_lo != 0 || n_hi != N)) return -1;
  long nf = N / 2 + 1;
  REAL* hp = (REAL*)calloc((size_t)N, sizeof(REAL));
  REAL* hc = (REAL*)calloc((size_t)N, sizeof(REAL));
  REAL* y = (REAL*)calloc((size_t)6 * N, sizeof(REAL));
  REAL* tdi = (REAL*)calloc((size_t)3 * N, sizeof(REAL));
  cplx* spec = loglike ? (cplx*)malloc((size_t)3 * nf * sizeof(cplx)) : NULL;
  if (!hp || !hc || !y || !tdi || (loglike && !spec)) return -3;
  /* index ranges reached by the requested outputs */
  long y_lo = n_lo - margin_lo, y_hi = n_hi + margin_hi;
  if (y_lo < 0) y_lo = 0;
  if (y_hi > N) y_hi = N;
  long h_lo = y_lo - margin_y, h_hi = y_hi + margin_y;
  if (h_lo < 0) h_lo = 0;
  if (h_hi > N) h_hi = N;
  int rc = 0;
  for (int b = 0; b < B && rc == 0; ++b) {
    const double* al = alpha ? alpha + (size_t)b * N : NULL;
    const double* be = alpha ? beta + (size_t)b * N : NULL;
    const double* ga = alpha ? gamma + (size_t)b * N : NULL;
    s1_core(1, N, n_modes, l, m, amp + (size_t)b * n_modes * N, phase + (size_t)b * n_modes * N,
            al, be, ga, iota + b, phi + b, psi + b, euler0 ? euler0 + 3 * b : NULL, h_lo, h_hi, hp,
            hc);
    s2_core(1, N, (REAL)t0, (REAL)dt, order, margin_y, hp, hc, lambda + b, beta_sky + b, orbit,
            y_lo, y_hi, y);
    s3_core(1, N, (REAL)t0, (REAL)dt, order, generation, out_kind, margin_lo, margin_hi, y, orbit,
            n_lo, n_hi, tdi);
    if (hp_out)
      for (long n = h_lo; n < h_hi; ++n) {
        hp_out[(size_t)b * N + n] = (double)hp[n];
        hc_out[(size_t)b * N + n] = (double)hc[n];
      }
    if (y_out)
      for (int k = 0; k < 6; ++k)
        for (long n = y_lo; n < y_hi; ++n)
          y_out[((size_t)b * 6 + k) * N + n] = (double)y[(size_t)k * N + n];
    if (tdi_out)
      for (int c = 0; c < 3; ++c)
        for (long n = n_lo; n < n_hi; ++n)
          tdi_out[((size_t)b * 3 + c) * N + n] = (double)tdi[(size_t)c * N + n];
    if (loglike) {
      for (int c = 0; c < 3 && rc == 0; ++c)
        rc = fft_r2c_core(N, tdi + (size_t)c * N, spec + (size_t)c * nf);
      if (rc) break;
      REAL ll, sdh, shh;
      loglike_core(nf, spec, data_spec, weight, kmin, kmax, &ll, &sdh, &shh);
      loglike[b] = (double)ll;
      if (dh) dh[b] = (double)sdh;
      if (hh) hh[b] = (double)shh;
    }
  }
  free(hp);
  free(hc);
  free(y);
  free(tdi);
  free(spec);
  return rc;
}

/* Spectrum of a [3][N] TDI triple in REAL, returned as double [3][N/2+1][2]
 * (used to build the zero-noise injection data of config 4, fn. 4). */
int orc_spectrum3(long N, const double* tdi, double* spec_out) {
  long nf = N / 2 + 1;
  int rc = 0;
  for (int c = 0; c < 3 && rc == 0; ++c) rc = orc_fft_r2c(N, tdi + (size_t)c * N, spec_out + 2 * (size_t)c * nf);
  return rc;
}
