// api.cu -- the extern "C" boundary of liblisa_td (include/lisa_td.h): argument validation,
// host-side preparation of the constant tables handed to the kernels, the end-to-end host
// pipeline and the DFMA probe.  No arithmetic of the method runs on the host; there is no
// CPU fallback.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "common.cuh"

namespace lisa {

// ------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";

int set_error(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
int check_cuda(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return LISA_TD_OK;
  return set_error(e == cudaErrorMemoryAllocation ? LISA_TD_ENOMEM : LISA_TD_ECUDA, "%s: %s (%s)", what,
                   cudaGetErrorString(e), cudaGetErrorName(e));
}

int sm_count() {
  static thread_local int cached_dev = -1, cached = 0;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 148;
  if (dev != cached_dev) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    cached_dev = dev;
    cached = n;
  }
  return cached;
}

// ------------------------------------------------------------------ sticky device-side errors
unsigned int* device_error_words() {
  static unsigned int* words = nullptr;
  static bool tried = false;
  if (!tried) {  // benign race: two first calls from two threads would leak 16 bytes of pinned memory
    tried = true;
    void* p = nullptr;
    if (cudaHostAlloc(&p, DEVERR_COUNT * sizeof(unsigned int), cudaHostAllocMapped | cudaHostAllocPortable) == cudaSuccess) {
      memset(p, 0, DEVERR_COUNT * sizeof(unsigned int));
      words = static_cast<unsigned int*>(p);
    } else {
      cudaGetLastError();
    }
  }
  return words;
}
// Call after a synchronisation: reports and clears what the kernels raised since the last check.
int take_device_errors(const char* fn) {
  volatile unsigned int* w = device_error_words();
  if (!w) return LISA_TD_OK;
  const unsigned k2 = w[DEVERR_K2_WINDOW], k3 = w[DEVERR_K3_WINDOW], la = w[DEVERR_LASER_WINDOW];
  if (!(k2 | k3 | la)) return LISA_TD_OK;
  w[DEVERR_K2_WINDOW] = w[DEVERR_K3_WINDOW] = w[DEVERR_LASER_WINDOW] = 0;
  return set_error(LISA_TD_EINVAL,
                   "%s: a kernel found a delay outside the range the host-side orbit bounds promised (%s%s%s): "
                   "the outputs written since the last check are invalid (orbit far from the bounds of its "
                   "description, e.g. a TABLE orbit whose arms or centroid move faster than its nodes suggest)",
                   fn, k2 ? "link-response strain window " : "", k3 ? "TDI stencil window " : "",
                   la ? "laser-link window" : "");
}

// Test-only dispatch switch, read from the environment at every call (NOT part of the ABI):
// LISA_TD_DISPATCH=1 routes S1/S2/S3 through the generic (any mode list, runtime-order, unmerged)
// kernels even where a specialised instantiation exists, 2 keeps the specialised kernels but
// routes the five-mode S1 through its non-TMA variant; unset or 0 = normal.
int dispatch_mode() {
  const char* e = getenv("LISA_TD_DISPATCH");
  return e ? atoi(e) : 0;
}

// ------------------------------------------------------------------ constant tables
void make_lagw(int order, LagW* out) {
  const int H = (order + 1) / 2;
  for (int i = 0; i < MAX_HALF; ++i) out->w[i] = 0.0;
  for (int k = 1; k <= H; ++k) {
    long double f = 1.0L;  // (k+H-1)! (H-k)!
    for (int i = 2; i <= k + H - 1; ++i) f *= i;
    for (int i = 2; i <= H - k; ++i) f *= i;
    long double w = 1.0L / f;
    if ((H - k) & 1) w = -w;
    out->w[k - 1] = (double)w;
  }
}

void make_lags(int order, LagS* out) {
  const int H = (order + 1) / 2;
  long double w[MAX_HALF];
  long double logabs = 0.0L;
  int neg = 0;
  for (int k = 1; k <= H; ++k) {
    long double f = 1.0L;  // (k+H-1)! (H-k)!
    for (int i = 2; i <= k + H - 1; ++i) f *= i;
    for (int i = 2; i <= H - k; ++i) f *= i;
    w[k - 1] = 1.0L / f;
    if ((H - k) & 1) {
      w[k - 1] = -w[k - 1];
      ++neg;
    }
    logabs += logl(fabsl(w[k - 1]));
  }
  const long double R = expl(logabs / H);  // |prod w|^(1/H)
  for (int i = 0; i < MAX_HALF; ++i) out->rho[i] = out->rc[i] = 0.0;
  // g is formed from the ROUNDED rho_k: g prod_{i != k} rho_i = R / rho_k (1 + O(1e-19)), so
  // the effective weight of pair k is off from w_k by the rounding of rho_k alone (<= 1.1e-16).
  long double g = R;
  for (int k = 1; k <= H; ++k) {
    const double rho = (double)(R / w[k - 1]);
    out->rho[k - 1] = rho;
    out->rc[k - 1] = (double)((long double)rho * (long double)(k * (1 - k)));
    g /= (long double)rho;
  }
  out->g = (double)g;
  (void)neg;
}

// KEPLER1 on the host (long double), used only to bound |r| and L for margin validation.
static void kepler1_host(const lisa_td_orbit* o, long double t, long double r[3][3]) {
  const long double PI_L = 3.14159265358979323846264338327950288L;
  long double a = o->a_m, delta = (long double)o->L_m / (2 * a), sq3 = sqrtl(3.0L);
  long double e = sqrtl(1 + 2 * delta / sq3 + 4 * delta * delta / 3) - 1;
  long double inc = atanl(delta / (1 + delta / sq3));
  for (int k = 0; k < 3; ++k) {
    long double sigma = 2 * PI_L * k / 3;
    long double M = 2 * PI_L * (t - o->t_ref) / o->year_s - sigma - o->phase0;
    long double psi = M + e * sinl(M);
    long double x = a * (cosl(psi) - e) * cosl(inc), y = a * sqrtl(1 - e * e) * sinl(psi);
    long double z = a * (cosl(psi) - e) * sinl(inc);
    r[k][0] = cosl(sigma) * x - sinl(sigma) * y;
    r[k][1] = sinl(sigma) * x + cosl(sigma) * y;
    r[k][2] = z;
  }
}

}  // namespace lisa

// Tabulated orbit: device copy for the kernels, host-side bounds for the margin / halo checks.
struct lisa_td_orbit_table {
  int n_tab, order;
  double t_tab0, dt_tab;
  double* dev;
  double max_r, max_L, max_off, max_rate;  // metres, metres, metres, metres per second
};

namespace lisa {

static int make_orbit_dev_kind(const lisa_td_orbit* o, OrbitDev* d);
int make_orbit_dev(const lisa_td_orbit* o, OrbitDev* d) {
  if (!o) return set_error(LISA_TD_EINVAL, "orbit_host is NULL");
  if ((o->tt_order != 0 && o->tt_order != 1) || (o->tdi_nested != 0 && o->tdi_nested != 1))
    return set_error(LISA_TD_EINVAL, "orbit: tt_order=%d and tdi_nested=%d must be 0 or 1", o->tt_order, o->tdi_nested);
  int rc = make_orbit_dev_kind(o, d);
  if (rc) return rc;
  d->nested = o->tdi_nested;
  if (o->kind != 0 && o->tt_order) {  // A22: L = (d/c)(1 + n.v/c), |v|/c < 1.2e-4 for any heliocentric 1 AU orbit
    d->tt_order = 1;
    d->max_L *= 1.0 + 1.2e-4;
  }
  return LISA_TD_OK;
}
static int make_orbit_dev_kind(const lisa_td_orbit* o, OrbitDev* d) {
  memset(d, 0, sizeof(*d));
  d->kind = o->kind;
  if (o->kind == 2) {
    const lisa_td_orbit_table* t = o->table;
    if (!t) return set_error(LISA_TD_EINVAL, "orbit: kind TABLE needs a lisa_td_orbit_table");
    d->tab = t->dev;
    d->n_tab = t->n_tab;
    d->tab_order = t->order;
    d->t_tab0 = t->t_tab0;
    d->inv_dt_tab = 1.0 / t->dt_tab;
    for (int i = 0; i <= t->order; ++i) {
      long double den = 1.0L;
      for (int m = 0; m <= t->order; ++m)
        if (m != i) den *= (long double)(i - m);
      d->tab_w[i] = (double)(1.0L / den);
    }
    d->max_r_over_c = t->max_r * 1.01 / C_LIGHT;
    d->max_L = t->max_L * 1.01 / C_LIGHT;
    d->max_off_over_c = t->max_off * 1.01 / C_LIGHT;
    d->max_dc_rate = t->max_rate * 1.05 / C_LIGHT;
    return LISA_TD_OK;
  }
  if (o->kind == 0) {
    double mr = 0.0, mL = 0.0;
    for (int k = 0; k < 3; ++k) {
      double s = 0.0;
      for (int j = 0; j < 3; ++j) {
        d->r[k][j] = o->r_static[k][j];
        s += o->r_static[k][j] * o->r_static[k][j];
      }
      mr = fmax(mr, sqrt(s));
    }
    for (int l = 0; l < 6; ++l) {
      if (!(o->L_static[l] >= 0.0)) return set_error(LISA_TD_EINVAL, "orbit: L_static[%d] must be >= 0", l);
      d->L[l] = o->L_static[l];
      mL = fmax(mL, o->L_static[l]);
    }
    d->max_r_over_c = mr / C_LIGHT;
    d->max_off_over_c = mr / C_LIGHT;
    d->max_dc_rate = 0.0;
    d->max_L = mL;
    return LISA_TD_OK;
  }
  if (o->kind != 1) return set_error(LISA_TD_EINVAL, "orbit: unknown kind %d", o->kind);
  if (!(o->a_m > 0) || !(o->L_m > 0) || !(o->year_s > 0))
    return set_error(LISA_TD_EINVAL, "orbit: KEPLER1 needs a_m, L_m, year_s > 0");
  // the bounds below take ~3 ms of long-double libm per evaluation: remember the last orbit of
  // this thread (a sampler calls with the same orbit millions of times)
  struct Memo { bool valid; double key[5]; OrbitDev dev; };
  static thread_local Memo memo = {false, {0, 0, 0, 0, 0}, {}};
  const double key[5] = {o->L_m, o->a_m, o->year_s, o->phase0, o->t_ref};
  if (memo.valid && memcmp(memo.key, key, sizeof(key)) == 0) {
    *d = memo.dev;
    return LISA_TD_OK;
  }
  const long double PI_L = 3.14159265358979323846264338327950288L;
  long double a = o->a_m, delta = (long double)o->L_m / (2 * a), sq3 = sqrtl(3.0L);
  long double e = sqrtl(1 + 2 * delta / sq3 + 4 * delta * delta / 3) - 1;
  long double inc = atanl(delta / (1 + delta / sq3));
  long double bq = sqrtl(1 - e * e);
  d->w = (double)(2 * PI_L / o->year_s);
  d->t_ref = o->t_ref;
  d->phase0 = o->phase0;
  d->a = o->a_m;
  d->a_over_c = (double)(a / (long double)C_LIGHT);
  d->e = (double)e;
  d->ci = (double)cosl(inc);
  d->si = (double)sinl(inc);
  d->dci = (double)(-2 * sinl(inc / 2) * sinl(inc / 2));
  d->bq = (double)bq;
  d->dbq = (double)(-e * e / (1 + bq));
  for (int k = 0; k < 3; ++k) {
    d->cs[k] = (double)cosl(2 * PI_L * k / 3);
    d->sn[k] = (double)sinl(2 * PI_L * k / 3);
  }
  // bounds over one orbital period (the motion is periodic), 4096 points, 0.1 % head-room
  long double mr = 0, mL = 0, mo = 0;
  for (int i = 0; i < 4096; ++i) {
    long double r[3][3];
    const long double ti = o->t_ref + (long double)o->year_s * i / 4096;
    kepler1_host(o, ti, r);
    const long double Mc = 2 * PI_L * (ti - o->t_ref) / o->year_s - o->phase0;
    for (int k = 0; k < 3; ++k) {
      const long double ox = r[k][0] - a * cosl(Mc), oy = r[k][1] - a * sinl(Mc);
      mo = fmaxl(mo, sqrtl(ox * ox + oy * oy + r[k][2] * r[k][2]));
      mr = fmaxl(mr, sqrtl(r[k][0] * r[k][0] + r[k][1] * r[k][1] + r[k][2] * r[k][2]));
      const int k2 = (k + 1) % 3;
      long double dx = r[k][0] - r[k2][0], dy = r[k][1] - r[k2][1], dz = r[k][2] - r[k2][2];
      mL = fmaxl(mL, sqrtl(dx * dx + dy * dy + dz * dz));
    }
  }
  d->max_r_over_c = (double)(mr * 1.001L / C_LIGHT);
  d->max_L = (double)(mL * 1.001L / C_LIGHT);
  d->max_off_over_c = (double)(mo * 1.001L / C_LIGHT);
  d->max_dc_rate = d->a_over_c * d->w;
  memcpy(memo.key, key, sizeof(key));
  memo.dev = *d;
  memo.valid = true;
  return LISA_TD_OK;
}

// kernels (other translation units)
int run_modes_to_pol(int, long long, int, const int*, const int*, const double*, const double*,
                     const double*, const double*, const double*, const double*, const double*,
                     const double*, const double*, double*, double*, cudaStream_t);
int run_link_response(int, long long, double, double, int, long long, const double*, const double*,
                      const double*, const double*, const OrbitDev&, double*, cudaStream_t, int up2 = 0);
int run_laser_links(long long, double, double, int, long long, const double*, const OrbitDev&,
                    double*, cudaStream_t);
int run_tdi(int, long long, double, double, int, int, int, long long, long long, const double*,
            const OrbitDev&, double*, cudaStream_t, double* tab_ws = nullptr, long long tab_ws_bytes = 0);
long long tdi_workspace_bytes(long long N);
int run_tdi_static(int, long long, double, double, int, int, int, long long, long long, const double*,
                   const OrbitDev&, double*, int check, cudaStream_t);
struct Plan;
int plan_create(Plan**, int, long long);
int plan_destroy(Plan*);
int run_spectrum(Plan*, int, long long, const double*, double*, cudaStream_t);
int run_loglike(Plan*, int, long long, const double*, const double*, const double*, long long,
                long long, double*, double*, double*, cudaStream_t, int n_ch);
int run_fisher(Plan*, int, long long, const double*, const double*, const double*, long long, long long,
               double*, cudaStream_t);

// ------------------------------------------------------------------ validation helpers
static int check_common(const char* fn, int B, long long N, double dt, int order) {
  if (B <= 0) return set_error(LISA_TD_EINVAL, "%s: B must be > 0 (got %d)", fn, B);
  if (N <= 0) return set_error(LISA_TD_EINVAL, "%s: N must be > 0 (got %lld)", fn, N);
  if (!(dt > 0)) return set_error(LISA_TD_EINVAL, "%s: dt must be > 0", fn);
  if (order < 1 || order > 63 || !(order & 1))
    return set_error(LISA_TD_EINVAL, "%s: order must be odd in [1,63] (got %d)", fn, order);
  if (B > 65535) return set_error(LISA_TD_EINVAL, "%s: B must be <= 65535", fn);
  return LISA_TD_OK;
}
#define REQUIRE_PTR(fn, p)                                                              \
  do {                                                                                  \
    if (!(p)) return set_error(LISA_TD_EINVAL, "%s: %s is NULL", fn, #p);               \
    if (!aligned16(p)) return set_error(LISA_TD_EALIGN, "%s: %s is not 16-byte aligned", fn, #p); \
  } while (0)
#define OPTIONAL_PTR(fn, p)                                                             \
  do {                                                                                  \
    if ((p) && !aligned16(p)) return set_error(LISA_TD_EALIGN, "%s: %s is not 16-byte aligned", fn, #p); \
  } while (0)

static int check_margin_y(const char* fn, long long N, double dt, int order, long long margin_y, const OrbitDev& od) {
  const long long need = (long long)ceil((od.max_r_over_c + od.max_L) / dt) + (order + 1) / 2;
  if (margin_y < need)
    return set_error(LISA_TD_EINVAL, "%s: margin_y=%lld does not cover the stencil reach %lld", fn, margin_y, need);
  if (margin_y > 8192) return set_error(LISA_TD_EINVAL, "%s: margin_y=%lld too large (max 8192)", fn, margin_y);
  if (N < 2 * margin_y) return set_error(LISA_TD_EINVAL, "%s: N=%lld must be >= 2*margin_y", fn, N);
  return LISA_TD_OK;
}
// margin_y: the margin of the link responses that feed this TDI call when the library knows it (the
// combined entry points), 0 otherwise: TDI must not interpolate across the hard-zeroed edge of y
// (reading A7: m_lo >= m_y + reach, m_hi >= m_y + (p+1)/2).
static int check_margin_tdi(const char* fn, long long N, double dt, int order, int generation,
                            long long margin_lo, long long margin_hi, const OrbitDev& od, long long margin_y = 0) {
  if (generation != 15 && generation != 20)
    return set_error(LISA_TD_EINVAL, "%s: generation must be 15 or 20 (got %d)", fn, generation);
  const int h = (order + 1) / 2;
  const long long need_lo = margin_y + (long long)ceil((generation == 20 ? 7 : 3) * od.max_L / dt) + h;
  if (margin_lo < need_lo)
    return set_error(LISA_TD_EINVAL, "%s: margin_lo=%lld does not cover margin_y=%lld plus the stencil reach (need %lld)", fn,
                     margin_lo, margin_y, need_lo);
  if (margin_hi < margin_y + h)
    return set_error(LISA_TD_EINVAL, "%s: margin_hi=%lld must be >= margin_y + (order+1)/2 = %lld", fn, margin_hi,
                     margin_y + h);
  if (N < margin_lo + margin_hi) return set_error(LISA_TD_EINVAL, "%s: N=%lld smaller than the margins", fn, N);
  return LISA_TD_OK;
}

static int check_table_range(const char* fn, const lisa_td_orbit* o, long long N, double t0, double dt) {
  if (!o || o->kind != 2 || !o->table) return LISA_TD_OK;
  const lisa_td_orbit_table* t = o->table;
  const double t_end = t->t_tab0 + (t->n_tab - 1) * t->dt_tab;
  if (t0 < t->t_tab0 || t0 + (double)N * dt > t_end)
    return set_error(LISA_TD_EINVAL, "%s: the orbit table [%g, %g] s does not cover the grid [%g, %g] s", fn,
                     t->t_tab0, t_end, t0, t0 + (double)N * dt);
  return LISA_TD_OK;
}

}  // namespace lisa

using namespace lisa;

// ====================================================================== C ABI
extern "C" {

const char* lisa_td_last_error(void) { return g_err; }

int lisa_td_orbit_table_create(lisa_td_orbit_table** out, int n_tab, double t_tab0, double dt_tab,
                               int interp_order, const double* r_host) {
  const char* fn = "lisa_td_orbit_table_create";
  if (!out || !r_host) return set_error(LISA_TD_EINVAL, "%s: NULL argument", fn);
  if (interp_order < 1 || interp_order > 15 || !(interp_order & 1))
    return set_error(LISA_TD_EINVAL, "%s: interp_order must be odd in [1,15] (got %d)", fn, interp_order);
  if (n_tab <= interp_order) return set_error(LISA_TD_EINVAL, "%s: n_tab must exceed interp_order", fn);
  if (!(dt_tab > 0)) return set_error(LISA_TD_EINVAL, "%s: dt_tab must be > 0", fn);
  lisa_td_orbit_table* t = new lisa_td_orbit_table();
  t->n_tab = n_tab; t->order = interp_order; t->t_tab0 = t_tab0; t->dt_tab = dt_tab; t->dev = nullptr;
  t->max_r = t->max_L = t->max_off = t->max_rate = 0.0;
  double prev_c[3] = {0, 0, 0};
  for (int j = 0; j < n_tab; ++j) {
    const double* r = r_host + (size_t)j * 9;
    double c[3];
    for (int x = 0; x < 3; ++x) c[x] = (r[x] + r[3 + x] + r[6 + x]) / 3.0;
    for (int k = 0; k < 3; ++k) {
      const double* a = r + 3 * k;
      const double* b = r + 3 * ((k + 1) % 3);
      t->max_r = fmax(t->max_r, sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]));
      t->max_L = fmax(t->max_L, sqrt((a[0] - b[0]) * (a[0] - b[0]) + (a[1] - b[1]) * (a[1] - b[1]) + (a[2] - b[2]) * (a[2] - b[2])));
      t->max_off = fmax(t->max_off, sqrt((a[0] - c[0]) * (a[0] - c[0]) + (a[1] - c[1]) * (a[1] - c[1]) + (a[2] - c[2]) * (a[2] - c[2])));
    }
    if (j > 0)
      t->max_rate = fmax(t->max_rate, sqrt((c[0] - prev_c[0]) * (c[0] - prev_c[0]) + (c[1] - prev_c[1]) * (c[1] - prev_c[1]) +
                                           (c[2] - prev_c[2]) * (c[2] - prev_c[2])) / dt_tab);
    for (int x = 0; x < 3; ++x) prev_c[x] = c[x];
  }
  int rc = check_cuda(cudaMalloc(&t->dev, sizeof(double) * 9 * (size_t)n_tab), "cudaMalloc(orbit table)");
  if (rc == LISA_TD_OK)
    rc = check_cuda(cudaMemcpy(t->dev, r_host, sizeof(double) * 9 * (size_t)n_tab, cudaMemcpyHostToDevice), "cudaMemcpy(orbit table)");
  if (rc != LISA_TD_OK) {
    cudaFree(t->dev);
    delete t;
    return rc;
  }
  *out = t;
  return LISA_TD_OK;
}
int lisa_td_orbit_table_destroy(lisa_td_orbit_table* t) {
  if (!t) return LISA_TD_OK;
  cudaFree(t->dev);
  delete t;
  return LISA_TD_OK;
}
int lisa_td_version(void) { return 100; }
int lisa_td_check(void* stream) {
  const char* fn = "lisa_td_check";
  LISA_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  return take_device_errors(fn);
}

int lisa_td_modes_to_pol(int B, long long N, int n_modes, const int* l_host, const int* m_host,
                         const double* amp, const double* phase, const double* alpha,
                         const double* beta, const double* gamma, const double* iota,
                         const double* phi, const double* psi, const double* euler0,
                         double* hplus, double* hcross, void* stream) {
  const char* fn = "lisa_td_modes_to_pol";
  if (B <= 0 || B > 65535) return set_error(LISA_TD_EINVAL, "%s: B must be in [1,65535] (got %d)", fn, B);
  if (N <= 0) return set_error(LISA_TD_EINVAL, "%s: N must be > 0", fn);
  if (n_modes <= 0 || n_modes > 16) return set_error(LISA_TD_EINVAL, "%s: n_modes must be in [1,16]", fn);
  if (!l_host || !m_host) return set_error(LISA_TD_EINVAL, "%s: l_host / m_host is NULL", fn);
  for (int k = 0; k < n_modes; ++k)
    if (l_host[k] < 2 || l_host[k] > 8 || m_host[k] < -l_host[k] || m_host[k] > l_host[k])
      return set_error(LISA_TD_EINVAL, "%s: mode %d = (%d,%d) outside 2<=l<=8, |m|<=l", fn, k, l_host[k], m_host[k]);
  REQUIRE_PTR(fn, amp); REQUIRE_PTR(fn, phase); REQUIRE_PTR(fn, iota); REQUIRE_PTR(fn, phi);
  REQUIRE_PTR(fn, psi); REQUIRE_PTR(fn, hplus); REQUIRE_PTR(fn, hcross);
  const int nang = (alpha != 0) + (beta != 0) + (gamma != 0);
  if (nang != 0 && nang != 3) return set_error(LISA_TD_EINVAL, "%s: alpha, beta, gamma must be all NULL or all given", fn);
  OPTIONAL_PTR(fn, alpha); OPTIONAL_PTR(fn, beta); OPTIONAL_PTR(fn, gamma); OPTIONAL_PTR(fn, euler0);
  return run_modes_to_pol(B, N, n_modes, l_host, m_host, amp, phase, alpha, beta, gamma, iota, phi, psi,
                          euler0, hplus, hcross, (cudaStream_t)stream);
}

int lisa_td_link_response(int B, long long N, double t0, double dt, int order, long long margin_y,
                          const double* hplus, const double* hcross, const double* lambda,
                          const double* beta_sky, const lisa_td_orbit* orbit_host, double* y,
                          void* stream) {
  const char* fn = "lisa_td_link_response";
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  REQUIRE_PTR(fn, hplus); REQUIRE_PTR(fn, hcross); REQUIRE_PTR(fn, lambda); REQUIRE_PTR(fn, beta_sky);
  REQUIRE_PTR(fn, y);
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_y(fn, N, dt, order, margin_y, od))) return rc;
  return run_link_response(B, N, t0, dt, order, margin_y, hplus, hcross, lambda, beta_sky, od, y,
                           (cudaStream_t)stream);
}

int lisa_td_link_response_up2(int B, long long N, double t0, double dt, int order, long long margin_y,
                              const double* hplus_c, const double* hcross_c, const double* lambda,
                              const double* beta_sky, const lisa_td_orbit* orbit_host, double* y,
                              void* stream) {
  const char* fn = "lisa_td_link_response_up2";
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  if (N & 1) return set_error(LISA_TD_EINVAL, "%s: N must be even (got %lld)", fn, N);
  REQUIRE_PTR(fn, hplus_c); REQUIRE_PTR(fn, hcross_c); REQUIRE_PTR(fn, lambda); REQUIRE_PTR(fn, beta_sky);
  REQUIRE_PTR(fn, y);
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_y(fn, N, dt, order, margin_y, od))) return rc;
  return run_link_response(B, N, t0, dt, order, margin_y, hplus_c, hcross_c, lambda, beta_sky, od, y,
                           (cudaStream_t)stream, 1);
}

int lisa_td_laser_links(long long N, double t0, double dt, int order, long long margin,
                        const double* p, const lisa_td_orbit* orbit_host, double* y, void* stream) {
  const char* fn = "lisa_td_laser_links";
  int rc = check_common(fn, 1, N, dt, order);
  if (rc) return rc;
  REQUIRE_PTR(fn, p); REQUIRE_PTR(fn, y);
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  const long long need = (long long)ceil(od.max_L / dt) + (order + 1) / 2;
  if (margin < need || N < 2 * margin)
    return set_error(LISA_TD_EINVAL, "%s: margin=%lld must be >= %lld and N >= 2*margin", fn, margin, need);
  return run_laser_links(N, t0, dt, order, margin, p, od, y, (cudaStream_t)stream);
}

int lisa_td_tdi2(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
                 long long margin_lo, long long margin_hi, const double* y,
                 const lisa_td_orbit* orbit_host, double* tdi, void* stream) {
  const char* fn = "lisa_td_tdi2";
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  if (out_kind != 0 && out_kind != 1) return set_error(LISA_TD_EINVAL, "%s: out_kind must be 0 (XYZ) or 1 (AET)", fn);
  REQUIRE_PTR(fn, y); REQUIRE_PTR(fn, tdi);
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_tdi(fn, N, dt, order, generation, margin_lo, margin_hi, od))) return rc;
  return run_tdi(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi, y, od, tdi,
                 (cudaStream_t)stream);
}

// lisa_td_tdi2 with its scratch in a file-scope device array (k3_tdi.cu): no allocation of any kind
int lisa_td_tdi2_static(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
                        long long margin_lo, long long margin_hi, const double* y,
                        const lisa_td_orbit* orbit_host, double* tdi, int check, void* stream) {
  const char* fn = "lisa_td_tdi2_static";
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  if (N > LISA_TD_TDI2_STATIC_MAX_N)
    return set_error(LISA_TD_EINVAL, "%s: N=%lld exceeds LISA_TD_TDI2_STATIC_MAX_N=%d samples (the size of the static scratch array)",
                     fn, N, LISA_TD_TDI2_STATIC_MAX_N);
  if (out_kind != 0 && out_kind != 1) return set_error(LISA_TD_EINVAL, "%s: out_kind must be 0 (XYZ) or 1 (AET)", fn);
  REQUIRE_PTR(fn, y); REQUIRE_PTR(fn, tdi);
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_tdi(fn, N, dt, order, generation, margin_lo, margin_hi, od))) return rc;
  return run_tdi_static(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi, y, od, tdi, check,
                        (cudaStream_t)stream);
}

// [B][6][N] link responses, then the anchor tables of S3 (k3_tdi.cu)
static long long links_bytes(int B, long long N) { return ((long long)sizeof(double) * 6 * (long long)B * N + 255) / 256 * 256; }
long long lisa_td_response_tdi_workspace_bytes(int B, long long N) {
  if (B <= 0 || N <= 0) return 0;
  return links_bytes(B, N) + tdi_workspace_bytes(N);
}

int lisa_td_response_tdi(int B, long long N, double t0, double dt, int order, long long margin_y,
                         int generation, int out_kind, long long margin_lo, long long margin_hi,
                         const double* hplus, const double* hcross, const double* lambda,
                         const double* beta_sky, const lisa_td_orbit* orbit_host, double* tdi,
                         void* workspace, long long workspace_bytes, void* stream) {
  const char* fn = "lisa_td_response_tdi";
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  if (out_kind != 0 && out_kind != 1) return set_error(LISA_TD_EINVAL, "%s: out_kind must be 0 or 1", fn);
  REQUIRE_PTR(fn, hplus); REQUIRE_PTR(fn, hcross); REQUIRE_PTR(fn, lambda); REQUIRE_PTR(fn, beta_sky);
  REQUIRE_PTR(fn, tdi); REQUIRE_PTR(fn, workspace);
  if (workspace_bytes < lisa_td_response_tdi_workspace_bytes(B, N))
    return set_error(LISA_TD_ENOMEM, "%s: workspace of %lld bytes is smaller than the %lld needed", fn,
                     workspace_bytes, lisa_td_response_tdi_workspace_bytes(B, N));
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_y(fn, N, dt, order, margin_y, od))) return rc;
  if ((rc = check_margin_tdi(fn, N, dt, order, generation, margin_lo, margin_hi, od, margin_y))) return rc;
  double* y = static_cast<double*>(workspace);
  if ((rc = run_link_response(B, N, t0, dt, order, margin_y, hplus, hcross, lambda, beta_sky, od, y,
                              (cudaStream_t)stream)))
    return rc;
  return run_tdi(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi, y, od, tdi,
                 (cudaStream_t)stream, reinterpret_cast<double*>(static_cast<char*>(workspace) + links_bytes(B, N)),
                 tdi_workspace_bytes(N));
}

struct lisa_td_plan {
  lisa::Plan* p;
};

int lisa_td_plan_create(lisa_td_plan** out, int B, long long N) {
  const char* fn = "lisa_td_plan_create";
  if (!out) return set_error(LISA_TD_EINVAL, "%s: out is NULL", fn);
  if (B <= 0 || B > 65535 || N < 2 || (N & 1))
    return set_error(LISA_TD_EINVAL, "%s: need 0 < B <= 65535 and even N >= 2", fn);
  lisa::Plan* p = nullptr;
  int rc = plan_create(&p, B, N);
  if (rc) return rc;
  *out = new lisa_td_plan{p};
  return LISA_TD_OK;
}
int lisa_td_plan_destroy(lisa_td_plan* plan) {
  if (!plan) return LISA_TD_OK;
  plan_destroy(plan->p);
  delete plan;
  return LISA_TD_OK;
}

static int check_band(const char* fn, long long N, long long kmin, long long kmax) {
  if (kmin < 0 || kmin > kmax || kmax > N / 2)
    return set_error(LISA_TD_EINVAL, "%s: need 0 <= kmin <= kmax <= N/2 (got %lld, %lld)", fn, kmin, kmax);
  return LISA_TD_OK;
}

int lisa_td_loglike(lisa_td_plan* plan, int B, long long N, const double* tdi,
                    const double* data_spec, const double* weight, long long kmin, long long kmax,
                    double* loglike, double* dh, double* hh, void* stream) {
  const char* fn = "lisa_td_loglike";
  if (!plan) return set_error(LISA_TD_EINVAL, "%s: plan is NULL", fn);
  if (B <= 0) return set_error(LISA_TD_EINVAL, "%s: B must be > 0", fn);
  int rc = check_band(fn, N, kmin, kmax);
  if (rc) return rc;
  REQUIRE_PTR(fn, tdi); REQUIRE_PTR(fn, data_spec); REQUIRE_PTR(fn, weight); REQUIRE_PTR(fn, loglike);
  return run_loglike(plan->p, B, N, tdi, data_spec, weight, kmin, kmax, loglike, dh, hh, (cudaStream_t)stream, 3);
}

// ---- S1..S5 from DEVICE inputs in one call
static long long al256(long long v) { return (v + 255) / 256 * 256; }
long long lisa_td_loglike_from_modes_workspace_bytes(int B, long long N) {
  if (B <= 0 || N <= 0) return 0;
  const long long d = (long long)sizeof(double);
  // h+, hx [B][N] | y [B][6][N] | tdi [B][3][N] | anchor tables of S3
  return 2 * al256(d * B * N) + al256(d * 6 * B * N) + al256(d * 3 * B * N) + tdi_workspace_bytes(N);
}

int lisa_td_loglike_from_modes(lisa_td_plan* plan, int B, long long N, int n_modes, const int* l_host, const int* m_host,
                               const double* amp, const double* phase, const double* alpha, const double* beta,
                               const double* gamma, const double* iota, const double* phi, const double* psi,
                               const double* lambda, const double* beta_sky, double t0, double dt, int order,
                               long long margin_y, int generation, long long margin_lo, long long margin_hi,
                               const lisa_td_orbit* orbit_host, const double* data_spec, const double* weight,
                               long long kmin, long long kmax, double* loglike, double* dh, double* hh, void* workspace,
                               long long workspace_bytes, void* stream) {
  const char* fn = "lisa_td_loglike_from_modes";
  if (!plan) return set_error(LISA_TD_EINVAL, "%s: plan is NULL", fn);
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  if (n_modes <= 0 || n_modes > 16) return set_error(LISA_TD_EINVAL, "%s: n_modes must be in [1,16]", fn);
  if (!l_host || !m_host) return set_error(LISA_TD_EINVAL, "%s: l_host / m_host is NULL", fn);
  for (int k = 0; k < n_modes; ++k)
    if (l_host[k] < 2 || l_host[k] > 8 || m_host[k] < -l_host[k] || m_host[k] > l_host[k])
      return set_error(LISA_TD_EINVAL, "%s: mode %d = (%d,%d) outside 2<=l<=8, |m|<=l", fn, k, l_host[k], m_host[k]);
  REQUIRE_PTR(fn, amp); REQUIRE_PTR(fn, phase); REQUIRE_PTR(fn, iota); REQUIRE_PTR(fn, phi); REQUIRE_PTR(fn, psi);
  REQUIRE_PTR(fn, lambda); REQUIRE_PTR(fn, beta_sky); REQUIRE_PTR(fn, data_spec); REQUIRE_PTR(fn, weight);
  REQUIRE_PTR(fn, loglike); REQUIRE_PTR(fn, workspace);
  const int nang = (alpha != 0) + (beta != 0) + (gamma != 0);
  if (nang != 0 && nang != 3) return set_error(LISA_TD_EINVAL, "%s: alpha, beta, gamma must be all NULL or all given", fn);
  OPTIONAL_PTR(fn, alpha); OPTIONAL_PTR(fn, beta); OPTIONAL_PTR(fn, gamma);
  if ((rc = check_band(fn, N, kmin, kmax))) return rc;
  if (workspace_bytes < lisa_td_loglike_from_modes_workspace_bytes(B, N))
    return set_error(LISA_TD_ENOMEM, "%s: workspace of %lld bytes is smaller than the %lld needed", fn, workspace_bytes,
                     lisa_td_loglike_from_modes_workspace_bytes(B, N));
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_y(fn, N, dt, order, margin_y, od))) return rc;
  if ((rc = check_margin_tdi(fn, N, dt, order, generation, margin_lo, margin_hi, od, margin_y))) return rc;
  const long long d = (long long)sizeof(double);
  char* w = static_cast<char*>(workspace);
  double* hp = reinterpret_cast<double*>(w);
  double* hc = reinterpret_cast<double*>(w + al256(d * B * N));
  double* y = reinterpret_cast<double*>(w + 2 * al256(d * B * N));
  double* tdi = reinterpret_cast<double*>(w + 2 * al256(d * B * N) + al256(d * 6 * B * N));
  double* tab = reinterpret_cast<double*>(w + 2 * al256(d * B * N) + al256(d * 6 * B * N) + al256(d * 3 * B * N));
  cudaStream_t st = (cudaStream_t)stream;
  if ((rc = run_modes_to_pol(B, N, n_modes, l_host, m_host, amp, phase, alpha, beta, gamma, iota, phi, psi, nullptr, hp, hc, st)))
    return rc;
  if ((rc = run_link_response(B, N, t0, dt, order, margin_y, hp, hc, lambda, beta_sky, od, y, st))) return rc;
  if ((rc = run_tdi(B, N, t0, dt, order, generation, 1, margin_lo, margin_hi, y, od, tdi, st, tab, tdi_workspace_bytes(N))))
    return rc;
  return run_loglike(plan->p, B, N, tdi, data_spec, weight, kmin, kmax, loglike, dh, hh, st, 3);
}

int lisa_td_loglike_channels(lisa_td_plan* plan, int B, long long N, int n_channels, const double* tdi,
                             const double* data_spec, const double* weight, long long kmin, long long kmax,
                             double* loglike, double* dh, double* hh, void* stream) {
  const char* fn = "lisa_td_loglike_channels";
  if (!plan) return set_error(LISA_TD_EINVAL, "%s: plan is NULL", fn);
  if (B <= 0) return set_error(LISA_TD_EINVAL, "%s: B must be > 0", fn);
  if (n_channels < 1 || n_channels > 3)
    return set_error(LISA_TD_EINVAL, "%s: n_channels=%d must be 1 (A), 2 (A,E) or 3 (A,E,T)", fn, n_channels);
  int rc = check_band(fn, N, kmin, kmax);
  if (rc) return rc;
  REQUIRE_PTR(fn, tdi); REQUIRE_PTR(fn, data_spec); REQUIRE_PTR(fn, weight); REQUIRE_PTR(fn, loglike);
  return run_loglike(plan->p, B, N, tdi, data_spec, weight, kmin, kmax, loglike, dh, hh, (cudaStream_t)stream,
                     n_channels);
}

int lisa_td_fisher(lisa_td_plan* plan, int D, long long N, const double* tdi, const double* delta_host,
                   const double* weight, long long kmin, long long kmax, double* fisher, void* stream) {
  const char* fn = "lisa_td_fisher";
  if (!plan) return set_error(LISA_TD_EINVAL, "%s: plan is NULL", fn);
  if (!delta_host) return set_error(LISA_TD_EINVAL, "%s: delta_host is NULL", fn);
  int rc = check_band(fn, N, kmin, kmax);
  if (rc) return rc;
  REQUIRE_PTR(fn, tdi); REQUIRE_PTR(fn, weight); REQUIRE_PTR(fn, fisher);
  return run_fisher(plan->p, D, N, tdi, delta_host, weight, kmin, kmax, fisher, (cudaStream_t)stream);
}

int lisa_td_spectrum(lisa_td_plan* plan, int B, long long N, const double* tdi, double* spec, void* stream) {
  const char* fn = "lisa_td_spectrum";
  if (!plan) return set_error(LISA_TD_EINVAL, "%s: plan is NULL", fn);
  if (B <= 0) return set_error(LISA_TD_EINVAL, "%s: B must be > 0", fn);
  REQUIRE_PTR(fn, tdi); REQUIRE_PTR(fn, spec);
  return run_spectrum(plan->p, B, N, tdi, spec, (cudaStream_t)stream);
}

int lisa_td_psd_weights(long long N, double dt, double acc_noise, double oms_noise, double arm_s,
                        int generation, double* weight_host) {
  const char* fn = "lisa_td_psd_weights";
  if (N < 2 || !(dt > 0) || !weight_host) return set_error(LISA_TD_EINVAL, "%s: bad arguments", fn);
  if (generation != 15 && generation != 20) return set_error(LISA_TD_EINVAL, "%s: generation must be 15 or 20", fn);
  const long long nf = N / 2 + 1;
  const double PI = 3.14159265358979323846;
  const double df = 1.0 / ((double)N * dt);
  for (int c = 0; c < 3; ++c) weight_host[(size_t)c * nf] = 0.0;
  for (long long k = 1; k < nf; ++k) {
    const double f = k * df, om = 2 * PI * f, oc = om / C_LIGHT;
    // Eq. 2.14 (shapes as printed; amplitudes are arguments, A15)
    const double r1 = 4e-4 / f, r2 = f / 0.008, r3 = 0.002 / f;
    const double s_acc = acc_noise * acc_noise * (1 + r1 * r1) * (1 + r2 * r2 * r2 * r2) / (om * om * om * om) * oc * oc;
    const double s_op = oms_noise * oms_noise * (1 + r3 * r3 * r3 * r3) * oc * oc;
    // Eq. 2.15 with x = 2 pi f L/c (A14)
    const double x = om * arm_s, sx = sin(x), cx = cos(x), sh = sin(0.5 * x);
    double s_ae = 8 * sx * sx * (2 * s_acc * (3 + 2 * cx + cos(2 * x)) + s_op * (2 + cx));
    // 1 - cos x written as 2 sin^2(x/2): no cancellation at low frequency
    double s_t = 16 * s_op * (2 * sh * sh) * sx * sx + 128 * s_acc * sx * sx * sh * sh * sh * sh;
    if (generation == 20) {
      const double g = 4 * sin(2 * x) * sin(2 * x);
      s_ae *= g;
      s_t *= g;
    }
    const double num = 4 * df * dt * dt;
    weight_host[k] = num / s_ae;
    weight_host[nf + k] = num / s_ae;
    weight_host[2 * nf + k] = num / s_t;
  }
  return LISA_TD_OK;
}

// ---------------------------------------------------------------------- host pipeline
struct lisa_td_pipeline {
  int chunk_B, n_modes, twisted;
  long long N, nf;
  cudaStream_t s_copy, s_comp;
  cudaEvent_t copied[2], done[2];
  double* in[2];      // per buffer: amp, phase [cB][M][N], (alpha,beta,gamma [cB][N]), 5 scalars [cB]
  double *hp, *hc, *y, *tdi, *ll;  // ll: [3][cB] (loglike, dh, hh)
  double* tab;                     // anchor tables of S3
  double *data_spec, *weight;
  lisa::Plan* plan;
  size_t in_doubles;
};

int lisa_td_pipeline_destroy(lisa_td_pipeline* p) {
  if (!p) return LISA_TD_OK;
  for (int i = 0; i < 2; ++i) {
    cudaFree(p->in[i]);
    if (p->copied[i]) cudaEventDestroy(p->copied[i]);
    if (p->done[i]) cudaEventDestroy(p->done[i]);
  }
  cudaFree(p->hp); cudaFree(p->hc); cudaFree(p->y); cudaFree(p->tdi); cudaFree(p->ll); cudaFree(p->tab);
  cudaFree(p->data_spec); cudaFree(p->weight);
  if (p->plan) plan_destroy(p->plan);
  if (p->s_copy) cudaStreamDestroy(p->s_copy);
  if (p->s_comp) cudaStreamDestroy(p->s_comp);
  delete p;
  return LISA_TD_OK;
}

int lisa_td_pipeline_create(lisa_td_pipeline** out, int chunk_B, long long N, int n_modes, int twisted) {
  const char* fn = "lisa_td_pipeline_create";
  if (!out || chunk_B <= 0 || N < 2 || (N & 1) || n_modes <= 0 || n_modes > 16)
    return set_error(LISA_TD_EINVAL, "%s: bad arguments", fn);
  lisa_td_pipeline* p = new lisa_td_pipeline();
  memset(p, 0, sizeof(*p));
  p->chunk_B = chunk_B; p->N = N; p->nf = N / 2 + 1; p->n_modes = n_modes; p->twisted = twisted;
  const size_t cB = chunk_B;
  p->in_doubles = cB * (2 * (size_t)n_modes + (twisted ? 3 : 0)) * N + 8 * cB + 32;
  int rc = LISA_TD_OK;
#define PIPE_TRY(call) do { if (rc == LISA_TD_OK) rc = check_cuda((call), #call); } while (0)
  PIPE_TRY(cudaStreamCreateWithFlags(&p->s_copy, cudaStreamNonBlocking));
  PIPE_TRY(cudaStreamCreateWithFlags(&p->s_comp, cudaStreamNonBlocking));
  for (int i = 0; i < 2; ++i) {
    PIPE_TRY(cudaMalloc(&p->in[i], sizeof(double) * p->in_doubles));
    PIPE_TRY(cudaEventCreateWithFlags(&p->copied[i], cudaEventDisableTiming));
    PIPE_TRY(cudaEventCreateWithFlags(&p->done[i], cudaEventDisableTiming));
  }
  PIPE_TRY(cudaMalloc(&p->hp, sizeof(double) * cB * N));
  PIPE_TRY(cudaMalloc(&p->hc, sizeof(double) * cB * N));
  PIPE_TRY(cudaMalloc(&p->y, sizeof(double) * cB * 6 * N));
  PIPE_TRY(cudaMalloc(&p->tdi, sizeof(double) * cB * 3 * N));
  PIPE_TRY(cudaMalloc(&p->tab, (size_t)tdi_workspace_bytes(N)));
  PIPE_TRY(cudaMalloc(&p->ll, sizeof(double) * (4 * cB + 8)));
  PIPE_TRY(cudaMalloc(&p->data_spec, sizeof(double) * 6 * p->nf));
  PIPE_TRY(cudaMalloc(&p->weight, sizeof(double) * 4 * p->nf));
#undef PIPE_TRY
  if (rc == LISA_TD_OK) rc = plan_create(&p->plan, chunk_B, N);
  if (rc != LISA_TD_OK) {
    lisa_td_pipeline_destroy(p);
    return rc;
  }
  *out = p;
  return LISA_TD_OK;
}

static int pipeline_run(const char* fn, int up2, lisa_td_pipeline* p, int B, long long N, int n_modes, const int* l_host,
                        const int* m_host, const double* amp_host, const double* phase_host,
                        const double* alpha_host, const double* beta_host,
                        const double* gamma_host, const double* iota_host,
                        const double* phi_host, const double* psi_host,
                        const double* lambda_host, const double* beta_sky_host, double t0,
                        double dt, int order, long long margin_y, int generation,
                        long long margin_lo, long long margin_hi,
                        const lisa_td_orbit* orbit_host, const double* data_spec_host,
                        const double* weight_host, long long kmin, long long kmax,
                        double* loglike_host, double* dh_host, double* hh_host) {
  if (!p) return set_error(LISA_TD_EINVAL, "%s: pipeline is NULL", fn);
  int rc = check_common(fn, B, N, dt, order);
  if (rc) return rc;
  if (N != p->N || n_modes != p->n_modes) return set_error(LISA_TD_EINVAL, "%s: N / n_modes differ from the pipeline's", fn);
  const bool tw = alpha_host != nullptr;
  if (tw != (p->twisted != 0)) return set_error(LISA_TD_EINVAL, "%s: twisted flag differs from the pipeline's", fn);
  if (!amp_host || !phase_host || !iota_host || !phi_host || !psi_host || !lambda_host || !beta_sky_host ||
      !data_spec_host || !weight_host || !loglike_host || !l_host || !m_host || (tw && (!beta_host || !gamma_host)))
    return set_error(LISA_TD_EINVAL, "%s: a required host pointer is NULL", fn);
  for (int k = 0; k < n_modes; ++k)
    if (l_host[k] < 2 || l_host[k] > 8 || m_host[k] < -l_host[k] || m_host[k] > l_host[k])
      return set_error(LISA_TD_EINVAL, "%s: mode %d outside 2<=l<=8, |m|<=l", fn, k);
  if ((rc = check_band(fn, N, kmin, kmax))) return rc;
  OrbitDev od;
  if ((rc = make_orbit_dev(orbit_host, &od))) return rc;
  if ((rc = check_table_range(fn, orbit_host, N, t0, dt))) return rc;
  if ((rc = check_margin_y(fn, N, dt, order, margin_y, od))) return rc;
  if ((rc = check_margin_tdi(fn, N, dt, order, generation, margin_lo, margin_hi, od, margin_y))) return rc;

  const size_t M = n_modes, cB = p->chunk_B;
  // up2 (reading A20): the mode and angle arrays live on the 2 dt grid, Nin = N/2 + 1 samples
  // per row; sub-arrays start on even offsets so that every device array stays 16-byte aligned
  const size_t Nin = up2 ? (size_t)(N / 2 + 1) : (size_t)N;
  auto even = [](size_t v) { return (v + 1) & ~(size_t)1; };
  // everything that enqueues work runs inside `enqueue`, so that a failure half way can still wait for
  // what is already in flight before returning: the caller may free its host buffers right after
  auto enqueue = [&]() -> int {
  LISA_CUDA(cudaMemcpyAsync(p->data_spec, data_spec_host, sizeof(double) * 6 * p->nf, cudaMemcpyHostToDevice, p->s_copy));
  LISA_CUDA(cudaMemcpyAsync(p->weight, weight_host, sizeof(double) * 3 * p->nf, cudaMemcpyHostToDevice, p->s_copy));
  int it = 0;
  for (int b0 = 0; b0 < B; b0 += (int)cB, ++it) {
    const int buf = it & 1;
    const size_t nb = (size_t)((B - b0) < (int)cB ? (B - b0) : (int)cB);
    double* d = p->in[buf];
    double* d_amp = d;
    double* d_pha = d_amp + even(cB * M * Nin);
    double* d_al = d_pha + even(cB * M * Nin);
    double* d_be = d_al + (tw ? even(cB * Nin) : 0);
    double* d_ga = d_be + (tw ? even(cB * Nin) : 0);
    double* d_sc = d_ga + (tw ? even(cB * Nin) : 0);  // 5 x [cB] scalars, each slot padded to an even count
    const size_t sc_stride = (cB + 1) & ~(size_t)1;
    // copies of chunk `it` wait until the kernels that last used this buffer are done
    if (it >= 2) LISA_CUDA(cudaStreamWaitEvent(p->s_copy, p->done[buf], 0));
#define H2D(dst, src, count) LISA_CUDA(cudaMemcpyAsync((dst), (src), sizeof(double) * (count), cudaMemcpyHostToDevice, p->s_copy))
    H2D(d_amp, amp_host + (size_t)b0 * M * Nin, nb * M * Nin);
    H2D(d_pha, phase_host + (size_t)b0 * M * Nin, nb * M * Nin);
    if (tw) {
      H2D(d_al, alpha_host + (size_t)b0 * Nin, nb * Nin);
      H2D(d_be, beta_host + (size_t)b0 * Nin, nb * Nin);
      H2D(d_ga, gamma_host + (size_t)b0 * Nin, nb * Nin);
    }
    H2D(d_sc + 0 * sc_stride, iota_host + b0, nb);
    H2D(d_sc + 1 * sc_stride, phi_host + b0, nb);
    H2D(d_sc + 2 * sc_stride, psi_host + b0, nb);
    H2D(d_sc + 3 * sc_stride, lambda_host + b0, nb);
    H2D(d_sc + 4 * sc_stride, beta_sky_host + b0, nb);
#undef H2D
    LISA_CUDA(cudaEventRecord(p->copied[buf], p->s_copy));
    LISA_CUDA(cudaStreamWaitEvent(p->s_comp, p->copied[buf], 0));
    if ((rc = run_modes_to_pol((int)nb, (long long)Nin, n_modes, l_host, m_host, d_amp, d_pha, tw ? d_al : nullptr,
                               tw ? d_be : nullptr, tw ? d_ga : nullptr, d_sc, d_sc + sc_stride,
                               d_sc + 2 * sc_stride, nullptr, p->hp, p->hc, p->s_comp)))
      return rc;
    if ((rc = run_link_response((int)nb, N, t0, dt, order, margin_y, p->hp, p->hc, d_sc + 3 * sc_stride,
                                d_sc + 4 * sc_stride, od, p->y, p->s_comp, up2)))
      return rc;
    if ((rc = run_tdi((int)nb, N, t0, dt, order, generation, 1, margin_lo, margin_hi, p->y, od, p->tdi, p->s_comp, p->tab,
                      tdi_workspace_bytes(N))))
      return rc;
    if ((rc = run_loglike(p->plan, (int)nb, N, p->tdi, p->data_spec, p->weight, kmin, kmax, p->ll, p->ll + sc_stride,
                          p->ll + 2 * sc_stride, p->s_comp, 3)))
      return rc;
    LISA_CUDA(cudaMemcpyAsync(loglike_host + b0, p->ll, sizeof(double) * nb, cudaMemcpyDeviceToHost, p->s_comp));
    if (dh_host) LISA_CUDA(cudaMemcpyAsync(dh_host + b0, p->ll + sc_stride, sizeof(double) * nb, cudaMemcpyDeviceToHost, p->s_comp));
    if (hh_host) LISA_CUDA(cudaMemcpyAsync(hh_host + b0, p->ll + 2 * sc_stride, sizeof(double) * nb, cudaMemcpyDeviceToHost, p->s_comp));
    LISA_CUDA(cudaEventRecord(p->done[buf], p->s_comp));
  }
  return LISA_TD_OK;
  };
  rc = enqueue();
  const cudaError_t e1 = cudaStreamSynchronize(p->s_copy), e2 = cudaStreamSynchronize(p->s_comp);
  if (rc) return rc;  // the first failure, reported after both streams have drained
  LISA_CUDA(e1);
  LISA_CUDA(e2);
  return take_device_errors(fn);
}

int lisa_td_pipeline_host(lisa_td_pipeline* p, int B, long long N, int n_modes, const int* l_host,
                          const int* m_host, const double* amp_host, const double* phase_host,
                          const double* alpha_host, const double* beta_host,
                          const double* gamma_host, const double* iota_host,
                          const double* phi_host, const double* psi_host,
                          const double* lambda_host, const double* beta_sky_host, double t0,
                          double dt, int order, long long margin_y, int generation,
                          long long margin_lo, long long margin_hi,
                          const lisa_td_orbit* orbit_host, const double* data_spec_host,
                          const double* weight_host, long long kmin, long long kmax,
                          double* loglike_host, double* dh_host, double* hh_host) {
  return pipeline_run("lisa_td_pipeline_host", 0, p, B, N, n_modes, l_host, m_host, amp_host, phase_host, alpha_host,
                      beta_host, gamma_host, iota_host, phi_host, psi_host, lambda_host, beta_sky_host, t0, dt, order,
                      margin_y, generation, margin_lo, margin_hi, orbit_host, data_spec_host, weight_host, kmin, kmax,
                      loglike_host, dh_host, hh_host);
}

int lisa_td_pipeline_host_up2(lisa_td_pipeline* p, int B, long long N, int n_modes, const int* l_host,
                              const int* m_host, const double* amp_host, const double* phase_host,
                              const double* alpha_host, const double* beta_host,
                              const double* gamma_host, const double* iota_host,
                              const double* phi_host, const double* psi_host,
                              const double* lambda_host, const double* beta_sky_host, double t0,
                              double dt, int order, long long margin_y, int generation,
                              long long margin_lo, long long margin_hi,
                              const lisa_td_orbit* orbit_host, const double* data_spec_host,
                              const double* weight_host, long long kmin, long long kmax,
                              double* loglike_host, double* dh_host, double* hh_host) {
  return pipeline_run("lisa_td_pipeline_host_up2", 1, p, B, N, n_modes, l_host, m_host, amp_host, phase_host, alpha_host,
                      beta_host, gamma_host, iota_host, phi_host, psi_host, lambda_host, beta_sky_host, t0, dt, order,
                      margin_y, generation, margin_lo, margin_hi, orbit_host, data_spec_host, weight_host, kmin, kmax,
                      loglike_host, dh_host, hh_host);
}

}  // extern "C"
