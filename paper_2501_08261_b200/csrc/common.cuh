// common.cuh -- shared device/host helpers of liblisa_td (sm_100a only).
//
// Nothing in this directory includes, links or reads anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lisa_td.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "liblisa_td is written for sm_100a (B200) only"
#endif

namespace lisa {

// ------------------------------------------------------------------ errors (api.cu)
int set_error(int code, const char* fmt, ...);
int check_cuda(cudaError_t e, const char* what);
#define LISA_CUDA(call)                                        \
  do {                                                         \
    int _rc = ::lisa::check_cuda((call), #call);               \
    if (_rc != LISA_TD_OK) return _rc;                         \
  } while (0)
#define LISA_LAUNCH_CHECK(name) LISA_CUDA(cudaPeekAtLastError())

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
int sm_count();  // multiprocessors of the current device (api.cu)

// ------------------------------------------------------------------ sticky device-side errors
// The kernels size their shared-memory tiles and merged stencil windows from HOST-side bounds on
// the orbit (max |r|, max L, drift of the common delay).  Where an index computed on the device
// falls outside what those bounds promised, the kernel sets one of these words (and clamps the
// index for memory safety only): the result is then wrong, and the next synchronising call
// (lisa_td_check, lisa_td_pipeline_host) returns LISA_TD_EINVAL instead of a silent wrong answer.
// The words live in mapped pinned host memory (one allocation per process, host pointer ==
// device pointer under unified addressing), so reading them costs no copy.
enum DevErr { DEVERR_K2_WINDOW = 0, DEVERR_K3_WINDOW = 1, DEVERR_LASER_WINDOW = 2, DEVERR_COUNT = 4 };
unsigned int* device_error_words();  // api.cu; NULL if the allocation failed (checks are then skipped)
int take_device_errors(const char* fn);  // after a synchronisation: LISA_TD_EINVAL if a word is set (and clears it)
int dispatch_mode();  // test-only: environment variable LISA_TD_DISPATCH (0 normal, 1 generic kernels, 2 S1 without TMA)

constexpr double C_LIGHT = 299792458.0;  // m/s
constexpr int MAX_HALF = 32;             // (p+1)/2 for p <= 63

// ------------------------------------------------------------------ Lagrange weights
// Taps j = -H+1 .. H (H = (p+1)/2).  Nodes are paired (k, 1-k), k = 1..H:
//   (eps-k)(eps-(1-k)) = eps(eps-1) + k(1-k),
// and the barycentric weights satisfy w_{1-k} = -w_k,  w_k = (-1)^{H-k} / ((k+H-1)! (H-k)!).
// w[k-1] holds w_k, computed on the host in long double.  Passed to kernels BY VALUE so it
// lands in the constant bank (no global state, no races between streams).
struct LagW {
  double w[MAX_HALF];
};
void make_lagw(int order, LagW* out);

// Scaled form of the same weights for the compile-time-order kernels.  With rho_k = R / w_k
// and g = (prod_i w_i) / R^(H-1) one has  g * prod_{i != k} rho_i = w_k,  so the pair factors
// can carry the weights:  Q'_k = rho_k (q + k(1-k)) = fma(rho[k-1], q, rc[k-1]),
//   a_k = w_k prod_{i != k} Q_i = (g prod_{i<k} Q'_i) (prod_{i>k} Q'_i)
// -- one FMA and three multiplies per node pair instead of an add and four multiplies.
// R = |prod w_i|^(1/H) keeps every partial product far from over/underflow.
struct LagS {
  double rho[MAX_HALF];
  double rc[MAX_HALF];
  double g;
};
void make_lags(int order, LagS* out);

// ------------------------------------------------------------------ orbit (device form)
// KEPLER1 is evaluated as  r_k(t) = a (cos M, sin M, 0) + delta_k(t)  with the common 1 AU
// part split off ALGEBRAICALLY (exact rearrangement of reading A8), so that arm vectors and
// the differential delays between spacecraft are formed from ~1e9 m quantities rather than
// as differences of 1.5e11 m ones ("delay arithmetic").
struct OrbitDev {
  int kind;
  double w, t_ref, phase0;        // mean motion 2 pi / year
  double a, a_over_c;             // semi-major axis [m], [s]
  double e, ci, si, dci, bq, dbq; // eccentricity, cos/sin inclination, ci-1, sqrt(1-e^2), bq-1
  double cs[3], sn[3];            // cos/sin of sigma_k = 2 pi k / 3
  double r[3][3];                 // STATIC positions [m]
  double L[6];                    // STATIC light travel times [s]
  double max_r_over_c;            // host-side bounds used for margin validation [s]
  double max_L;                   // [s]
  double max_off_over_c;          // max |r_k - common part| / c (STATIC: max |r_k| / c) [s]
  double max_dc_rate;             // max |d/dt (common part)| / c: drift of the common delay [s/s]
  // TABLE (reading A21): positions tabulated at t_tab0 + j dt_tab, Lagrange degree tab_order
  const double* tab;              // DEVICE [n_tab][3][3] metres (owned by a lisa_td_orbit_table)
  int n_tab, tab_order;
  double t_tab0, inv_dt_tab;
  double tab_w[16];               // 1 / prod_{m != i} (i - m), i = 0..tab_order
  // delay model (reading A22): first-order light travel times, TDI delays chained along the path
  int tt_order, nested;
};
int make_orbit_dev(const lisa_td_orbit* o, OrbitDev* out);

#ifdef __CUDACC__

__device__ __forceinline__ void raise_error(unsigned int* words, int which) {
  if (words) reinterpret_cast<volatile unsigned int*>(words)[which] = 1u;
}

// Link index 0..5 <-> l = [1,2,3,-1,-2,-3]; sender / receiver spacecraft (0-based).
__host__ __device__ constexpr int link_s(int l) { return l < 3 ? (l + 2) % 3 : (l - 3 + 1) % 3; }
__host__ __device__ constexpr int link_r(int l) { return l < 3 ? (l + 1) % 3 : (l - 3 + 2) % 3; }

// ------------------------------------------------------------------ sincos
// fp64 sin/cos with a two-constant Cody-Waite reduction done with FMAs.  x - k*PIO2_HI is
// exact (both are multiples of 2^-52 and the result is < 1), the second FMA rounds once, and
// the neglected tail of pi/2 is 1.5e-33*k, so the reduced argument is good to ~6e-17 for any
// |x| < 2^30 -- no Payne-Hanek slow path for the 1e5..1e6 rad phases of a months-long chirp.
// Kernels: Taylor polynomials on |r| <= pi/4 (remainders 8e-20 and 2e-18).
__device__ __forceinline__ void sincos_d(double x, double& s, double& c) {
  const double TWO_OVER_PI = 0.6366197723675814;
  const double PIO2_HI = 1.5707963267948966;
  const double PIO2_LO = 6.123233995736766e-17;
  // round to nearest by adding and subtracting 1.5 * 2^52 (exact for |x 2/pi| < 2^51): two DADDs on the
  // fp64 pipe instead of FRND + F2I on the quarter-rate conversion pipe; the quadrant is in the low
  // bits of the biased sum
  const double SHIFTER = 6755399441055744.0;
  const double kb = fma(x, TWO_OVER_PI, SHIFTER);
  const int q = __double2loint(kb);
  const double kd = kb - SHIFTER;
  double r = fma(-kd, PIO2_HI, x);
  r = fma(-kd, PIO2_LO, r);
  double r2 = r * r;
  // sin r = r + r^3 (-1/3! + r^2/5! - ... + r^14/17!)
  double ps = 2.8114572543455206e-15;
  ps = fma(ps, r2, -7.647163731819816e-13);
  ps = fma(ps, r2, 1.6059043836821613e-10);
  ps = fma(ps, r2, -2.505210838544172e-08);
  ps = fma(ps, r2, 2.7557319223985893e-06);
  ps = fma(ps, r2, -0.0001984126984126984);
  ps = fma(ps, r2, 0.008333333333333333);
  ps = fma(ps, r2, -0.16666666666666666);
  double sr = fma(ps * r2, r, r);
  // cos r = 1 - r^2/2 + r^4 (1/4! - r^2/6! + ... + r^12/16!)
  double pc = 4.779477332387385e-14;
  pc = fma(pc, r2, -1.1470745597729725e-11);
  pc = fma(pc, r2, 2.08767569878681e-09);
  pc = fma(pc, r2, -2.755731922398589e-07);
  pc = fma(pc, r2, 2.48015873015873e-05);
  pc = fma(pc, r2, -0.001388888888888889);
  pc = fma(pc, r2, 0.041666666666666664);
  double cr = fma(pc * r2, r2, fma(-0.5, r2, 1.0));
  double ss = (q & 1) ? cr : sr;
  double cc = (q & 1) ? sr : cr;
  s = (q & 2) ? -ss : ss;
  c = ((q + 1) & 2) ? -cc : cc;
}

// ------------------------------------------------------------------ orbit evaluation
// TABLE: Lagrange interpolation of degree q on the nodes j0..j0+q, j0 = floor(u) - (q-1)/2
// clamped to the table, u = (t - t_tab0)/dt_tab (reading A21); the common part is the centroid.
// WITH_V: also the velocities v[k][xyz] [m/s], the derivative of the same interpolant.
template <bool WITH_V>
__device__ __forceinline__ void orbit_table_eval(const OrbitDev& o, double t, double (&d)[3][3], double (&rc_s)[3],
                                                 double (&v)[3][3]) {
  const int q = o.tab_order;
  const double u = (t - o.t_tab0) * o.inv_dt_tab;
  int j0 = (int)floor(u) - (q - 1) / 2;
  j0 = max(0, min(j0, o.n_tab - q - 1));
  const double x = u - (double)j0;
  double r[3][3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      r[k][j] = 0.0;
      if (WITH_V) v[k][j] = 0.0;
    }
#pragma unroll 1
  for (int i = 0; i <= q; ++i) {
    double c = o.tab_w[i], dc = 0.0;  // c = w_i prod (x - m), dc = its x-derivative (product rule, running)
#pragma unroll 1
    for (int m = 0; m <= q; ++m)
      if (m != i) {
        const double g = x - (double)m;
        if (WITH_V) dc = fma(dc, g, c);
        c *= g;
      }
    const double* row = o.tab + (size_t)(j0 + i) * 9;
    if (WITH_V) dc *= o.inv_dt_tab;
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const double rij = __ldg(row + 3 * k + j);
        r[k][j] = fma(c, rij, r[k][j]);
        if (WITH_V) v[k][j] = fma(dc, rij, v[k][j]);
      }
  }
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    const double c = (r[0][j] + r[1][j] + r[2][j]) * (1.0 / 3.0);
    rc_s[j] = c / C_LIGHT;
#pragma unroll
    for (int k = 0; k < 3; ++k) d[k][j] = r[k][j] - c;
  }
}

// d[k][xyz]: spacecraft positions minus a common part; rc_s: that common part as a light
// travel time [s] per unit direction.  KEPLER1: common part a(cos M, sin M, 0); STATIC: zero
// (d = the positions themselves); TABLE: the centroid.
// WITH_V: also the (full, not split) velocities v[k][xyz] [m/s] (reading A22).
template <bool WITH_V>
__device__ __forceinline__ void orbit_offsets_v(const OrbitDev& o, double t, double (&d)[3][3],
                                                double (&rc_s)[3], double (&v)[3][3]) {
  if (o.kind == 0) {
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        d[k][j] = o.r[k][j];
        if (WITH_V) v[k][j] = 0.0;
      }
    rc_s[0] = rc_s[1] = rc_s[2] = 0.0;
    return;
  }
  if (o.kind == 2) {
    orbit_table_eval<WITH_V>(o, t, d, rc_s, v);
    return;
  }
  double cM, sM;
  double M = fma(o.w, t - o.t_ref, -o.phase0);
  sincos_d(M, sM, cM);
  rc_s[0] = o.a_over_c * cM;
  rc_s[1] = o.a_over_c * sM;
  rc_s[2] = 0.0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    // M_k = M - sigma_k
    double cMk = fma(cM, o.cs[k], sM * o.sn[k]);
    double sMk = fma(sM, o.cs[k], -cM * o.sn[k]);
    // psi_k = M_k + s, s = e sin M_k;  cos psi_k = cMk + dc, sin psi_k = sMk + ds
    double s = o.e * sMk, sh, ch;
    sincos_d(0.5 * s, sh, ch);
    double sins = 2.0 * sh * ch, cosm1 = -2.0 * sh * sh;
    double dc = fma(cMk, cosm1, -sMk * sins);
    double ds = fma(sMk, cosm1, cMk * sins);
    double u1 = dc - o.e;
    double px = fma(o.dci, cMk, o.ci * u1);  // x/a - cos M_k
    double py = fma(o.dbq, sMk, o.bq * ds);  // y/a - sin M_k
    d[k][0] = o.a * fma(o.cs[k], px, -o.sn[k] * py);
    d[k][1] = o.a * fma(o.sn[k], px, o.cs[k] * py);
    d[k][2] = o.a * o.si * (cMk + u1);
    if (WITH_V) {
      // d psi_k/dt = w (1 + e cos M_k);  (x, y, z)' = a (-sin psi ci, bq cos psi, -sin psi si) psi'
      const double aw = o.a * o.w * fma(o.e, cMk, 1.0);
      const double sp = sMk + ds, cp = cMk + dc;
      const double vx = -aw * sp * o.ci, vy = aw * o.bq * cp;
      v[k][0] = fma(o.cs[k], vx, -o.sn[k] * vy);
      v[k][1] = fma(o.sn[k], vx, o.cs[k] * vy);
      v[k][2] = -aw * sp * o.si;
    }
  }
}
__device__ __forceinline__ void orbit_offsets(const OrbitDev& o, double t, double (&d)[3][3],
                                              double (&rc_s)[3]) {
  double v[3][3];
  orbit_offsets_v<false>(o, t, d, rc_s, v);
}

// Light travel times of the six links at time t (link order [1,2,3,-1,-2,-3]).
__device__ __forceinline__ void orbit_arm_times(const OrbitDev& o, double t, double (&L)[6]) {
  if (o.kind == 0) {
#pragma unroll
    for (int l = 0; l < 6; ++l) L[l] = o.L[l];
    return;
  }
  double d[3][3], rc_s[3], v[3][3];
  if (o.tt_order) orbit_offsets_v<true>(o, t, d, rc_s, v);
  else orbit_offsets_v<false>(o, t, d, rc_s, v);
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    const int s = (l + 2) % 3, r = (l + 1) % 3;  // link l+1: sender, receiver
    double dx = d[r][0] - d[s][0], dy = d[r][1] - d[s][1], dz = d[r][2] - d[s][2];
    double dist = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
    double len = dist / C_LIGHT;
    L[l] = len;
    L[l + 3] = len;
    if (o.tt_order) {  // A22: (d/c)(1 + n.v_sender/c); link -(l+1) runs the other way
      const double sc = 1.0 / (dist * C_LIGHT);
      L[l] = fma(len, fma(dx, v[s][0], fma(dy, v[s][1], dz * v[s][2])) * sc, len);
      L[l + 3] = fma(len, -fma(dx, v[r][0], fma(dy, v[r][1], dz * v[r][2])) * sc, len);
    }
  }
}

// ------------------------------------------------------------------ Lagrange stencil
// Array-free ("Horner in node pairs") form of the interpolant.  With the scaled pair factors of
// LagS, Q'_k = rho_k (q + k(1-k)), q = eps (eps - 1), prefix P_k = g prod_{i<k} Q'_i and
//   v_k = (eps+k-1) x_k + (k-eps) x_{1-k},
// the sum  sum_k P_k (prod_{i>k} Q'_i) v_k  is the end value of  T_k = Q'_k T_{k-1} + P_k v_k,
// T_0 = 0:  no prefix array, no suffix chain, 11 fp64 ops per node pair for two series, and so
// few live registers that the tap loads can be issued far ahead of their use.
// HT > 0: half-width known at compile time (fully unrolled); HT = 0: runtime half-width Hrt.
//
// Two ADJACENT output samples a, b = a+1 with the same integer delay: their windows are
// x[e+1-H .. e+H] and x[e+2-H .. e+H+1], so one pass loads 2H+1 taps for both instead of 4H.
// The series is stored split by parity of the element index (xe[i] = x[2i], xo[i] = x[2i+1])
// so that a warp whose lanes own sample pairs (stride 2 elements) reads consecutive 16-byte
// words -- conflict-free LDS.128.  e = element index of tap j = 0 of sample a.
template <int HT>
__device__ __forceinline__ void lagrange_dot2h_x2(double epsa, double epsb, int Hrt, const LagS& ls,
                                                  const double2* __restrict__ xe,
                                                  const double2* __restrict__ xo, int e,
                                                  double (&sp)[2], double (&sc)[2]) {
  const int H = HT > 0 ? HT : Hrt;
  // x[e + o] = (o even ? p0[o/2] : p1[(o-1)/2])
  const double2* p0 = ((e & 1) ? xo : xe) + (e >> 1);
  const double2* p1 = (e & 1) ? xe + (e >> 1) + 1 : xo + (e >> 1);
#define LISA_X(o) (((o) & 1) ? p1[((o) - 1) >> 1] : p0[(o) >> 1])
  const double qa = epsa * (epsa - 1.0), qb = epsb * (epsb - 1.0);
  double Pa = ls.g, Pb = ls.g, Tpa = 0.0, Tca = 0.0, Tpb = 0.0, Tcb = 0.0;
  double2 ucur = LISA_X(1), dprev = ucur;  // x[e+k], x[e+2-k] at k = 1
#pragma unroll
  for (int k = 1; k <= H; ++k) {
    const double2 unext = LISA_X(k + 1), dcur = LISA_X(1 - k);
    const double rho = ls.rho[k - 1], rc = ls.rc[k - 1];
    {  // sample a: taps x[e+k], x[e+1-k]
      const double Q = fma(rho, qa, rc);
      const double t = Pa * epsa;
      const double ck = k == 1 ? t : fma(Pa, (double)(k - 1), t);
      const double cm = fma(Pa, (double)k, -t);
      Tpa = fma(Tpa, Q, fma(ck, ucur.x, cm * dcur.x));
      Tca = fma(Tca, Q, fma(ck, ucur.y, cm * dcur.y));
      Pa *= Q;
    }
    {  // sample b: taps x[e+1+k], x[e+2-k]
      const double Q = fma(rho, qb, rc);
      const double t = Pb * epsb;
      const double ck = k == 1 ? t : fma(Pb, (double)(k - 1), t);
      const double cm = fma(Pb, (double)k, -t);
      Tpb = fma(Tpb, Q, fma(ck, unext.x, cm * dprev.x));
      Tcb = fma(Tcb, Q, fma(ck, unext.y, cm * dprev.y));
      Pb *= Q;
    }
    ucur = unext;
    dprev = dcur;
  }
#undef LISA_X
  sp[0] = Tpa; sc[0] = Tca; sp[1] = Tpb; sc[1] = Tcb;
}

// One sample from the parity-split storage (any element index): the rare path of a sample
// pair whose integer delays differ.  Runtime loop, never unrolled (it is cold code).
__device__ __forceinline__ void lagrange_dot2h_split(double eps, int H, const LagS& ls,
                                                  const double2* __restrict__ xe,
                                                  const double2* __restrict__ xo, int e,
                                                  double& sp, double& sc) {
  const double q = eps * (eps - 1.0);
  double P = ls.g, Tp = 0.0, Tc = 0.0;
#pragma unroll 1
  for (int k = 1; k <= H; ++k) {
    const int iu = e + k, id = e + 1 - k;
    const double2 xk = (iu & 1) ? xo[iu >> 1] : xe[iu >> 1];
    const double2 xm = (id & 1) ? xo[id >> 1] : xe[id >> 1];
    const double Q = fma(ls.rho[k - 1], q, ls.rc[k - 1]);
    const double t = P * eps;
    const double ck = fma(P, (double)(k - 1), t);
    const double cm = fma(P, (double)k, -t);
    Tp = fma(Tp, Q, fma(ck, xk.x, cm * xm.x));
    Tc = fma(Tc, Q, fma(ck, xk.y, cm * xm.y));
    P *= Q;
  }
  sp = Tp;
  sc = Tc;
}

// Same for a single series.
template <int HT>
__device__ __forceinline__ double lagrange_dot1(double eps, int Hrt, const LagW& lw,
                                                const double* __restrict__ x) {
  const int H = HT > 0 ? HT : Hrt;
  double P[HT > 0 ? HT + 1 : MAX_HALF + 1];
  const double q = eps * (eps - 1.0);
  P[1] = 1.0;
#pragma unroll
  for (int k = 1; k < H; ++k) P[k + 1] = P[k] * (q + (double)(k * (1 - k)));
  double S = 1.0, a0 = 0.0, a1 = 0.0;
#pragma unroll
  for (int k = H; k >= 1; --k) {
    double a = (lw.w[k - 1] * P[k]) * S;
    a0 = fma(a * (eps + (double)(k - 1)), x[k], a0);
    a1 = fma(a * ((double)k - eps), x[1 - k], a1);
    S *= q + (double)(k * (1 - k));
  }
  return a0 + a1;
}

#endif  // __CUDACC__

}  // namespace lisa
