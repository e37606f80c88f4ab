// k2_link_response.cu -- S2: h+, hx -> six link responses (Eq. 2.7-2.8, PAPER.md:138-161;
// readings A7, A8, A11 of DESIGN.md), and the link-level laser-noise helper (A12).
//
// One block = K2_T consecutive output samples x a group of up to K2_G walkers; a thread owns
// TWO ADJACENT samples.
//  - The orbit geometry of a sample (spacecraft offsets, arm lengths) does not depend on the
//    walker: it is evaluated once per block into shared memory (geo[field][sample]) and reused
//    by every walker of the group.
//  - Per walker the strain tile is staged in shared memory by cp.async (double buffered) as
//    (h+, hx) pairs, split by parity of the sample index (see lagrange_dot2h_x2).  The tile
//    follows the walker's own 1 AU delay: it starts at n0 - Kc - halo with Kc = rint(Dc(n0)),
//    so its length is K2_T + 2 halo (halo ~ 25 samples) whatever margin_y is.
//  - Per sample pair: nine evaluation times (3 receivers + 6 emitters), each one fused
//    "Lagrange coefficient sweep + two dot products" for both samples of the pair, which
//    share all but one of their taps: 2H+1 shared-memory loads instead of 4H (the one-sample-
//    per-thread version saturated the shared-memory pipe at 98 %, profiles/r1_s3_*.md).
#include "common.cuh"

namespace lisa {

constexpr int K2_T = 256;        // output samples per block
constexpr int K2_THREADS = 128;  // two adjacent samples per thread
constexpr int K2_G = 16;         // walkers per block (upper bound; 32 measured the same)
constexpr int K2_NGEO = 21;      // geometry fields per sample

struct K2Params {
  int B;
  long long N;
  double t0, dt, inv_dt;
  int half;    // (p+1)/2
  int margin;  // margin_y
  int group;   // walkers per block
  int halo;    // tile halo in samples (bound on |D - Kc| + half + slack)
  int up2;     // 1: hplus/hcross are [B][N/2+1] on the 2 dt grid, linearly interpolated while staging (A20)
  const double* hplus;
  const double* hcross;
  const double* lambda;
  const double* beta_sky;
  double* y;
  unsigned int* err;  // sticky device error words (common.cuh)
  OrbitDev orb;
  LagS ls;
};

__device__ __forceinline__ void k2_cp_async8_zfill(void* smem, const void* gmem, bool valid) {
  unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(sa), "l"(gmem), "r"(sz));
}

// 1/x for the geometric factors 1/((1 - k.n_A)(1 - k.n_B)), x in (0, 4]: the hardware seed (MUFU.RCP64H,
// ~23 bits) and two Newton steps, good to one ulp -- a third of the instructions of the IEEE-exact
// division, whose slow-path test and call sit six times in every walker's loop body.
__device__ __forceinline__ double k2_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  r = fma(fma(-x, r, 1.0), r, r);
  r = fma(fma(-x, r, 1.0), r, r);
  return r;
}

// Fractional-delay reads of (h+, hx) for the sample pair (a, b = a+1) at delays
// D = Dc + Dl (samples).  The integer part is decided from the rounded sum, the fraction is
// formed as (K - Dc) - Dl so that the common 1 AU part (up to ~100 samples) does not cost the
// differential delays their low bits.  ea0 = tile element of sample a at zero delay + Kc.
template <int HT>
__device__ __forceinline__ void read_pair2(const double2* __restrict__ xe, const double2* __restrict__ xo,
                                           int elo, int ehi, int ea0, const double (&Dc)[2],
                                           double Dla, double Dlb, const K2Params& p,
                                           double (&vp)[2], double (&vc)[2]) {
  const double Ka = ceil(Dc[0] + Dla), Kb = ceil(Dc[1] + Dlb);
  const double epsa = (Ka - Dc[0]) - Dla, epsb = (Kb - Dc[1]) - Dlb;
  // the halo (sized from host-side bounds on the orbit) must keep every window inside the tile;
  // if it does not, say so (the clamp is for memory safety only: the value is then wrong).
  // One unsigned compare per read on the hot path: ea in [elo, ehi].
  int ea = ea0 - (int)Ka;
  if ((unsigned)(ea - elo) > (unsigned)(ehi - elo)) {
    raise_error(p.err, DEVERR_K2_WINDOW);
    ea = max(elo, min(ea, ehi));
  }
  if (Ka == Kb) {
    lagrange_dot2h_x2<HT>(epsa, epsb, p.half, p.ls, xe, xo, ea, vp, vc);
  } else {  // cold path: the two samples of the pair have different integer delays
    int eb = ea0 + 1 - (int)Kb;
    if (eb < elo || eb > ehi + 1) {
      raise_error(p.err, DEVERR_K2_WINDOW);
      eb = max(elo, min(eb, ehi));
    }
    lagrange_dot2h_split(epsa, p.half, p.ls, xe, xo, ea, vp[0], vc[0]);
    lagrange_dot2h_split(epsb, p.half, p.ls, xe, xo, eb, vp[1], vc[1]);
  }
}

// Walker-independent geometry of the thread's two samples na, na + 1 -> geo[field][sample]
// (fields: 0,1,20 common delay per unit k; 2..10 spacecraft offsets as delays per unit k;
// 11..13 / 14..16 light travel times of links +a / -a; 17..19 reciprocal arm lengths; samples).
template <int KIND>
__device__ __forceinline__ void k2_geometry(const K2Params& p, double* geo, long long na) {
#pragma unroll 1
  for (int c = 0; c < 2; ++c) {
    double* gq = geo + 2 * threadIdx.x + c;
    double d[3][3], rc_s[3], vel[3][3];
    if (p.orb.tt_order) orbit_offsets_v<true>(p.orb, fma((double)(na + c), p.dt, p.t0), d, rc_s, vel);
    else orbit_offsets_v<false>(p.orb, fma((double)(na + c), p.dt, p.t0), d, rc_s, vel);
    const double sc = p.inv_dt / C_LIGHT;
    gq[0 * K2_T] = rc_s[0] * p.inv_dt;   // common (1 AU) delay per unit k (samples)
    gq[1 * K2_T] = rc_s[1] * p.inv_dt;
    gq[20 * K2_T] = rc_s[2] * p.inv_dt;
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j) gq[(2 + 3 * k + j) * K2_T] = d[k][j] * sc;  // offsets as delays per unit k
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int s = link_s(a), r = link_r(a);
      const double dx = d[r][0] - d[s][0], dy = d[r][1] - d[s][1], dz = d[r][2] - d[s][2];
      const double len = sqrt(fma(dx, dx, fma(dy, dy, dz * dz))) * sc;  // arm length in samples
      double Lp = len, Lm = len;  // light travel times of links +a, -a (KEPLER1, TABLE: |r_r - r_s|/c)
      if (KIND != 0 && p.orb.tt_order) {  // A22: (d/c)(1 + n.v_sender/c); link -a runs r -> s
        const double q = sc / (len * C_LIGHT);  // n.v/c = (d.v) q with d in metres, len in samples
        Lp = fma(len, fma(dx, vel[s][0], fma(dy, vel[s][1], dz * vel[s][2])) * q, len);
        Lm = fma(len, -fma(dx, vel[r][0], fma(dy, vel[r][1], dz * vel[r][2])) * q, len);
      }
      gq[(11 + a) * K2_T] = KIND == 0 ? p.orb.L[a] * p.inv_dt : Lp;
      gq[(14 + a) * K2_T] = KIND == 0 ? p.orb.L[a + 3] * p.inv_dt : Lm;
      gq[(17 + a) * K2_T] = 1.0 / len;  // n_a = (offset_r - offset_s) / len
    }
  }
}

template <int HT, int KIND>
__global__ void __launch_bounds__(K2_THREADS, 4) k2_link_response(const K2Params p) {
  extern __shared__ double2 smem2[];  // [2 buffers][even, odd][LE] strain tiles, then geo[K2_NGEO][K2_T]
  __shared__ double sky[K2_G][9];     // k, u, v of the block's walkers (Eq. 2.7)
  __shared__ int Kc[K2_G];            // rint of the common 1 AU delay at the block's first sample
  const int R = p.margin;
  const int tile_len = K2_T + 2 * p.halo;
  const int LE = (tile_len + 1) / 2 + 1;
  const long long n0 = (long long)blockIdx.x * K2_T;
  const int w0 = blockIdx.y * p.group;
  const int nw = min(p.group, p.B - w0);
  double* geo = reinterpret_cast<double*>(smem2 + 4 * (size_t)LE);
#define GEO2(f) (*reinterpret_cast<const double2*>(geo + (f) * K2_T + 2 * threadIdx.x))

  if (threadIdx.x < nw) {
    double sl, cl, sb, cb;
    sincos_d(p.lambda[w0 + threadIdx.x], sl, cl);
    sincos_d(p.beta_sky[w0 + threadIdx.x], sb, cb);
    double* s = sky[threadIdx.x];
    s[0] = -cb * cl; s[1] = -cb * sl; s[2] = -sb;  // k
    s[3] = sl;       s[4] = -cl;      s[5] = 0.0;  // u
    s[6] = -sb * cl; s[7] = -sb * sl; s[8] = cb;   // v
    double Dc0 = 0.0;
    if (KIND == 1) {
      double sM, cM;
      sincos_d(fma(p.orb.w, fma((double)n0, p.dt, p.t0) - p.orb.t_ref, -p.orb.phase0), sM, cM);
      Dc0 = p.orb.a_over_c * p.inv_dt * fma(s[0], cM, s[1] * sM);
    } else if (KIND == 2) {
      double d0[3][3], rc0[3];
      orbit_offsets(p.orb, fma((double)n0, p.dt, p.t0), d0, rc0);
      Dc0 = p.inv_dt * fma(s[0], rc0[0], fma(s[1], rc0[1], s[2] * rc0[2]));
    }
    Kc[threadIdx.x] = __double2int_rn(Dc0);
  }
  __syncthreads();

  auto prefetch = [&](int w, int buf) {
    double2* dst = smem2 + (size_t)buf * 2 * LE;
    const long long g0 = n0 - Kc[w] - p.halo;
    if (p.up2) {
      // strain sampled every 2 dt, linearly interpolated to the dt grid
      const long long Nc = p.N / 2 + 1;
      const double* hp = p.hplus + (size_t)(w0 + w) * Nc;
      const double* hc = p.hcross + (size_t)(w0 + w) * Nc;
      for (int i = threadIdx.x; i < tile_len; i += K2_THREADS) {
        const long long g = g0 + i;
        double2 v = make_double2(0.0, 0.0);
        if (g >= 0 && g < p.N) {
          const long long c = g >> 1;
          v = make_double2(hp[c], hc[c]);
          if (g & 1) v = make_double2((v.x + hp[c + 1]) * 0.5, (v.y + hc[c + 1]) * 0.5);
        }
        dst[(i & 1) * LE + (i >> 1)] = v;
      }
      asm volatile("cp.async.commit_group;\n" ::);  // keeps the group count of the cp.async path
      return;
    }
    const double* hp = p.hplus + (size_t)(w0 + w) * p.N;
    const double* hc = p.hcross + (size_t)(w0 + w) * p.N;
    for (int i = threadIdx.x; i < tile_len; i += K2_THREADS) {
      const long long g = g0 + i;
      const bool ok = g >= 0 && g < p.N;
      const long long src = ok ? g : 0;
      double2* d = dst + (i & 1) * LE + (i >> 1);
      k2_cp_async8_zfill(&d->x, hp + src, ok);
      k2_cp_async8_zfill(&d->y, hc + src, ok);
    }
    asm volatile("cp.async.commit_group;\n" ::);
  };
  prefetch(0, 0);

  // ---- walker-independent geometry of this thread's two samples -> geo[field][sample]
  const long long na = n0 + 2 * threadIdx.x;
  k2_geometry<KIND>(p, geo, na);
  const bool act[2] = {na >= R && na < p.N - R, na + 1 >= R && na + 1 < p.N - R};
  const bool vec_store = (p.N & 1) == 0;
  const int elo = p.half - 1, ehi = tile_len - 2 - p.half;

  for (int w = 0; w < nw; ++w) {
    const int buf = w & 1;
    asm volatile("cp.async.wait_group 0;\n" ::);
    // ONE barrier per walker: the tile of walker w (and, first time round, geo[]) is visible to everyone,
    // and everyone is done reading the other buffer (walker w-1), so it can be refilled right away
    __syncthreads();
    if (w + 1 < nw) prefetch(w + 1, buf ^ 1);
    double* yb = p.y + (size_t)(w0 + w) * 6 * p.N + na;
    auto store2 = [&](int l, double v0, double v1) {
      double* dst = yb + (size_t)l * p.N;
      v0 = act[0] ? v0 : 0.0;
      v1 = act[1] ? v1 : 0.0;
      if (vec_store) {
        if (na < p.N) *reinterpret_cast<double2*>(dst) = make_double2(v0, v1);
      } else {
        if (na < p.N) dst[0] = v0;
        if (na + 1 < p.N) dst[1] = v1;
      }
    };
    if (act[0] || act[1]) {
      const double2* xe = smem2 + (size_t)buf * 2 * LE;
      const double2* xo = xe + LE;
      const int ea0 = 2 * threadIdx.x + p.halo + Kc[w];
      const double* s = sky[w];
      const double kx = s[0], ky = s[1], kz = s[2];
      const double ux = s[3], uy = s[4];  // uz = 0
      const double vx = s[6], vy = s[7], vz = s[8];
      double Dc[2];
      {
        const double2 g0 = GEO2(0), g1 = GEO2(1);
        Dc[0] = fma(kx, g0.x, ky * g1.x);
        Dc[1] = fma(kx, g0.y, ky * g1.y);
        if (KIND == 2) {  // the centroid of a tabulated orbit has a z component
          const double2 g2 = GEO2(20);
          Dc[0] = fma(kz, g2.x, Dc[0]);
          Dc[1] = fma(kz, g2.y, Dc[1]);
        }
      }
      {
        // Receiver-major order: iteration k handles spacecraft k as RECEIVER -- its reception-time read
        // and the two links it receives: link +(k+2) from spacecraft k+1 and link -(k+1) from spacecraft
        // k+2 (indices mod 3).  The offsets of the three spacecraft are re-read from geo[] by runtime
        // field index each time, so no per-slot state lives across iterations: no slot rotation, and
        // ~50 fewer live registers during the sweeps (the price: arm projections are formed per link
        // instead of per arm, +75 fp64 operations per walker-sample).
#pragma unroll 1
        for (int k = 0; k < 3; ++k) {
          const int k1 = k == 2 ? 0 : k + 1, k2 = k == 0 ? 2 : k - 1;
          double kd0[2], DsA[2], DsB[2], xpA[2], xcA[2], fA[2], xpB[2], xcB[2], fB[2];
          {
            const double2 rx = GEO2(2 + 3 * k), ry = GEO2(3 + 3 * k), rz = GEO2(4 + 3 * k);
            const double2 ax = GEO2(2 + 3 * k1), ay = GEO2(3 + 3 * k1), az = GEO2(4 + 3 * k1);
            const double2 bx = GEO2(2 + 3 * k2), by = GEO2(3 + 3 * k2), bz = GEO2(4 + 3 * k2);
            const double2 LA = GEO2(11 + k2), ilA = GEO2(17 + k2);  // link +(k+2): k1 -> k
            const double2 LB = GEO2(14 + k1), ilB = GEO2(17 + k1);  // link -(k+1): k2 -> k
            const double rxs[2] = {rx.x, rx.y}, rys[2] = {ry.x, ry.y}, rzs[2] = {rz.x, rz.y};
            const double eAx[2] = {rx.x - ax.x, rx.y - ax.y}, eAy[2] = {ry.x - ay.x, ry.y - ay.y}, eAz[2] = {rz.x - az.x, rz.y - az.y};
            const double eBx[2] = {rx.x - bx.x, rx.y - bx.y}, eBy[2] = {ry.x - by.x, ry.y - by.y}, eBz[2] = {rz.x - bz.x, rz.y - bz.y};
            const double LAs[2] = {LA.x, LA.y}, LBs[2] = {LB.x, LB.y}, ilAs[2] = {ilA.x, ilA.y}, ilBs[2] = {ilB.x, ilB.y};
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              kd0[c] = fma(kx, rxs[c], fma(ky, rys[c], kz * rzs[c]));
              const double keA = fma(kx, eAx[c], fma(ky, eAy[c], kz * eAz[c]));  // k.(r_k - r_k1)
              const double keB = fma(kx, eBx[c], fma(ky, eBy[c], kz * eBz[c]));
              DsA[c] = LAs[c] + (kd0[c] - keA);  // L + k.r_sender
              DsB[c] = LBs[c] + (kd0[c] - keB);
              const double unA = fma(ux, eAx[c], uy * eAy[c]) * ilAs[c], vnA = fma(vx, eAx[c], fma(vy, eAy[c], vz * eAz[c])) * ilAs[c];
              const double unB = fma(ux, eBx[c], uy * eBy[c]) * ilBs[c], vnB = fma(vx, eBx[c], fma(vy, eBy[c], vz * eBz[c])) * ilBs[c];
              xpA[c] = fma(unA, unA, -vnA * vnA);
              xcA[c] = 2.0 * unA * vnA;
              xpB[c] = fma(unB, unB, -vnB * vnB);
              xcB[c] = 2.0 * unB * vnB;
              const double omA = 1.0 - keA * ilAs[c], omB = 1.0 - keB * ilBs[c];  // 1 - k.n of each link
              const double inv = 0.5 * k2_rcp(omA * omB);
              fA[c] = omB * inv;
              fB[c] = omA * inv;
            }
          }
          double hpr[2], hcr[2], hps[2], hcs[2];
          read_pair2<HT>(xe, xo, elo, ehi, ea0, Dc, kd0[0], kd0[1], p, hpr, hcr);
          read_pair2<HT>(xe, xo, elo, ehi, ea0, Dc, DsA[0], DsA[1], p, hps, hcs);
          store2(k2, fma(xpA[0], hps[0] - hpr[0], xcA[0] * (hcs[0] - hcr[0])) * fA[0],
                 fma(xpA[1], hps[1] - hpr[1], xcA[1] * (hcs[1] - hcr[1])) * fA[1]);
          read_pair2<HT>(xe, xo, elo, ehi, ea0, Dc, DsB[0], DsB[1], p, hps, hcs);
          store2(k1 + 3, fma(xpB[0], hps[0] - hpr[0], xcB[0] * (hcs[0] - hcr[0])) * fB[0],
                 fma(xpB[1], hps[1] - hpr[1], xcB[1] * (hcs[1] - hcr[1])) * fB[1]);
        }
      }
    } else {
#pragma unroll
      for (int l = 0; l < 6; ++l) store2(l, 0.0, 0.0);
    }
  }
#undef GEO2
}

// ---------------------------------------------------------------- linear interpolation (p = 1)
// The paper's own GPU code interpolates linearly.  With two taps per read there
// is nothing to stage: each thread reads its taps straight from global memory (adjacent
// threads read adjacent samples; the nine reads of a walker fall within ~100 samples, so they
// hit L1), the walker loop has no barrier, all nine reads are unrolled, and a block serves up
// to K2L_G walkers with one evaluation of the orbit geometry.
constexpr int K2L_G = 32;

__device__ __forceinline__ void read_pair_lin(const double* __restrict__ hp, const double* __restrict__ hc,
                                              long long na, long long N, const double (&Dc)[2], double Dla,
                                              double Dlb, unsigned int* err, double (&vp)[2], double (&vc)[2]) {
  const double Ka = ceil(Dc[0] + Dla), Kb = ceil(Dc[1] + Dlb);
  const double epsa = (Ka - Dc[0]) - Dla, epsb = (Kb - Dc[1]) - Dlb;
  // taps j = 0, 1: x[n - K], x[n - K + 1] with weights 1 - eps, eps.  margin_y (checked on the host
  // against bounds on the orbit) keeps every window inside [0, N); if it does not, say so (the
  // clamp is for memory safety only).  The odd-N tail sample na + 1 = N is never stored.
  long long ia = na - (long long)Ka, ib = na + 1 - (long long)Kb;
  if (ia < 0 || ia > N - 2 || ib < 0 || ib > N - 1) {
    raise_error(err, DEVERR_K2_WINDOW);
    ia = max(0LL, min(ia, N - 2));
  }
  ib = max(0LL, min(ib, N - 2));
  const double a0 = __ldg(hp + ia), a1 = __ldg(hp + ia + 1);
  const double c0 = __ldg(hc + ia), c1 = __ldg(hc + ia + 1);
  const bool shared_tap = ib == ia + 1;  // same integer delay: sample b starts on a's second tap
  const double b0 = shared_tap ? a1 : __ldg(hp + ib), d0 = shared_tap ? c1 : __ldg(hc + ib);
  const double b1 = __ldg(hp + ib + 1), d1 = __ldg(hc + ib + 1);
  vp[0] = fma(epsa, a1 - a0, a0);
  vc[0] = fma(epsa, c1 - c0, c0);
  vp[1] = fma(epsb, b1 - b0, b0);
  vc[1] = fma(epsb, d1 - d0, d0);
}

template <int KIND>
__global__ void __launch_bounds__(K2_THREADS, 4) k2_link_response_lin(const K2Params p) {
  extern __shared__ double geo[];    // [K2_NGEO][K2_T]; a thread only ever reads its own two samples
  __shared__ double sky[K2L_G][9];   // k, u, v of the block's walkers (Eq. 2.7)
  const int R = p.margin;
  const long long n0 = (long long)blockIdx.x * K2_T;
  const int w0 = blockIdx.y * p.group;
  const int nw = min(p.group, p.B - w0);
#define GEO2(f) (*reinterpret_cast<const double2*>(geo + (f) * K2_T + 2 * threadIdx.x))
  if (threadIdx.x < nw) {
    double sl, cl, sb, cb;
    sincos_d(p.lambda[w0 + threadIdx.x], sl, cl);
    sincos_d(p.beta_sky[w0 + threadIdx.x], sb, cb);
    double* s = sky[threadIdx.x];
    s[0] = -cb * cl; s[1] = -cb * sl; s[2] = -sb;  // k
    s[3] = sl;       s[4] = -cl;      s[5] = 0.0;  // u
    s[6] = -sb * cl; s[7] = -sb * sl; s[8] = cb;   // v
  }
  const long long na = n0 + 2 * threadIdx.x;
  k2_geometry<KIND>(p, geo, na);
  __syncthreads();
  const bool act[2] = {na >= R && na < p.N - R, na + 1 >= R && na + 1 < p.N - R};
  const bool vec_store = (p.N & 1) == 0;
  if (na >= p.N) return;

  for (int w = 0; w < nw; ++w) {
    const double* hp = p.hplus + (size_t)(w0 + w) * p.N;
    const double* hc = p.hcross + (size_t)(w0 + w) * p.N;
    double* yb = p.y + (size_t)(w0 + w) * 6 * p.N + na;
    auto store2 = [&](int l, double v0, double v1) {
      double* dst = yb + (size_t)l * p.N;
      v0 = act[0] ? v0 : 0.0;
      v1 = act[1] ? v1 : 0.0;
      if (vec_store) {
        *reinterpret_cast<double2*>(dst) = make_double2(v0, v1);
      } else {
        dst[0] = v0;
        if (na + 1 < p.N) dst[1] = v1;
      }
    };
    if (!(act[0] || act[1])) {
#pragma unroll
      for (int l = 0; l < 6; ++l) store2(l, 0.0, 0.0);
      continue;
    }
    const double* s = sky[w];
    const double kx = s[0], ky = s[1], kz = s[2];
    const double ux = s[3], uy = s[4];  // uz = 0
    const double vx = s[6], vy = s[7], vz = s[8];
    double Dc[2];
    {
      const double2 g0 = GEO2(0), g1 = GEO2(1);
      Dc[0] = fma(kx, g0.x, ky * g1.x);
      Dc[1] = fma(kx, g0.y, ky * g1.y);
      if (KIND == 2) {
        const double2 g2 = GEO2(20);
        Dc[0] = fma(kz, g2.x, Dc[0]);
        Dc[1] = fma(kz, g2.y, Dc[1]);
      }
    }
    double kd[3][2], ud[3][2], vd[3][2], hpr[3][2], hcr[3][2];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const double2 dx = GEO2(2 + 3 * k), dy = GEO2(3 + 3 * k), dz = GEO2(4 + 3 * k);
      kd[k][0] = fma(kx, dx.x, fma(ky, dy.x, kz * dz.x));
      kd[k][1] = fma(kx, dx.y, fma(ky, dy.y, kz * dz.y));
      ud[k][0] = fma(ux, dx.x, uy * dy.x);
      ud[k][1] = fma(ux, dx.y, uy * dy.y);
      vd[k][0] = fma(vx, dx.x, fma(vy, dy.x, vz * dz.x));
      vd[k][1] = fma(vx, dx.y, fma(vy, dy.y, vz * dz.y));
      read_pair_lin(hp, hc, na, p.N, Dc, kd[k][0], kd[k][1], p.err, hpr[k], hcr[k]);  // h(t - k.r_k/c)
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {  // links a and -a share x+, xx and have opposite n
      const int sd = link_s(a), rc = link_r(a);
      const double2 Lp = GEO2(11 + a), Lm = GEO2(14 + a), il = GEO2(17 + a);
      const double ila[2] = {il.x, il.y};
      double xp[2], xc2[2], fp[2], fm[2];
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const double un = (ud[rc][c] - ud[sd][c]) * ila[c];
        const double vn = (vd[rc][c] - vd[sd][c]) * ila[c];
        const double kn = (kd[rc][c] - kd[sd][c]) * ila[c];
        xp[c] = fma(un, un, -vn * vn);
        xc2[c] = 2.0 * un * vn;
        const double om = 1.0 - kn, opl = 1.0 + kn;
        const double inv = 0.5 * k2_rcp(om * opl);
        fp[c] = opl * inv;
        fm[c] = om * inv;
      }
      double hps[2], hcs[2];
      read_pair_lin(hp, hc, na, p.N, Dc, Lp.x + kd[sd][0], Lp.y + kd[sd][1], p.err, hps, hcs);  // link +a: s -> r
      store2(a, fma(xp[0], hps[0] - hpr[rc][0], xc2[0] * (hcs[0] - hcr[rc][0])) * fp[0],
             fma(xp[1], hps[1] - hpr[rc][1], xc2[1] * (hcs[1] - hcr[rc][1])) * fp[1]);
      read_pair_lin(hp, hc, na, p.N, Dc, Lm.x + kd[rc][0], Lm.y + kd[rc][1], p.err, hps, hcs);  // link -a: r -> s
      store2(a + 3, fma(xp[0], hps[0] - hpr[sd][0], xc2[0] * (hcs[0] - hcr[sd][0])) * fm[0],
             fma(xp[1], hps[1] - hpr[sd][1], xc2[1] * (hcs[1] - hcr[sd][1])) * fm[1]);
    }
  }
#undef GEO2
}

template <int KIND>
static int launch_k2_lin_kind(const K2Params& p, cudaStream_t st) {
  const size_t smem = (size_t)K2_NGEO * K2_T * sizeof(double);
  dim3 grid((unsigned)((p.N + K2_T - 1) / K2_T), (unsigned)((p.B + p.group - 1) / p.group));
  k2_link_response_lin<KIND><<<grid, K2_THREADS, smem, st>>>(p);
  LISA_LAUNCH_CHECK("k2_link_response_lin");
  return LISA_TD_OK;
}
static int launch_k2_lin(const K2Params& p, cudaStream_t st) {
  if (p.orb.kind == 0) return launch_k2_lin_kind<0>(p, st);
  if (p.orb.kind == 2) return launch_k2_lin_kind<2>(p, st);
  return launch_k2_lin_kind<1>(p, st);
}

// A12: y_l[n] = p(n - L_l(t_n)/dt) - p[n].  Small helper kernel, reads p from global memory.
struct LaserParams {
  long long N;
  double t0, dt, inv_dt;
  int half;
  long long margin;
  const double* p;
  double* y;
  unsigned int* err;
  OrbitDev orb;
  LagW lw;
};

__global__ void __launch_bounds__(256) k_laser_links(const LaserParams q) {
  const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= q.N) return;
  if (n < q.margin || n >= q.N - q.margin) {
    for (int l = 0; l < 6; ++l) q.y[(size_t)l * q.N + n] = 0.0;
    return;
  }
  double L[6];
  orbit_arm_times(q.orb, fma((double)n, q.dt, q.t0), L);
  for (int l = 0; l < 6; ++l) {
    const double D = L[l] * q.inv_dt;
    const double Kf = ceil(D);
    const double eps = Kf - D;
    long long b = n - (long long)Kf;
    if (b < q.half - 1 || b > q.N - 1 - q.half) {  // the margin did not cover the delay after all
      raise_error(q.err, DEVERR_LASER_WINDOW);
      b = max((long long)(q.half - 1), min(b, q.N - 1 - q.half));
    }
    q.y[(size_t)l * q.N + n] = lagrange_dot1<0>(eps, q.half, q.lw, q.p + b) - q.p[n];
  }
}

template <int HT>
static int launch_k2(const K2Params& p, cudaStream_t st) {
  const int tile_len = K2_T + 2 * p.halo;
  const size_t smem = (size_t)4 * ((tile_len + 1) / 2 + 1) * sizeof(double2) + (size_t)K2_NGEO * K2_T * sizeof(double);
  if (smem > 220 * 1024) return set_error(LISA_TD_EINVAL, "link_response: delay spread of %d samples too large for the shared-memory tile", p.halo);
  dim3 grid((unsigned)((p.N + K2_T - 1) / K2_T), (unsigned)((p.B + p.group - 1) / p.group));
  if (p.orb.kind == 0) {
    LISA_CUDA(cudaFuncSetAttribute(k2_link_response<HT, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k2_link_response<HT, 0><<<grid, K2_THREADS, smem, st>>>(p);
  } else if (p.orb.kind == 2) {
    LISA_CUDA(cudaFuncSetAttribute(k2_link_response<HT, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k2_link_response<HT, 2><<<grid, K2_THREADS, smem, st>>>(p);
  } else {
    LISA_CUDA(cudaFuncSetAttribute(k2_link_response<HT, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k2_link_response<HT, 1><<<grid, K2_THREADS, smem, st>>>(p);
  }
  LISA_LAUNCH_CHECK("k2_link_response");
  return LISA_TD_OK;
}


int run_link_response(int B, long long N, double t0, double dt, int order, long long margin_y,
                      const double* hplus, const double* hcross, const double* lambda,
                      const double* beta_sky, const OrbitDev& orb, double* y, cudaStream_t st, int up2) {
  K2Params p;
  p.up2 = up2;
  p.B = B; p.N = N; p.t0 = t0; p.dt = dt; p.inv_dt = 1.0 / dt;
  p.half = (order + 1) / 2; p.margin = (int)margin_y;
  p.hplus = hplus; p.hcross = hcross; p.lambda = lambda; p.beta_sky = beta_sky; p.y = y;
  p.orb = orb;
  p.err = device_error_words();
  p.group = B < K2_G ? B : K2_G;
  // |K - Kc| <= |Dl| + drift of Dc over the tile + 1.5; the pair window adds half + 1
  p.halo = (int)ceil((orb.max_off_over_c + orb.max_L) / dt + orb.max_dc_rate * K2_T + 1.5) + p.half + 2;
  make_lags(order, &p.ls);
  const bool generic = dispatch_mode() == 1;
  if (!generic && p.half == 1 && !up2) {  // the paper's linear interpolation: its own kernel
    p.group = B < K2L_G ? B : K2L_G;
    return launch_k2_lin(p, st);
  }
  if (!generic) {
    switch (p.half) {
      case 1: return launch_k2<1>(p, st);
      case 2: return launch_k2<2>(p, st);
      case 4: return launch_k2<4>(p, st);
      case 8: return launch_k2<8>(p, st);
      case 16: return launch_k2<16>(p, st);
      default: break;
    }
  }
  return launch_k2<0>(p, st);
}

int run_laser_links(long long N, double t0, double dt, int order, long long margin,
                    const double* pser, const OrbitDev& orb, double* y, cudaStream_t st) {
  LaserParams q;
  q.N = N; q.t0 = t0; q.dt = dt; q.inv_dt = 1.0 / dt; q.half = (order + 1) / 2;
  q.margin = margin; q.p = pser; q.y = y; q.orb = orb; q.err = device_error_words();
  make_lagw(order, &q.lw);
  k_laser_links<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(q);
  LISA_LAUNCH_CHECK("k_laser_links");
  return LISA_TD_OK;
}

}  // namespace lisa
