// k1_modes_to_pol.cu -- S1: co-precessing modes -> h+, hx by the paper's single-sum form
// (Eq. 2.4-2.6) with readings A1-A6 of DESIGN.md:
//
//   h+ - i hx = e^{2 i psi} sum_modes N_l [ h_lm frakD^l_{m,2}(Q) + (-1)^l conj(h_lm) frakD^l_{-m,2}(Q) ],
//   h_lm = amp e^{-i phase},  N_l = sqrt((2l+1)/4pi),
//   Q = Q(alpha,beta,gamma)(t) * Q(euler0) * Q(phi, iota, 0)          (one composed rotation),
//   Q(a,b,g) = (Qa, Qb) = (cos(b/2) e^{i(a+g)/2}, sin(b/2) e^{-i(a-g)/2})   (Eq. 2.5 / sqrt 2, A3).
//
// Eq. 2.6 (with A4) is used in its division-free polynomial form (A5): for row m' and column 2
//   frakD^l_{m',2} = PA(m'+2) PB(2-m') sum_rho coef_rho A^{eA0-i} B^{eB0+i},  A=|Qa|^2, B=|Qb|^2,
//   PA(k) = Qa^k (k>=0) or conj(Qa)^{-k},   PB(k) = Qb^k or conj(Qb)^{-k},
// so nothing is divided by |Qa|^2 when the total beta reaches pi.  The host turns the mode
// list into such "rows" (two per mode, one for m = 0); the kernel evaluates them.
#include <math.h>

#include "common.cuh"

namespace lisa {

constexpr int K1_MAX_MODES = 16;
constexpr int K1_MAX_ROWS = 2 * K1_MAX_MODES;
constexpr int K1_MAX_TERMS = 7;  // rho range of column 2 for l <= 8
constexpr int K1_PMAX = 10;      // largest power of Qa / Qb: l + 2
constexpr int K1_EMAX = 8;       // largest power of A / B
constexpr int K1_THREADS = 256;
constexpr int K1_PER_THREAD = 4;

struct K1Row {
  short mode, conj, ka, kb, eA0, eB0, nterms, pad;
  double coef[K1_MAX_TERMS];
};
struct K1Params {
  int B;
  long long N;
  int n_modes, n_rows, twisted, have_e0;
  const double *amp, *phase, *alpha, *beta, *gamma, *iota, *phi, *psi, *euler0;
  double *hplus, *hcross;
  K1Row row[K1_MAX_ROWS];
};

struct cplx {
  double re, im;
};
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return {fma(a.re, b.re, -a.im * b.im), fma(a.re, b.im, a.im * b.re)};
}
__device__ __forceinline__ cplx cconj(cplx a) { return {a.re, -a.im}; }

struct quat {
  cplx a, b;
};
__device__ __forceinline__ quat quat_from_euler(double al, double be, double ga) {
  // sin/cos of (al +- ga)/2 by angle addition from al/2 and ga/2: forming al + ga first would
  // round at ulp(|al|+|ga|) (1e-13 rad after a few hundred radians of precession).
  double sb, cb, sa, ca, sg, cg;
  sincos_d(0.5 * be, sb, cb);
  sincos_d(0.5 * al, sa, ca);
  sincos_d(0.5 * ga, sg, cg);
  const double cp = fma(ca, cg, -sa * sg), sp = fma(sa, cg, ca * sg);
  const double cm = fma(ca, cg, sa * sg), sm = fma(sa, cg, -ca * sg);
  return {{cb * cp, cb * sp}, {sb * cm, -sb * sm}};
}
// consecutive rotations R_p R_q:  (pa qa - conj(pb) qb,  pb qa + conj(pa) qb)
__device__ __forceinline__ quat quat_mul(quat p, quat q) {
  cplx t1 = cmul(p.a, q.a), t2 = cmul(cconj(p.b), q.b);
  cplx t3 = cmul(p.b, q.a), t4 = cmul(cconj(p.a), q.b);
  return {{t1.re - t2.re, t1.im - t2.im}, {t3.re + t4.re, t3.im + t4.im}};
}

struct PowTables {
  cplx qa[K1_PMAX + 1], qb[K1_PMAX + 1];
  double A[K1_EMAX + 1], B[K1_EMAX + 1];
};
__device__ __forceinline__ void build_tables(const quat& Q, PowTables& T) {
  T.qa[0] = {1.0, 0.0};
  T.qb[0] = {1.0, 0.0};
  T.A[0] = 1.0;
  T.B[0] = 1.0;
  const double A = fma(Q.a.re, Q.a.re, Q.a.im * Q.a.im);
  const double B = fma(Q.b.re, Q.b.re, Q.b.im * Q.b.im);
#pragma unroll
  for (int k = 1; k <= K1_PMAX; ++k) {
    T.qa[k] = cmul(T.qa[k - 1], Q.a);
    T.qb[k] = cmul(T.qb[k - 1], Q.b);
  }
#pragma unroll
  for (int k = 1; k <= K1_EMAX; ++k) {
    T.A[k] = T.A[k - 1] * A;
    T.B[k] = T.B[k - 1] * B;
  }
}
// N_l (+-)^l frakD^l_{m',2}(Q) of one row
__device__ __forceinline__ cplx row_weight(const K1Row& r, const PowTables& T) {
  cplx pa = r.ka >= 0 ? T.qa[r.ka] : cconj(T.qa[-r.ka]);
  cplx pb = r.kb >= 0 ? T.qb[r.kb] : cconj(T.qb[-r.kb]);
  double poly = 0.0;
  for (int i = 0; i < r.nterms; ++i) poly = fma(r.coef[i], T.A[r.eA0 - i] * T.B[r.eB0 + i], poly);
  cplx w = cmul(pa, pb);
  return {w.re * poly, w.im * poly};
}

__global__ void __launch_bounds__(K1_THREADS) k1_modes_to_pol(const K1Params p) {
  __shared__ quat Qc;             // Q(euler0) * Q(phi, iota, 0) of this walker
  __shared__ double rot[2];       // cos 2 psi, sin 2 psi
  __shared__ cplx Wc[K1_MAX_ROWS];  // aligned-spin case: constant row weights
  const int b = blockIdx.y;
  if (threadIdx.x == 0) {
    quat q = quat_from_euler(p.phi[b], p.iota[b], 0.0);  // footnote 1
    if (p.have_e0)
      q = quat_mul(quat_from_euler(p.euler0[3 * b], p.euler0[3 * b + 1], p.euler0[3 * b + 2]), q);
    Qc = q;
    double s2, c2;
    sincos_d(2.0 * p.psi[b], s2, c2);
    rot[0] = c2;
    rot[1] = s2;
  }
  __syncthreads();
  if (!p.twisted) {
    if (threadIdx.x < p.n_rows) {
      PowTables T;
      build_tables(Qc, T);
      Wc[threadIdx.x] = row_weight(p.row[threadIdx.x], T);
    }
    __syncthreads();
  }
  const size_t bN = (size_t)b * p.N;
  const double* amp = p.amp + bN * p.n_modes;
  const double* pha = p.phase + bN * p.n_modes;
  const long long n_base = (long long)blockIdx.x * (K1_THREADS * K1_PER_THREAD);
  for (int it = 0; it < K1_PER_THREAD; ++it) {
    const long long n = n_base + it * K1_THREADS + threadIdx.x;
    if (n >= p.N) break;
    PowTables T;
    if (p.twisted) {
      quat q = quat_mul(quat_from_euler(p.alpha[bN + n], p.beta[bN + n], p.gamma[bN + n]), Qc);
      build_tables(q, T);
    }
    double Hre = 0.0, Him = 0.0;
    for (int r = 0; r < p.n_rows; ++r) {
      const K1Row& row = p.row[r];
      const int k = row.mode;
      // rows of one mode are adjacent; the sincos is recomputed only when the mode changes
      double s, c;
      const double a = amp[(size_t)k * p.N + n];
      sincos_d(pha[(size_t)k * p.N + n], s, c);
      // h = a (c - i s);  conj row uses a (c + i s)
      const double hre = a * c, him = row.conj ? a * s : -a * s;
      cplx w = p.twisted ? row_weight(row, T) : Wc[r];
      Hre += fma(hre, w.re, -him * w.im);
      Him += fma(hre, w.im, him * w.re);
      if (r + 1 < p.n_rows && p.row[r + 1].mode == k) {  // the -m partner: reuse a, s, c
        ++r;
        const K1Row& row2 = p.row[r];
        const double him2 = row2.conj ? a * s : -a * s;
        cplx w2 = p.twisted ? row_weight(row2, T) : Wc[r];
        Hre += fma(hre, w2.re, -him2 * w2.im);
        Him += fma(hre, w2.im, him2 * w2.re);
      }
    }
    // e^{2 i psi};  h+ = Re H, hx = -Im H
    p.hplus[bN + n] = fma(Hre, rot[0], -Him * rot[1]);
    p.hcross[bN + n] = -fma(Hre, rot[1], Him * rot[0]);
  }
}

// ---------------------------------------------------------------- five-mode fast path
// For the paper's mode set {(2,2),(2,1),(3,3),(4,4),(5,5)} ("the 5-mode model")
// and any subset of it, every frakD^l_{+-m,2} is a monomial in Qa, Qb and their conjugates.
// With z = Qa conj(Qb):
//   N2 D^2_{2,2} = N2 Qa^4          N2 D^2_{-2,2} = N2 Qb^4
//   N2 D^2_{1,2} = 2 N2 Qa^3 Qb     N2 D^2_{-1,2} = 2 N2 Qa Qb^3
//   Nl D^l_{l,2} = c_l Qa^4 z^{l-2} (-)^l Nl D^l_{-l,2} = c_l Qb^4 conj(z)^{l-2},  l = 3,4,5
//   c3 = -sqrt(6) N3, c4 = 2 sqrt(7) N4, c5 = -sqrt(120) N5
// so  H = Qa^4 G + Qb^4 conj(G) + 2 N2 Qa Qb (Qa^2 h21 + Qb^2 conj(h21)),
//     G = N2 h22 + z (c3 h33 + z (c4 h44 + z c5 h55)).
// Everything stays in registers (the generic kernel keeps power tables in local memory).
struct K1FastParams {
  int B;
  long long N;
  int n_modes, twisted, have_e0;
  int idx[5];  // position of (2,2),(2,1),(3,3),(4,4),(5,5) in the mode list, -1 = absent
  double c22, c21, c33, c44, c55;
  const double *amp, *phase, *alpha, *beta, *gamma, *iota, *phi, *psi, *euler0;
  double *hplus, *hcross;
};

struct K1Pre {
  cplx Fa, Fb, z, qa2, qb2, qab;
};
__device__ __forceinline__ K1Pre k1_pre(const quat& q) {
  K1Pre r;
  r.qa2 = cmul(q.a, q.a);
  r.qb2 = cmul(q.b, q.b);
  r.Fa = cmul(r.qa2, r.qa2);
  r.Fb = cmul(r.qb2, r.qb2);
  r.z = cmul(q.a, cconj(q.b));
  r.qab = cmul(q.a, q.b);
  return r;
}

// One sample of the five-mode sum: amplitudes / phases of (2,2),(2,1),(3,3),(4,4),(5,5), the
// monomials of the sample's quaternion, the mode constants, e^{2 i psi}.
__device__ __forceinline__ void k1_std5_sample(const double (&am)[5], const double (&ph)[5], const K1Pre& pre,
                                               const double (&cc)[5], double rot_c, double rot_s, double& hp,
                                               double& hx) {
  // h_k = a (cos phi - i sin phi), scaled by its constant
  cplx h[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double s, c;
    const double a = am[k] * cc[k];
    sincos_d(ph[k], s, c);
    h[k] = {a * c, -a * s};
  }
  // G = h22 + z (h33 + z (h44 + z h55))
  cplx g = cmul(pre.z, h[4]);
  g = {g.re + h[3].re, g.im + h[3].im};
  g = cmul(pre.z, g);
  g = {g.re + h[2].re, g.im + h[2].im};
  g = cmul(pre.z, g);
  g = {g.re + h[0].re, g.im + h[0].im};
  cplx t1 = cmul(pre.Fa, g), t2 = cmul(pre.Fb, cconj(g));
  cplx u1 = cmul(pre.qa2, h[1]), u2 = cmul(pre.qb2, cconj(h[1]));
  cplx u = cmul(pre.qab, {u1.re + u2.re, u1.im + u2.im});
  const double Hre = (t1.re + t2.re) + u.re, Him = (t1.im + t2.im) + u.im;
  hp = fma(Hre, rot_c, -Him * rot_s);
  hx = -fma(Hre, rot_s, Him * rot_c);
}

// V samples per thread (V = 2: adjacent samples, 16-byte loads and stores; needs even N).  All 13
// input values of the thread are loaded BEFORE any arithmetic so that each thread has 13 x 8 V
// bytes in flight (the first version interleaved loads with the sincos evaluations and sat on
// the HBM latency: long_scoreboard 9.8 per issue at 52 % of HBM bandwidth).
template <int V>
__device__ __forceinline__ void k1_load(const double* __restrict__ ptr, size_t n, double (&out)[V]) {
  if constexpr (V == 2) {
    const double2 t = __ldg(reinterpret_cast<const double2*>(ptr + n));
    out[0] = t.x;
    out[1] = t.y;
  } else {
    out[0] = __ldg(ptr + n);
  }
}

template <int V>
__global__ void __launch_bounds__(K1_THREADS, 3) k1_modes_to_pol_std5(const K1FastParams p) {
  __shared__ quat Qc;
  __shared__ double rot[2];
  const int b = blockIdx.y;
  if (threadIdx.x == 0) {
    quat q = quat_from_euler(p.phi[b], p.iota[b], 0.0);  // footnote 1
    if (p.have_e0)
      q = quat_mul(quat_from_euler(p.euler0[3 * b], p.euler0[3 * b + 1], p.euler0[3 * b + 2]), q);
    Qc = q;
    double s2, c2;
    sincos_d(2.0 * p.psi[b], s2, c2);
    rot[0] = c2;
    rot[1] = s2;
  }
  __syncthreads();
  const size_t bN = (size_t)b * p.N;
  const double* amp = p.amp + bN * p.n_modes;
  const double* pha = p.phase + bN * p.n_modes;
  const long long n = ((long long)blockIdx.x * K1_THREADS + threadIdx.x) * V;
  if (n >= p.N) return;
  // ---- all loads first
  double al[V], be[V], ga[V], am[5][V], ph[5][V];
  if (p.twisted) {
    k1_load<V>(p.alpha, bN + n, al);
    k1_load<V>(p.beta, bN + n, be);
    k1_load<V>(p.gamma, bN + n, ga);
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
#pragma unroll
    for (int v = 0; v < V; ++v) am[k][v] = ph[k][v] = 0.0;
    if (p.idx[k] >= 0) {
      k1_load<V>(amp, (size_t)p.idx[k] * p.N + n, am[k]);
      k1_load<V>(pha, (size_t)p.idx[k] * p.N + n, ph[k]);
    }
  }
  const quat qc = Qc;
  K1Pre pre = k1_pre(qc);
  const double cc[5] = {p.c22, p.c21, p.c33, p.c44, p.c55};
  double hp[V], hx[V];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    if (p.twisted) pre = k1_pre(quat_mul(quat_from_euler(al[v], be[v], ga[v]), qc));
    const double amv[5] = {am[0][v], am[1][v], am[2][v], am[3][v], am[4][v]};
    const double phv[5] = {ph[0][v], ph[1][v], ph[2][v], ph[3][v], ph[4][v]};
    k1_std5_sample(amv, phv, pre, cc, rot[0], rot[1], hp[v], hx[v]);
  }
  if constexpr (V == 2) {
    *reinterpret_cast<double2*>(p.hplus + bN + n) = make_double2(hp[0], hp[1]);
    *reinterpret_cast<double2*>(p.hcross + bN + n) = make_double2(hx[0], hx[1]);
  } else {
    p.hplus[bN + n] = hp[0];
    p.hcross[bN + n] = hx[0];
  }
}

// ---------------------------------------------------------------- TMA-pipelined five-mode kernel
// Persistent blocks (two per SM) walk over (walker, tile of K1T_TILE samples) items.  The 13 input
// rows of an item arrive in shared memory by 1-D bulk copies (cp.async.bulk, completion counted in
// bytes on an mbarrier), double buffered: the copies of item i+1 are in flight while item i is
// evaluated, so the ~330 fp64 operations per sample (8 sincos) and the 104 bytes per sample
// overlap instead of alternating (the load-everything-first kernel above sits at 64 % of the HBM
// bandwidth AND 63 % of the fp64 pipe).  Needs even N (16-byte copy sizes and row offsets).
constexpr int K1T_THREADS = 256;          // measured: 256 x 2 blocks 1.81 ms, 128 x 4 1.83, 64 x 8 and 32 x 16 2.02 (small copies)
constexpr int K1T_BLOCKS_PER_SM = 2;
constexpr int K1T_TILE = 2 * K1T_THREADS;  // samples per item: two adjacent samples per thread
constexpr int K1T_ROWS = 13;              // amp x5, phase x5, alpha, beta, gamma
constexpr size_t K1T_SMEM = (size_t)2 * K1T_ROWS * K1T_TILE * sizeof(double);

__device__ __forceinline__ unsigned k1_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void k1_bulk_load(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(k1_smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(k1_smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void k1_mbar_wait(uint64_t* b, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(k1_smem_u32(b)), "r"(parity)
        : "memory");
  } while (!done);
}

__global__ void __launch_bounds__(K1T_THREADS, K1T_BLOCKS_PER_SM) k1_modes_to_pol_std5_tma(const K1FastParams p, const int tiles_per_row,
                                                                        const long long n_items) {
  extern __shared__ __align__(128) double k1_stage[];  // [2][K1T_ROWS][K1T_TILE]
  __shared__ __align__(8) uint64_t bar[2];
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(k1_smem_u32(&bar[0])) : "memory");
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(k1_smem_u32(&bar[1])) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  // one thread issues the copies of an item: present modes and, if twisted, the three angles
  auto issue = [&](long long item, int stage) {
    const int b = (int)(item / tiles_per_row);
    const long long n0 = (item % tiles_per_row) * K1T_TILE;
    const unsigned bytes = (unsigned)(min((long long)K1T_TILE, p.N - n0) * sizeof(double));
    int rows = p.twisted ? 3 : 0;
#pragma unroll
    for (int k = 0; k < 5; ++k) rows += p.idx[k] >= 0 ? 2 : 0;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(k1_smem_u32(&bar[stage])), "r"(bytes * rows)
                 : "memory");
    double* dst = k1_stage + (size_t)stage * K1T_ROWS * K1T_TILE;
    const size_t bN = (size_t)b * p.N;
#pragma unroll
    for (int k = 0; k < 5; ++k)
      if (p.idx[k] >= 0) {
        const size_t off = (bN * p.n_modes + (size_t)p.idx[k] * p.N) + n0;
        k1_bulk_load(dst + k * K1T_TILE, p.amp + off, bytes, &bar[stage]);
        k1_bulk_load(dst + (5 + k) * K1T_TILE, p.phase + off, bytes, &bar[stage]);
      }
    if (p.twisted) {
      k1_bulk_load(dst + 10 * K1T_TILE, p.alpha + bN + n0, bytes, &bar[stage]);
      k1_bulk_load(dst + 11 * K1T_TILE, p.beta + bN + n0, bytes, &bar[stage]);
      k1_bulk_load(dst + 12 * K1T_TILE, p.gamma + bN + n0, bytes, &bar[stage]);
    }
  };
  if (threadIdx.x == 0 && blockIdx.x < n_items) issue(blockIdx.x, 0);

  const double cc[5] = {p.c22, p.c21, p.c33, p.c44, p.c55};
  quat qc = {{1.0, 0.0}, {0.0, 0.0}};
  double rot_c = 1.0, rot_s = 0.0;
  K1Pre pre = k1_pre(qc);
  int b_have = -1;
  int it = 0;
  for (long long item = blockIdx.x; item < n_items; item += gridDim.x, ++it) {
    const int stage = it & 1;
    // every thread is past its reads of the other stage (barrier at the end of the last round)
    if (threadIdx.x == 0 && item + gridDim.x < n_items) issue(item + gridDim.x, stage ^ 1);
    const int b = (int)(item / tiles_per_row);
    const long long n = (item % tiles_per_row) * K1T_TILE + 2 * threadIdx.x;
    if (b != b_have) {  // per-walker constants (uniform branch; a walker spans many items)
      qc = quat_from_euler(p.phi[b], p.iota[b], 0.0);  // footnote 1
      if (p.have_e0) qc = quat_mul(quat_from_euler(p.euler0[3 * b], p.euler0[3 * b + 1], p.euler0[3 * b + 2]), qc);
      sincos_d(2.0 * p.psi[b], rot_s, rot_c);
      pre = k1_pre(qc);
      b_have = b;
    }
    k1_mbar_wait(&bar[stage], (unsigned)((it >> 1) & 1));
    if (n < p.N) {
      const double* src = k1_stage + (size_t)stage * K1T_ROWS * K1T_TILE + 2 * threadIdx.x;
      double2 am2[5], ph2[5];
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        am2[k] = ph2[k] = make_double2(0.0, 0.0);
        if (p.idx[k] >= 0) {
          am2[k] = *reinterpret_cast<const double2*>(src + k * K1T_TILE);
          ph2[k] = *reinterpret_cast<const double2*>(src + (5 + k) * K1T_TILE);
        }
      }
      double hp[2], hx[2];
      if (p.twisted) {
        const double2 al = *reinterpret_cast<const double2*>(src + 10 * K1T_TILE);
        const double2 be = *reinterpret_cast<const double2*>(src + 11 * K1T_TILE);
        const double2 ga = *reinterpret_cast<const double2*>(src + 12 * K1T_TILE);
        {
          const double amv[5] = {am2[0].x, am2[1].x, am2[2].x, am2[3].x, am2[4].x};
          const double phv[5] = {ph2[0].x, ph2[1].x, ph2[2].x, ph2[3].x, ph2[4].x};
          k1_std5_sample(amv, phv, k1_pre(quat_mul(quat_from_euler(al.x, be.x, ga.x), qc)), cc, rot_c, rot_s, hp[0], hx[0]);
        }
        {
          const double amv[5] = {am2[0].y, am2[1].y, am2[2].y, am2[3].y, am2[4].y};
          const double phv[5] = {ph2[0].y, ph2[1].y, ph2[2].y, ph2[3].y, ph2[4].y};
          k1_std5_sample(amv, phv, k1_pre(quat_mul(quat_from_euler(al.y, be.y, ga.y), qc)), cc, rot_c, rot_s, hp[1], hx[1]);
        }
      } else {
        const double amx[5] = {am2[0].x, am2[1].x, am2[2].x, am2[3].x, am2[4].x};
        const double phx[5] = {ph2[0].x, ph2[1].x, ph2[2].x, ph2[3].x, ph2[4].x};
        k1_std5_sample(amx, phx, pre, cc, rot_c, rot_s, hp[0], hx[0]);
        const double amy[5] = {am2[0].y, am2[1].y, am2[2].y, am2[3].y, am2[4].y};
        const double phy[5] = {ph2[0].y, ph2[1].y, ph2[2].y, ph2[3].y, ph2[4].y};
        k1_std5_sample(amy, phy, pre, cc, rot_c, rot_s, hp[1], hx[1]);
      }
      const size_t o = (size_t)b * p.N + n;
      *reinterpret_cast<double2*>(p.hplus + o) = make_double2(hp[0], hp[1]);
      *reinterpret_cast<double2*>(p.hcross + o) = make_double2(hx[0], hx[1]);
    }
    __syncthreads();  // this stage may be refilled from the next round on
  }
}

static double factorial_ld(int n) {
  long double f = 1;
  for (int i = 2; i <= n; ++i) f *= i;
  return (double)f;
}
static long double binom_ld(int n, int k) {
  if (k < 0 || k > n) return 0;
  long double r = 1;
  for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
  return r;
}


int run_modes_to_pol(int B, long long N, int n_modes, const int* l, const int* m, const double* amp,
                     const double* phase, const double* alpha, const double* beta,
                     const double* gamma, const double* iota, const double* phi,
                     const double* psi, const double* euler0, double* hplus, double* hcross,
                     cudaStream_t st) {
  // fast path: the mode list is a subset of {(2,2),(2,1),(3,3),(4,4),(5,5)}, each at most once
  {
    static const int SL[5] = {2, 2, 3, 4, 5}, SM[5] = {2, 1, 3, 4, 5};
    K1FastParams f;
    bool ok = dispatch_mode() != 1;
    for (int j = 0; j < 5; ++j) f.idx[j] = -1;
    for (int k = 0; k < n_modes && ok; ++k) {
      int j = 0;
      while (j < 5 && !(SL[j] == l[k] && SM[j] == m[k])) ++j;
      if (j == 5 || f.idx[j] >= 0) ok = false;
      else f.idx[j] = k;
    }
    if (ok) {
      const long double PI_L = 3.14159265358979323846264338327950288L;
      auto NL = [&](int ll) { return sqrtl((2 * ll + 1) / (4 * PI_L)); };
      f.c22 = (double)NL(2);
      f.c21 = (double)(2 * NL(2));
      f.c33 = (double)(-sqrtl(6.0L) * NL(3));
      f.c44 = (double)(2 * sqrtl(7.0L) * NL(4));
      f.c55 = (double)(-sqrtl(120.0L) * NL(5));
      f.B = B; f.N = N; f.n_modes = n_modes; f.twisted = alpha != nullptr; f.have_e0 = euler0 != nullptr;
      f.amp = amp; f.phase = phase; f.alpha = alpha; f.beta = beta; f.gamma = gamma;
      f.iota = iota; f.phi = phi; f.psi = psi; f.euler0 = euler0; f.hplus = hplus; f.hcross = hcross;
      if ((N & 1) == 0 && dispatch_mode() != 2) {  // 2: the load-everything-first five-mode kernel
        const int tiles_per_row = (int)((N + K1T_TILE - 1) / K1T_TILE);
        const long long n_items = (long long)tiles_per_row * B;
        int dev = 0, sms = 148;
        LISA_CUDA(cudaGetDevice(&dev));
        LISA_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        const long long blocks = n_items < (long long)K1T_BLOCKS_PER_SM * sms ? n_items : (long long)K1T_BLOCKS_PER_SM * sms;
        LISA_CUDA(cudaFuncSetAttribute(k1_modes_to_pol_std5_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K1T_SMEM));
        k1_modes_to_pol_std5_tma<<<(unsigned)blocks, K1T_THREADS, K1T_SMEM, st>>>(f, tiles_per_row, n_items);
      } else if ((N & 1) == 0) {
        dim3 grid((unsigned)((N / 2 + K1_THREADS - 1) / K1_THREADS), (unsigned)B);
        k1_modes_to_pol_std5<2><<<grid, K1_THREADS, 0, st>>>(f);
      } else {
        dim3 grid((unsigned)((N + K1_THREADS - 1) / K1_THREADS), (unsigned)B);
        k1_modes_to_pol_std5<1><<<grid, K1_THREADS, 0, st>>>(f);
      }
      LISA_LAUNCH_CHECK("k1_modes_to_pol_std5");
      return LISA_TD_OK;
    }
  }
  K1Params p;
  p.B = B; p.N = N; p.n_modes = n_modes; p.twisted = alpha != nullptr; p.have_e0 = euler0 != nullptr;
  p.amp = amp; p.phase = phase; p.alpha = alpha; p.beta = beta; p.gamma = gamma;
  p.iota = iota; p.phi = phi; p.psi = psi; p.euler0 = euler0; p.hplus = hplus; p.hcross = hcross;
  int nr = 0;
  const long double PI_L = 3.14159265358979323846264338327950288L;
  for (int k = 0; k < n_modes; ++k) {
    const int ll = l[k], mm = m[k];
    for (int sgn = +1; sgn >= -1; sgn -= 2) {
      if (sgn < 0 && mm == 0) break;
      const int mp = sgn * mm;
      K1Row& r = p.row[nr++];
      r.mode = (short)k; r.conj = sgn < 0; r.ka = (short)(mp + 2); r.kb = (short)(2 - mp); r.pad = 0;
      const int rmin = mp - 2 > 0 ? mp - 2 : 0;
      const int rmax = (ll + mp < ll - 2) ? ll + mp : ll - 2;
      r.eA0 = (short)(r.ka >= 0 ? ll - 2 - rmin : ll + mp - rmin);
      r.eB0 = (short)(r.kb >= 0 ? rmin : rmin - (mp - 2));
      r.nterms = (short)(rmax - rmin + 1);
      const long double pref = sqrtl((long double)factorial_ld(ll + 2) * factorial_ld(ll - 2) /
                                     ((long double)factorial_ld(ll + mp) * factorial_ld(ll - mp)));
      const long double norm = sqrtl((2 * ll + 1) / (4 * PI_L));
      for (int i = 0; i < K1_MAX_TERMS; ++i) r.coef[i] = 0.0;
      for (int rho = rmin; rho <= rmax; ++rho) {
        long double c = binom_ld(ll + mp, rho) * binom_ld(ll - mp, ll - rho - 2) * pref * norm;
        if (rho & 1) c = -c;
        if (sgn < 0 && (ll & 1)) c = -c;  // h_{l,-m} = (-1)^l conj(h_lm)  (A6)
        r.coef[rho - rmin] = (double)c;
      }
    }
  }
  p.n_rows = nr;
  dim3 grid((unsigned)((N + K1_THREADS * K1_PER_THREAD - 1) / (K1_THREADS * K1_PER_THREAD)), (unsigned)B);
  k1_modes_to_pol<<<grid, K1_THREADS, 0, st>>>(p);
  LISA_LAUNCH_CHECK("k1_modes_to_pol");
  return LISA_TD_OK;
}

}  // namespace lisa
