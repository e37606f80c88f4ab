// k3_tdi.cu -- S3: six links -> TDI X,Y,Z (generation 1.5 / 2) -> A,E,T
// (Eq. 2.9-2.11; readings A9, A10 of DESIGN.md).
//
// The delays of TDI are sums of light travel times L_l(t_n): they depend on time but NOT on
// the walker.  The fast kernel therefore gives one block a tile of 32 output samples and ALL
// walkers: each thread (sample, channel x series) first merges the 4 (generation 2) or 2
// (generation 1.5) delayed reads that hit its y series into ONE stencil of WIN taps held in
// registers (the interpolation is linear in y, so  sum_t s_t sum_j c_j(eps_t) y[n-K_t+j]  =
// sum_i C_i y[n+LOW+i]), then streams the walkers through shared memory (cp.async, double
// buffered) doing WIN FMAs per walker.  48 coefficient sets per output sample are thus paid
// once per tile instead of once per walker, and 16x32 taps shrink to 4xWIN.
//
// A plain one-thread-per-(walker, sample) kernel covers every other order / cadence.
#include <cuda.h>
#include <string.h>

#include "common.cuh"

namespace lisa {

struct K3Term {
  signed char sign;
  signed char mult[6];  // multiplicity of each L_l in the delay (summed delays, A10)
  signed char chain;    // chained delays (A22): bits 0-2 = number of legs, bit 3 = light path (0 A, 1 B)
};
struct K3Pair {
  int series;   // link index 0..5 of the y series
  int n_terms;  // 4 (generation 2) or 2 (generation 1.5)
  K3Term t[4];
};
struct K3Params {
  int B;
  long long N;
  double t0, dt, inv_dt;
  int half, generation, out_kind, kcap;
  long long margin_lo, margin_hi;
  const double* y;
  double* tdi;
  OrbitDev orb;
  LagW lw;
  LagS ls;
  K3Pair pair[12];  // [channel X,Y,Z][slot]
  signed char path[3][2][8];  // chained delays: link indices of the two light paths per channel
};

// ---- term tables, restated from the paper ----------------------------------------------
// Michelson X, one line per y series: "link : sign {delay labels}" (labels are signed link
// numbers, each standing for one light travel time L_label).
// Eq. 2.9:
//   y_{1-32} = link -3 : +{3,2,-2}  -{3}
//   y_{231}  = link  3 : +{2,-2}    -{}
//   y_{123}  = link  2 : +{-2}      -{-2,-3,3}
//   y_{3-21} = link -2 : +{}        -{-3,3}
// Eq. 2.10 adds, per series, the same two terms delayed by a further
// L2+L-2+L3+L-3 with opposite sign (y123 block per reading A9).
struct TermSpec {
  int link;
  int sign;
  int n;
  int d[7];
};
static const TermSpec kX15[8] = {
    {-3, +1, 3, {3, 2, -2}},  {-3, -1, 1, {3}},
    {3, +1, 2, {2, -2}},      {3, -1, 0, {}},
    {2, +1, 1, {-2}},         {2, -1, 3, {-2, -3, 3}},
    {-2, +1, 0, {}},          {-2, -1, 2, {-3, 3}},
};
static const TermSpec kX20extra[8] = {
    {-3, +1, 5, {-2, 2, 3, 3, -3}},         {-3, -1, 7, {3, 3, -3, -2, -2, 2, 2}},
    {3, +1, 4, {-2, 2, 3, -3}},             {3, -1, 6, {3, -3, -2, -2, 2, 2}},
    {2, +1, 7, {-2, -2, 2, 3, 3, -3, -3}},  {2, -1, 5, {3, -3, -2, -2, 2}},
    {-2, +1, 6, {-2, 2, 3, 3, -3, -3}},     {-2, -1, 4, {3, -3, -2, 2}},
};

// Chained delays (reading A22).  X compares two light paths that start and end on spacecraft 1.
// Traced BACK from the output time (link l is received at link_r(l); stepping back along it lands
// on link_s(l)) they are, as signed link labels,
//   A: 1 <- 2 <- 1 <- 3 <- 1 <- 3 <- 1 <- 2 <- 1     B: 1 <- 3 <- 1 <- 2 <- 1 <- 2 <- 1 <- 3 <- 1
// and every delay multiset of Eq. 2.9 / 2.10 is a leading piece of one of them, followed on that
// path by the term's own link (checked when the tables are built): the chained delay of that term is  tau_0 = 0,
// tau_{i+1} = tau_i + L_{path[i]}(t - tau_i)  over that piece.
static const int kPathA[8] = {3, -3, -2, 2, -2, 2, 3, -3};
static const int kPathB[8] = {-2, 2, 3, -3, 3, -3, -2, 2};

static int cyc_label(int label, int times) {  // 1->2->3->1 on |label|, sign kept
  int s = label < 0 ? -1 : 1, a = label < 0 ? -label : label;
  for (int i = 0; i < times; ++i) a = a % 3 + 1;
  return s * a;
}
static int label_index(int label) { return label > 0 ? label - 1 : -label + 2; }

// which path has ts.d as the multiset of its first ts.n labels: 0 (A) or 1 (B); -1 if none / both
static int match_path(const TermSpec& ts) {
  int hit = -1;
  for (int c = 0; c < 2; ++c) {
    const int* path = c == 0 ? kPathA : kPathB;
    int cnt[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < ts.n; ++i) {
      cnt[label_index(path[i])]++;
      cnt[label_index(ts.d[i])]--;
    }
    bool same = true;
    for (int i = 0; i < 6; ++i) same = same && cnt[i] == 0;
    // the term's link is the NEXT leg of the path (the beam that arrives where the piece ends);
    // this also separates the two pieces of four legs, which are equal as multisets
    if (same && path[ts.n] == ts.link) hit = hit == -1 ? c : -2;
  }
  return hit < 0 ? -1 : hit;
}

static int build_pairs(int generation, K3Pair* out, signed char (*path)[2][8]) {
  for (int c = 0; c < 3; ++c)
    for (int i = 0; i < 8; ++i) {
      path[c][0][i] = (signed char)label_index(cyc_label(kPathA[i], c));
      path[c][1][i] = (signed char)label_index(cyc_label(kPathB[i], c));
    }
  for (int c = 0; c < 3; ++c)
    for (int slot = 0; slot < 4; ++slot) {
      K3Pair& pr = out[c * 4 + slot];
      pr.series = label_index(cyc_label(kX15[2 * slot].link, c));
      pr.n_terms = 0;
      for (int pass = 0; pass < (generation == 20 ? 2 : 1); ++pass)
        for (int k = 0; k < 2; ++k) {
          const TermSpec& ts = pass == 0 ? kX15[2 * slot + k] : kX20extra[2 * slot + k];
          K3Term& t = pr.t[pr.n_terms++];
          t.sign = (signed char)ts.sign;
          const int which = match_path(ts);
          if (which < 0) return -1;
          t.chain = (signed char)(ts.n | (which << 3));
          for (int i = 0; i < 6; ++i) t.mult[i] = 0;
          for (int i = 0; i < ts.n; ++i) t.mult[label_index(cyc_label(ts.d[i], c))]++;
        }
      for (int k = pr.n_terms; k < 4; ++k) {
        pr.t[k].sign = 0;
        pr.t[k].chain = 0;
        for (int i = 0; i < 6; ++i) pr.t[k].mult[i] = 0;
      }
    }
  return 0;
}

__device__ __forceinline__ double term_delay(const K3Term& t, const double (&L)[6], double inv_dt) {
  double D = 0.0;
#pragma unroll
  for (int i = 0; i < 6; ++i) D = fma((double)t.mult[i], L[i], D);
  return D * inv_dt;
}

// Chained delays of one light path (A22): tau[i] = delay after i legs, i = 0..7, in seconds.
__device__ __forceinline__ void chain_delays(const OrbitDev& orb, double t, const signed char (&path)[8],
                                             double (&tau)[8]) {
  double acc = 0.0;
  tau[0] = 0.0;
#pragma unroll 1
  for (int i = 0; i < 7; ++i) {
    double L[6];
    orbit_arm_times(orb, t - acc, L);
    const int l = path[i];
    double Ll = L[0];
#pragma unroll
    for (int q = 1; q < 6; ++q) Ll = l == q ? L[q] : Ll;
    acc += Ll;
    tau[i + 1] = acc;
  }
}

// The same chain for an ANALYTIC orbit (KEPLER1), from the six L sampled at t, t - h, t - 2h with
// 2h = 7 max L (the longest chain): L_l(t - tau) is read off the quadratic through the three
// samples.  Its truncation error is |d3L/dt3| x 0.064 h^3 < 1e-16 s on a heliocentric orbit (the
// arm lengths breathe by ~1 % at the orbital rate 2e-7 rad/s), far below one ulp of the delay
// (12 samples x 2^-52 x dt = 1.3e-14 s): 3 orbit evaluations per sample instead of 42.
// Lq: [3][6] seconds.
__device__ __forceinline__ void chain_delays_quad(const double* __restrict__ Lq, double inv_h,
                                                  const signed char (&path)[8], double (&tau)[8]) {
  double acc = 0.0;
  tau[0] = 0.0;
#pragma unroll
  for (int i = 0; i < 7; ++i) {
    const int l = path[i];
    const double a = Lq[l], b = Lq[6 + l], c = Lq[12 + l];
    const double x = acc * inv_h;
    acc += fma(x * (x - 1.0), 0.5 * ((c - b) - (b - a)), fma(x, b - a, a));
    tau[i + 1] = acc;
  }
}

__device__ __forceinline__ void combine_out(int out_kind, double X, double Y, double Z, double (&o)[3]) {
  if (out_kind == 0) {
    o[0] = X; o[1] = Y; o[2] = Z;
  } else {  // Eq. 2.11
    o[0] = (Z - X) * 0.70710678118654752440;
    o[1] = (X - 2.0 * Y + Z) * 0.40824829046386301637;
    o[2] = (X + Y + Z) * 0.57735026918962576451;
  }
}

// ---------------------------------------------------------------- generic kernel
__global__ void __launch_bounds__(256) k3_tdi_generic(const K3Params p) {
  const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  if (n >= p.N) return;
  double* ob = p.tdi + (size_t)b * 3 * p.N;
  if (n < p.margin_lo || n >= p.N - p.margin_hi) {
    for (int c = 0; c < 3; ++c) ob[(size_t)c * p.N + n] = 0.0;
    return;
  }
  const double* yb = p.y + (size_t)b * 6 * p.N;
  double L[6];
  const double tn = fma((double)n, p.dt, p.t0);
  if (!p.orb.nested) orbit_arm_times(p.orb, tn, L);
  double xyz[3];
  for (int c = 0; c < 3; ++c) {
    double acc = 0.0;
    double tau[2][8];
    if (p.orb.nested) {
      chain_delays(p.orb, tn, p.path[c][0], tau[0]);
      chain_delays(p.orb, tn, p.path[c][1], tau[1]);
    }
    for (int s = 0; s < 4; ++s) {
      const K3Pair& pr = p.pair[c * 4 + s];
      const double* ser = yb + (size_t)pr.series * p.N;
      for (int k = 0; k < pr.n_terms; ++k) {
        const double D = p.orb.nested ? tau[(pr.t[k].chain >> 3) & 1][pr.t[k].chain & 7] * p.inv_dt
                                      : term_delay(pr.t[k], L, p.inv_dt);
        const double Kf = ceil(D);
        const double eps = Kf - D;
        long long base = n - (long long)Kf;
        base = max((long long)(p.half - 1), min(base, p.N - 1 - p.half));
        acc += (double)pr.t[k].sign * lagrange_dot1<0>(eps, p.half, p.lw, ser + base);
      }
    }
    xyz[c] = acc;
  }
  double o[3];
  combine_out(p.out_kind, xyz[0], xyz[1], xyz[2], o);
  for (int c = 0; c < 3; ++c) ob[(size_t)c * p.N + n] = o[c];
}

// ---------------------------------------------------------------- merged-stencil DMMA kernel
// Block = K3_TS = 32 output samples x ALL walkers.
//
// Phase 1 (once per block): warp = (channel, series) pair, lane = sample.  Each thread merges
// the 4 (generation 2) or 2 (generation 1.5) delayed reads of its pair into ONE stencil of WIN
// taps (the interpolation is linear in y: sum_t s_t sum_j c_j(eps_t) y[n-K_t+j] = sum_i C_i
// y[n+LOW+i]) and parks it in shared memory.  The light travel times of the 32 samples are
// evaluated once (32 threads) and shared.
//
// Phase 2: the merged stencils form, per pair, a banded matrix Cband[n][m]; the output is the
// banded product  out[n][w] = sum_pairs sum_m Cband_p[n][m] y_{series(p)}[m][w]  over the
// walkers w -- the one dense-ish contraction on this path whose left operand does NOT depend
// on the walker.  It runs on the FP64 tensor path (mma.sync m8n8k4 f64 -> DMMA.8x8x4): warp =
// (channel, block of 8 samples), A fragments (4 pairs x KSTEPS) live in registers for the
// whole block, B fragments (y of 8 walkers x 4 times) are one conflict-free LDS.64 each, and
// the four pairs of a channel accumulate in the same two accumulator registers.  One LDS.64
// per 8 FMA instead of one per FMA (the previous SIMT version was shared-memory bound at 22 %
// FP64-pipe activity).  Walkers stream through shared memory in chunks of 16 (cp.async,
// double buffered); X,Y,Z of a chunk meet in shared memory for the A,E,T combination.
constexpr int K3_TS = 32;                  // output samples per block (two 8-row MMA blocks)
constexpr int K3_PAIRS = 12;               // (channel, series) pairs
constexpr int K3_THREADS = K3_TS * K3_PAIRS;  // phase 1: thread = (pair, sample); phase 2: warp = (channel, row block)
constexpr int K3_RB = K3_TS / 8;           // 8-row blocks per tile
constexpr int K3_WC = 16;                  // walkers per shared-memory chunk (two MMA N-blocks)
constexpr int K3_XS = K3_WC + 1;           // row stride of the X,Y,Z exchange buffer

__device__ __forceinline__ void cp_async8_zfill(void* smem, const void* gmem, bool valid) {
  unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(sa), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int NKEEP>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(NKEEP));
}
// TMA (bulk async copy) of one contiguous run of global memory into shared memory, completion
// counted in bytes on an mbarrier.  dst, src and bytes must be multiples of 16.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
// One 2-D tiled TMA copy: box (TW samples x rows) at coordinates (c0 = sample, c1 = row) of the
// [B*6][N] y matrix; samples / rows outside the matrix arrive as zeros.
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* b) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(smem_u32(dst)),
      "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(b))
      : "memory");
}
// Spin on test_wait (try_wait suspends the warp for a system-dependent time; with one block per
// SM every warp waits for the same tile, and late wake-ups showed up as barrier stalls).
__device__ __forceinline__ void mbar_wait(uint64_t* b, unsigned parity) {
  unsigned done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(b)), "r"(parity)
        : "memory");
  } while (!done);
}
// D(8x8) += A(8x4, row) * B(4x8, col), fp64.  Lane l holds A[l/4][l%4], B[l%4][l/4] and
// D[l/4][2(l%4) + {0,1}].
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// Adds sgn * c_j(eps) into the merged stencil at compile-time offset OFF (scaled weights,
// common.cuh LagS: 7 fp64 ops per node pair + the two accumulations).
template <int H, int WIN, int OFF>
__device__ __forceinline__ void add_term_at(double (&C)[WIN], double eps, double sgn, const LagS& ls) {
  double P[H + 1];
  const double q = eps * (eps - 1.0);
  P[1] = ls.g * sgn;
#pragma unroll
  for (int k = 1; k < H; ++k) P[k + 1] = P[k] * fma(ls.rho[k - 1], q, ls.rc[k - 1]);
  double S = 1.0;
#pragma unroll
  for (int k = H; k >= 1; --k) {
    const double a = P[k] * S;
    const double t = a * eps;
    C[OFF + k + H - 1] += k == 1 ? t : fma(a, (double)(k - 1), t);
    C[OFF + H - k] += fma(a, (double)k, -t);
    if (k > 1) S *= fma(ls.rho[k - 1], q, ls.rc[k - 1]);
  }
}
template <int H, int WIN, int OFF>
struct TermDispatch {
  static __device__ __forceinline__ void run(double (&C)[WIN], int off, double eps, double sgn, const LagS& ls) {
    if (off == OFF) add_term_at<H, WIN, OFF>(C, eps, sgn, ls);
    else TermDispatch<H, WIN, OFF - 1>::run(C, off, eps, sgn, ls);
  }
};
template <int H, int WIN>
struct TermDispatch<H, WIN, -1> {
  static __device__ __forceinline__ void run(double (&)[WIN], int, double, double, const LagS&) {}
};

template <int H, int WIN>
struct K3Geom {
  static constexpr int KCAP = WIN - 2 * H;            // largest integer delay the window holds
  static constexpr int LOW = -(KCAP + H - 1);         // offset of stencil tap 0 relative to n
  static constexpr int KSTEPS = (WIN + 7 + 3) / 4;    // k-steps of one 8-sample row block
  static constexpr int PAD = (LOW % 2 != 0) ? 1 : 0;  // the tile starts at the even sample n0 + LOW - PAD (16-byte aligned rows)
  static constexpr int TWMIN = K3_TS - 8 + 4 * KSTEPS + PAD;  // y samples a block touches per series
  static constexpr int TW = TWMIN + ((2 - TWMIN % 4) + 4) % 4;  // == 2 mod 4: walker stride 6 TW == 4 or 12 mod 16
  static constexpr int CS = ((WIN + 2) / 8) * 8 + 5;  // odd, >= WIN, (CS-1) == 4 mod 8: conflict-free fragment reads
  static constexpr int YBUF = K3_WC * 6 * TW;         // doubles per walker-chunk buffer
  static constexpr int CBUF = K3_PAIRS * K3_TS * CS;  // doubles of the stencil staging area
  static constexpr int XBUF = 2 * 3 * K3_TS * K3_XS;  // double buffered X,Y,Z exchange (phase 1 with chained delays: [32][6][8] + [32][3][6])
  static_assert(XBUF >= K3_TS * (48 + 18), "chained-delay scratch");
  // y buffer 0 is private (its first TMA copy overlaps the coefficient phase); the stencil
  // staging area shares its space with y buffer 1, which is first filled after phase 1
  static constexpr int UNION_PRIV = YBUF + (YBUF > CBUF ? YBUF : CBUF);
  static constexpr int UNION_ALIAS = (2 * YBUF > CBUF ? 2 * YBUF : CBUF);
  // linear interpolation (H = 1): the stencils are short, two blocks share an SM
  static constexpr int BLOCKS_PER_SM = (K3_TS == 16 || H == 1) ? 2 : 1;
  static constexpr bool PRIVATE0 = (size_t)(UNION_PRIV + 2 * 3 * K3_TS * K3_XS + K3_TS * 6) * sizeof(double) <= (BLOCKS_PER_SM == 2 ? 112 : 227) * 1024;
  static constexpr int UNION = PRIVATE0 ? UNION_PRIV : UNION_ALIAS;
  static constexpr size_t SMEM = (size_t)(UNION + XBUF + K3_TS * 6) * sizeof(double);
};

template <int H, int WIN>
__global__ void __launch_bounds__(K3_THREADS, K3Geom<H, WIN>::BLOCKS_PER_SM)
    k3_tdi_mma(const K3Params p, const __grid_constant__ CUtensorMap tmap, const int use_tma) {
  using G = K3Geom<H, WIN>;
  constexpr int KCAP = G::KCAP, LOW = G::LOW, KSTEPS = G::KSTEPS, TW = G::TW, CS = G::CS, PAD = G::PAD;
  constexpr int NWARPS = K3_THREADS / 32;
  __shared__ __align__(8) uint64_t mbar[2];  // one per walker-chunk buffer (TMA completion)
  static_assert(CS >= WIN && (CS & 1), "stencil row stride");
  extern __shared__ __align__(128) double smem[];
  double* ys = smem;                    // [2][WC][6][TW]   (phase 2)
  double* cbuf = smem + (G::PRIVATE0 ? G::YBUF : 0);  // [12][32][CS]  (phase 1; aliased with y buffer 1, or with both)
  double* xs = smem + G::UNION;         // [2][3][TS][XS]
  double* Ls = xs + G::XBUF;            // [32][6]
  const int lane = threadIdx.x & 31;
  const int wid = threadIdx.x >> 5;
  const long long n0 = (long long)blockIdx.x * K3_TS;

  if (threadIdx.x == 0) {
    mbar_init(&mbar[0], 1);
    mbar_init(&mbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  const int n_chunks = (p.B + K3_WC - 1) / K3_WC;
  // Walker chunks arrive by TMA: ONE 2-D tiled copy per chunk (box = TW samples x 96 rows of the
  // [B*6][N] matrix; parts of the box outside the matrix are zero-filled by the hardware, which
  // covers both the grid edges and a ragged last chunk), completion counted on the buffer's
  // mbarrier.  The tensor map needs 16-byte row strides, so odd N takes the zero-filling
  // cp.async path instead.
  const long long g0 = n0 + LOW - PAD;
  auto prefetch = [&](int chunk, int buf) {
    double* dst = ys + (size_t)buf * G::YBUF;
    if (use_tma) {
      if (threadIdx.x == 0) {
        mbar_arrive_expect_tx(&mbar[buf], (unsigned)(G::YBUF * sizeof(double)));
        tma_load_2d(dst, &tmap, (int)g0, chunk * K3_WC * 6, &mbar[buf]);
      }
    } else {
      const int nrows = min(K3_WC, p.B - chunk * K3_WC) * 6;
      const double* src0 = p.y + (size_t)chunk * K3_WC * 6 * p.N + g0;
      for (int row = wid; row < K3_WC * 6; row += NWARPS) {
        const double* src = src0 + (size_t)row * p.N;
        for (int i = lane; i < TW; i += 32) {
          const long long g = g0 + i;
          const bool ok = row < nrows && g >= 0 && g < p.N;
          cp_async8_zfill(dst + row * TW + i, ok ? src + i : p.y, ok);
        }
      }
      cp_async_commit();
    }
  };
  if (G::PRIVATE0) prefetch(0, 0);  // chunk 0 lands in y buffer 0 while the coefficients are computed
  // ---- phase 1a: light travel times of the tile's samples
  // (chained delays, A22: thread = (sample, channel, light path) walks its path leg by leg and
  // parks the 8 delays in the X,Y,Z exchange area, which phase 2 has not touched yet)
  double* taus = xs;  // [32][3][2][8]
  if (p.orb.nested) {
    double* Lq = taus + K3_TS * 6 * 8;  // [32][3][6]: KEPLER1 only
    const double hq = 3.5 * p.orb.max_L;
    if (p.orb.kind == 1) {
      if (threadIdx.x < K3_TS * 3) {
        const int sm = threadIdx.x % K3_TS, k = threadIdx.x / K3_TS;
        double L[6];
        orbit_arm_times(p.orb, fma((double)(n0 + sm), p.dt, p.t0) - (double)k * hq, L);
#pragma unroll
        for (int l = 0; l < 6; ++l) Lq[(sm * 3 + k) * 6 + l] = L[l];
      }
      __syncthreads();
    }
    if (threadIdx.x < K3_TS * 6) {
      const int sm = threadIdx.x % K3_TS, cp = threadIdx.x / K3_TS;  // cp = channel * 2 + path
      double tau[8];
      if (p.orb.kind == 1) chain_delays_quad(Lq + sm * 18, 1.0 / hq, p.path[cp >> 1][cp & 1], tau);
      else chain_delays(p.orb, fma((double)(n0 + sm), p.dt, p.t0), p.path[cp >> 1][cp & 1], tau);
#pragma unroll
      for (int i = 0; i < 8; ++i) taus[(sm * 6 + cp) * 8 + i] = tau[i];
    }
  } else if (threadIdx.x < K3_TS) {
    double L[6];
    orbit_arm_times(p.orb, fma((double)(n0 + threadIdx.x), p.dt, p.t0), L);
#pragma unroll
    for (int l = 0; l < 6; ++l) Ls[threadIdx.x * 6 + l] = L[l];
  }
  __syncthreads();
  // ---- phase 1b: merged stencil of (pair = wid, sample = lane)
  {
    double C[WIN];
#pragma unroll
    for (int i = 0; i < WIN; ++i) C[i] = 0.0;
    const int pi = threadIdx.x / K3_TS, sm = threadIdx.x % K3_TS;  // pair, sample
    const K3Pair& pr = p.pair[pi];
    const long long n = n0 + sm;
    if (n >= p.margin_lo && n < p.N - p.margin_hi) {
      double L[6];
#pragma unroll
      for (int l = 0; l < 6; ++l) L[l] = Ls[sm * 6 + l];
      for (int k = 0; k < pr.n_terms; ++k) {
        const int chn = pr.t[k].chain;
        const double D = p.orb.nested ? taus[(sm * 6 + (pi / 4) * 2 + ((chn >> 3) & 1)) * 8 + (chn & 7)] * p.inv_dt
                                      : term_delay(pr.t[k], L, p.inv_dt);
        const double Kf = ceil(D);
        const double eps = Kf - D;
        int off = KCAP - (int)Kf;
        off = max(0, min(off, KCAP));
        TermDispatch<H, WIN, KCAP>::run(C, off, eps, (double)pr.t[k].sign, p.ls);
      }
    }
    double* dst = cbuf + (size_t)(pi * K3_TS + sm) * CS;
#pragma unroll
    for (int i = 0; i < WIN; ++i) dst[i] = C[i];
  }
  __syncthreads();
  // ---- phase 1c: A fragments of (channel ch, row block rb): 4 pairs x KSTEPS values
  const int ch = wid / K3_RB, rb = wid % K3_RB;
  const int r = lane >> 2, kk = lane & 3;
  double A[4][KSTEPS];
  int ser[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    ser[q] = p.pair[ch * 4 + q].series;
    const double* src = cbuf + (size_t)((ch * 4 + q) * K3_TS + rb * 8 + r) * CS;
#pragma unroll
    for (int ks = 0; ks < KSTEPS; ++ks) {
      const int i = 4 * ks + kk - r;
      A[q][ks] = (i >= 0 && i < WIN) ? src[i] : 0.0;
    }
  }
  // cbuf (generic-proxy writes and reads) is about to become y buffer 1 (async-proxy TMA writes):
  // every thread that touched it fences, THEN the barrier, then one thread issues the copy
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  __syncthreads();  // cbuf is dead from here on: its space becomes the y buffers

  // ---- phase 2: stream walkers
  if (!G::PRIVATE0) prefetch(0, 0);
  for (int c = 0; c < n_chunks; ++c) {
    const int buf = c & 1;
    if (c + 1 < n_chunks) prefetch(c + 1, buf ^ 1);
    if (use_tma) {
      mbar_wait(&mbar[buf], (unsigned)((c >> 1) & 1));
    } else {
      if (c + 1 < n_chunks) cp_async_wait<1>();
      else cp_async_wait<0>();
    }
    // TMA path: the mbarrier wait makes the tile visible to each waiting thread, and the
    // X,Y,Z exchange buffer alternates, so ONE barrier per chunk (after the MMAs) is enough:
    // warps that finish their stores early start the next chunk's MMAs.
    if (!use_tma) __syncthreads();  // cp.async path: other threads' copies become visible here
    double* xsc = xs + (size_t)buf * (3 * K3_TS * K3_XS);
    // lane's B element: walker (r | r + 8) of the chunk, time rb*8 + 4 ks + kk
    const double* yb = ys + (size_t)buf * G::YBUF + (size_t)r * 6 * TW + rb * 8 + kk + PAD;
    double d00 = 0.0, d01 = 0.0, d10 = 0.0, d11 = 0.0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const double* y0 = yb + ser[q] * TW;
      const double* y1 = y0 + 8 * 6 * TW;
#pragma unroll
      for (int ks = 0; ks < KSTEPS; ++ks) {
        dmma884(d00, d01, A[q][ks], y0[4 * ks]);
        dmma884(d10, d11, A[q][ks], y1[4 * ks]);
      }
    }
    {
      double* xr = xsc + (size_t)(ch * K3_TS + rb * 8 + r) * K3_XS + 2 * kk;
      xr[0] = d00; xr[1] = d01; xr[8] = d10; xr[9] = d11;
    }
    __syncthreads();  // X,Y,Z of chunk c complete; every warp is done reading y buffer `buf`
    // thread = (walker, two adjacent samples): X,Y,Z -> the three output channels, one 16-byte
    // store per channel
    const bool vec = (p.N & 1) == 0;
    for (int e = threadIdx.x; e < K3_WC * (K3_TS / 2); e += K3_THREADS) {
      const int l2 = e % (K3_TS / 2), w = e / (K3_TS / 2);
      const int b = c * K3_WC + w;
      const long long nn = n0 + 2 * l2;
      if (b >= p.B || nn >= p.N) continue;
      double v[3][2];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int ln = 2 * l2 + h;
        const double X = xsc[(0 * K3_TS + ln) * K3_XS + w];
        const double Y = xsc[(1 * K3_TS + ln) * K3_XS + w];
        const double Z = xsc[(2 * K3_TS + ln) * K3_XS + w];
        double out[3];
        combine_out(p.out_kind, X, Y, Z, out);
        const bool zero = nn + h < p.margin_lo || nn + h >= p.N - p.margin_hi;
#pragma unroll
        for (int o = 0; o < 3; ++o) v[o][h] = zero ? 0.0 : out[o];
      }
#pragma unroll
      for (int o = 0; o < 3; ++o) {
        double* dst = p.tdi + ((size_t)b * 3 + o) * p.N + nn;
        if (vec) {
          *reinterpret_cast<double2*>(dst) = make_double2(v[o][0], v[o][1]);
        } else {
          dst[0] = v[o][0];
          if (nn + 1 < p.N) dst[1] = v[o][1];
        }
      }
    }
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(ptr);
  }
  return fn;
}

template <int H, int WIN>
static int launch_mma(const K3Params& p, cudaStream_t st) {
  using G = K3Geom<H, WIN>;
  static_assert(G::SMEM <= 227 * 1024, "k3_tdi_mma shared memory");
  static_assert((G::YBUF * sizeof(double)) % 128 == 0, "TMA destination alignment");
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  int use_tma = 0;
  EncodeTiledFn enc = encode_tiled_fn();
  if (enc && (p.N & 1) == 0 && p.N < (1LL << 31)) {
    const cuuint64_t gdim[2] = {(cuuint64_t)p.N, (cuuint64_t)p.B * 6};
    const cuuint64_t gstr[1] = {(cuuint64_t)p.N * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)G::TW, (cuuint32_t)(K3_WC * 6)};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(p.y), gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    use_tma = r == CUDA_SUCCESS;
  }
  LISA_CUDA(cudaFuncSetAttribute(k3_tdi_mma<H, WIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM));
  k3_tdi_mma<H, WIN><<<(unsigned)((p.N + K3_TS - 1) / K3_TS), K3_THREADS, G::SMEM, st>>>(p, tmap, use_tma);
  LISA_LAUNCH_CHECK("k3_tdi_mma");
  return LISA_TD_OK;
}

extern int g_force_generic;

int run_tdi(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
            long long margin_lo, long long margin_hi, const double* y, const OrbitDev& orb,
            double* tdi, cudaStream_t st) {
  K3Params p;
  p.B = B; p.N = N; p.t0 = t0; p.dt = dt; p.inv_dt = 1.0 / dt;
  p.half = (order + 1) / 2; p.generation = generation; p.out_kind = out_kind;
  p.margin_lo = margin_lo; p.margin_hi = margin_hi; p.y = y; p.tdi = tdi; p.orb = orb;
  make_lagw(order, &p.lw);
  make_lags(order, &p.ls);
  if (build_pairs(generation, p.pair, p.path))
    return set_error(LISA_TD_EINVAL, "tdi: internal term table does not match the light paths");
  const int nL = generation == 20 ? 7 : 3;
  const int kcap = (int)ceil(nL * orb.max_L / dt);
  p.kcap = kcap;
  const int need = kcap + 2 * p.half;
  if (!g_force_generic) {
    if (p.half == 16) {
      if (need <= 40) return launch_mma<16, 40>(p, st);
      if (need <= 44) return launch_mma<16, 44>(p, st);
      if (need <= 48) return launch_mma<16, 48>(p, st);
    } else if (p.half == 1) {
      if (need <= 8) return launch_mma<1, 8>(p, st);
      if (need <= 16) return launch_mma<1, 16>(p, st);
    }
  }
  dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
  k3_tdi_generic<<<grid, 256, 0, st>>>(p);
  LISA_LAUNCH_CHECK("k3_tdi_generic");
  return LISA_TD_OK;
}

}  // namespace lisa
