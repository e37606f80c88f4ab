// k3_tdi.cu -- S3: six links -> TDI X,Y,Z (generation 1.5 / 2) -> A,E,T
// (Eq. 2.9-2.11; readings A9, A10 of DESIGN.md).
//
// The delays of TDI are sums of light travel times L_l(t_n): they depend on time but NOT on
// the walker.  The fast kernel (k3_tdi_mma, below) therefore merges the delayed reads of every
// (channel, y series) pair into one stencil per output sample, shared by all walkers, and
// applies it as a banded matrix product on the FP64 tensor path.
//
// A plain one-thread-per-(walker, sample) kernel covers every other order / cadence.
#include <cuda.h>
#include <stdlib.h>
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
  unsigned int* err;  // sticky device error words (common.cuh)
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
// One (walker, sample): every delayed read its own stencil of runtime (HT = 0) or compile-time order.
template <int HT>
__device__ __forceinline__ void k3_generic_sample(const K3Params& p, long long n, int b) {
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
        if (base < p.half - 1 || base > p.N - 1 - p.half) {  // the margins did not cover the delay after all
          raise_error(p.err, DEVERR_K3_WINDOW);
          base = max((long long)(p.half - 1), min(base, p.N - 1 - p.half));
        }
        acc += (double)pr.t[k].sign * lagrange_dot1<HT>(eps, p.half, p.lw, ser + base);
      }
    }
    xyz[c] = acc;
  }
  double o[3];
  combine_out(p.out_kind, xyz[0], xyz[1], xyz[2], o);
  for (int c = 0; c < 3; ++c) ob[(size_t)c * p.N + n] = o[c];
}

// One thread per (walker, sample): the whole job for orders / cadences the merged-stencil kernel has
// no instantiation for.
__global__ void __launch_bounds__(256) k3_tdi_generic(const K3Params p) {
  const long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (n < p.N) k3_generic_sample<0>(p, n, blockIdx.y);
}

// Fix-up pass behind the merged-stencil kernel: recomputes, sample by sample, the tiles of `tile`
// samples (an anchor group, a divisor of 256) that k3_anchor_tables listed (list[0] = count,
// list[1..] = group indices).  Work item = (listed group, 256 / tile walkers), thread = (sample,
// walker); blocks without an item leave at once.
template <int HT>
__global__ void __launch_bounds__(256) k3_tdi_fixup(const K3Params p, const int* __restrict__ list, const int tile) {
  const int wpi = 256 / tile;  // walkers per item
  const int groups = (p.B + wpi - 1) / wpi;
  const int items = list[0] * groups;
  for (int item = blockIdx.x; item < items; item += gridDim.x) {
    const long long n = (long long)list[1 + item / groups] * tile + (threadIdx.x % tile);
    const int b = (item % groups) * wpi + threadIdx.x / tile;
    if (n < p.N && b < p.B) k3_generic_sample<HT>(p, n, b);
  }
}

// ---------------------------------------------------------------- merged-stencil DMMA kernel
// The delays of TDI are sums (or chains) of light travel times: they depend on time but NOT on
// the walker, and they change by ~1e-7 samples per sample.  The kernel uses both facts.
//
// Tile = K3_TS = 32 output samples x ALL walkers.  Per (channel, y series) pair the 4 (generation
// 2) or 2 (generation 1.5) delayed reads that hit the series merge into ONE stencil of WIN taps
// (the interpolation is linear in y:  sum_t s_t sum_j c_j(eps_t) y[n-K_t+j] = sum_i C_i y[n+LOW+i]),
// so the output is a banded product  out[n][w] = sum_pairs sum_m Cband_p[n][m] y_{series(p)}[m][w]
// whose left operand is shared by every walker: it runs on the FP64 tensor path (mma.sync m8n8k4
// f64 -> DMMA.8x8x4), warp = (channel, block of 8 samples), A fragments (4 pairs x KSTEPS) in
// registers for the whole tile, B fragments (y of 8 walkers x 4 times) one conflict-free LDS.64
// each.  Walkers stream through shared memory in chunks of 16, one 2-D tensor-map TMA copy per
// chunk (double buffered, mbarrier completion); X,Y,Z of a chunk meet in shared memory for A,E,T.
//
// Merged stencils from three anchors.  Within a group of four tiles (128 samples) no integer delay
// changes (checked), so every tap of the merged stencil is a smooth function of the sample: it is
// evaluated EXACTLY at the anchor samples 0, 64, 128 of the group (3 x 48 coefficient sweeps
// instead of 128 x 48) and every row gets the quadratic through the anchors (truncation
// |f'''| 64^3 0.064 ~ 5e-15 of a tap on a heliocentric orbit).  Tiles where an integer delay does change (one in ~1e4), where
// the delay is not smooth enough, or that straddle a node of a tabulated orbit are flagged and
// listed, and recomputed sample by sample by a fix-up pass (k3_tdi_fixup).
//
// The anchor stencils do not depend on the walkers either, and a thirteenth warp to prepare them
// next to the MMA warps does not fit (the A fragments need 104 of the 168 registers a thread can
// have at three warps per scheduler; four warps per scheduler cap everyone at 128).  They are
// therefore written by a small kernel of their own (k3_anchor_tables: 12 x 3 x WIN doubles and a
// split flag per tile, 13 KB) into a workspace, and the persistent MMA kernel (one block per SM,
// walking over tiles) pulls the table of the NEXT tile into shared memory with one bulk TMA copy
// while the walkers of the current tile stream through the DMMA loop, and forms the next tile's A
// fragments under the DMMAs of the current tile's last walker chunk.
constexpr int K3_TS = 32;                     // output samples per tile (four 8-row MMA blocks)
constexpr int K3_PAIRS = 12;                  // (channel, series) pairs
constexpr int K3_THREADS = K3_TS * K3_PAIRS;  // 384: warp = (channel, row block)
// a delay is "a parabola over the tile" if its value at sample 8 is within this many samples of the
// parabola through samples 0, 16, 32: ~10x the rounding noise of a delay of ~12 samples formed from
// six square roots (4e-15 rms), far below anything that matters for a tap (|dc/deps| ~ 3)
constexpr double K3_SMOOTH_TOL = 1e-13;
constexpr int K3_TAB_TILES = 2;               // anchor groups per block of k3_anchor_tables
constexpr int K3_TAB_THREADS = 96;
constexpr int K3_RB = K3_TS / 8;              // 8-row blocks per tile
constexpr int K3_WC = 16;                     // walkers per shared-memory chunk (two MMA N-blocks)
constexpr int K3_XS = K3_WC + 1;              // row stride of the X,Y,Z exchange buffer
constexpr int K3_GT = 4;                      // tiles per anchor group: one table serves 128 samples
constexpr int K3_GS = K3_GT * K3_TS;          // samples per anchor group
constexpr int K3_AH = K3_GS / 2;              // anchor spacing: anchors at group samples 0, 64, 128

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
// 1-D bulk TMA copy global -> shared (bytes a multiple of 16), completion on an mbarrier
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, unsigned bytes, uint64_t* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(b))
               : "memory");
}
// D(8x8) += A(8x4, row) * B(4x8, col), fp64.  Lane l holds A[l/4][l%4], B[l%4][l/4] and
// D[l/4][2(l%4) + {0,1}].
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// row[j + H - 1] += sgn * c_j(eps), j = -H+1..H, on a shared-memory row owned by the calling
// thread (scaled weights, common.cuh LagS: 7 fp64 ops per node pair + the two accumulations).
template <int H>
__device__ __forceinline__ void add_term_row(double* __restrict__ row, double eps, double sgn, const LagS& ls) {
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
    row[k + H - 1] += k == 1 ? t : fma(a, (double)(k - 1), t);
    row[H - k] += fma(a, (double)k, -t);
    if (k > 1) S *= fma(ls.rho[k - 1], q, ls.rc[k - 1]);
  }
}

template <int H, int WIN>
struct K3Geom {
  static constexpr int KCAP = WIN - 2 * H;            // largest integer delay the window holds
  static constexpr int LOW = -(KCAP + H - 1);         // offset of stencil tap 0 relative to n
  static constexpr int KSTEPS = (WIN + 7 + 3) / 4;    // k-steps of one 8-sample row block
  static constexpr int PAD = (LOW % 2 != 0) ? 1 : 0;  // the tile starts at the even sample n0 + LOW - PAD (16-byte aligned rows)
  static constexpr int TWMIN = K3_TS - 8 + 4 * KSTEPS + PAD;  // y samples a tile touches per series
  static constexpr int TW = TWMIN + ((2 - TWMIN % 4) + 4) % 4;  // == 2 mod 4: walker stride 6 TW == 4 or 12 mod 16
  static constexpr int YBUF = K3_WC * 6 * TW;         // doubles per walker-chunk buffer
  static constexpr int XBUF = 2 * 3 * K3_TS * K3_XS;  // double buffered X,Y,Z exchange
  static constexpr int QS = WIN | 1;                  // odd row stride of the anchor stencils: conflict-free sweeps
  static constexpr int QBUF = K3_PAIRS * 3 * QS;      // one table: [pair][anchor][QS]
  static constexpr int NA = 4;                        // anchor samples 0, 16, 32 and the check sample 8
  static constexpr int QFLAG = QS - 1;                // spare slot of row 0: the tile's split flag (0.0 / 1.0)
  static_assert((QBUF * sizeof(double)) % 16 == 0, "bulk copy size");
  static constexpr size_t SMEM = (size_t)(2 * YBUF + XBUF + 2 * QBUF) * sizeof(double);
  // linear interpolation (H = 1): short stencils and few registers, two blocks share an SM if they fit
  static constexpr int BLOCKS_PER_SM = (H == 1 && SMEM <= 113 * 1024) ? 2 : 1;
};

__device__ __forceinline__ int k3_anchor_sample(int a) { return a == 3 ? K3_AH / 2 : a * K3_AH; }

// Anchor tables.  Block = K3_TAB_TILES anchor groups (called "tiles" below; a group is K3_GS = 128
// samples = four MMA tiles).  Phase A: the delays of every group at its anchor samples n0,
// n0 + 64, n0 + 128 and at the check sample n0 + 32.  Phase B: thread = (tile, pair,
// anchor) sweeps the terms of its pair into one row of WIN taps.  A tile is flagged `split` (the MMA
// kernel then takes the exact per-row path) if an integer delay differs between its anchors, if
// the delay is not a parabola in the sample to 1e-13 samples (checked at sample 32, where the cubic
// term equals the largest interpolation error over the tile), or if it straddles a node of a
// tabulated orbit.  tab: [n_groups][12][3][QS], flag in slot QFLAG of row 0; flagged groups are also
// appended to `list` (count, then tile indices) for the fix-up pass.
template <int H, int WIN>
__global__ void __launch_bounds__(K3_TAB_THREADS) k3_anchor_tables(const __grid_constant__ K3Params p, double* __restrict__ tab,
                                                                   int* __restrict__ list, const int n_tiles) {
  using G = K3Geom<H, WIN>;
  constexpr int KCAP = G::KCAP, QS = G::QS, NA = G::NA, T = K3_TAB_TILES;
  __shared__ double rows[T * G::QBUF];
  __shared__ double Lanc[T * NA * 6];        // light travel times at the anchors
  __shared__ double Lq[T * NA * 3 * 6];      // KEPLER1, chained delays: L at t, t - h, t - 2h per anchor
  __shared__ double taus[T * NA * 6 * 8];    // chained delays per anchor and (channel, path)
  __shared__ int split[T];
  const int tid = threadIdx.x;
  const int tile0 = blockIdx.x * T;
  for (int i = tid; i < T * G::QBUF; i += K3_TAB_THREADS) rows[i] = 0.0;
  if (tid < T) {
    int sp = 0;
    if (p.orb.kind == 2) {  // a tabulated orbit is a different polynomial on either side of a table node
      const long long n0 = (long long)(tile0 + tid) * K3_GS;
      const double reach = p.orb.nested ? 8.0 * p.orb.max_L : 0.0;
      const double ua = (fma((double)n0, p.dt, p.t0) - reach - p.orb.t_tab0) * p.orb.inv_dt_tab;
      const double ub = (fma((double)(n0 + K3_GS), p.dt, p.t0) - p.orb.t_tab0) * p.orb.inv_dt_tab;
      sp = floor(ua) != floor(ub);
    }
    split[tid] = sp;
  }
  // ---- phase A
  const double hq = 3.5 * p.orb.max_L;
  if (p.orb.nested) {
    if (p.orb.kind == 1) {
      if (tid < T * NA * 3) {
        const int tl = tid / (NA * 3), a = (tid / 3) % NA, k = tid % 3;
        const long long n = (long long)(tile0 + tl) * K3_GS + k3_anchor_sample(a);
        double L[6];
        orbit_arm_times(p.orb, fma((double)n, p.dt, p.t0) - (double)k * hq, L);
#pragma unroll
        for (int l = 0; l < 6; ++l) Lq[tid * 6 + l] = L[l];
      }
      __syncthreads();
    }
    if (tid < T * NA * 6) {
      const int tl = tid / (NA * 6), a = (tid / 6) % NA, cp = tid % 6;  // cp = channel * 2 + path
      const long long n = (long long)(tile0 + tl) * K3_GS + k3_anchor_sample(a);
      double tau[8];
      if (p.orb.kind == 1) chain_delays_quad(Lq + (tl * NA + a) * 18, 1.0 / hq, p.path[cp >> 1][cp & 1], tau);
      else chain_delays(p.orb, fma((double)n, p.dt, p.t0), p.path[cp >> 1][cp & 1], tau);
#pragma unroll
      for (int i = 0; i < 8; ++i) taus[tid * 8 + i] = tau[i];
    }
  } else if (tid < T * NA) {
    const int tl = tid / NA, a = tid % NA;
    const long long n = (long long)(tile0 + tl) * K3_GS + k3_anchor_sample(a);
    double L[6];
    orbit_arm_times(p.orb, fma((double)n, p.dt, p.t0), L);
#pragma unroll
    for (int l = 0; l < 6; ++l) Lanc[tid * 6 + l] = L[l];
  }
  __syncthreads();
  // ---- phase B
  if (tid < T * K3_PAIRS * 3) {
    const int tl = tid / (K3_PAIRS * 3), pi = (tid / 3) % K3_PAIRS, a = tid % 3;
    const K3Pair& pr = p.pair[pi];
    double* row = rows + (size_t)tl * G::QBUF + (pi * 3 + a) * QS;
    auto delay = [&](int k, int an) {
      if (p.orb.nested) {
        const int chn = pr.t[k].chain;
        return taus[((tl * NA + an) * 6 + (pi / 4) * 2 + ((chn >> 3) & 1)) * 8 + (chn & 7)] * p.inv_dt;
      }
      double L[6];
#pragma unroll
      for (int l = 0; l < 6; ++l) L[l] = Lanc[(tl * NA + an) * 6 + l];
      return term_delay(pr.t[k], L, p.inv_dt);
    };
    for (int k = 0; k < pr.n_terms; ++k) {
      const double D = delay(k, a);
      const double Kf = ceil(D);
      if (a == 0) {
        const double D1 = delay(k, 1), D2 = delay(k, 2), D8 = delay(k, 3);
        const bool same_k = Kf == ceil(D1) && Kf == ceil(D2) && Kf == ceil(D8);
        const bool smooth = fabs(fma(0.375, D, fma(0.75, D1, -0.125 * D2)) - D8) <= K3_SMOOTH_TOL;
        if (!(same_k && smooth)) split[tl] = 1;
      }
      int off = KCAP - (int)Kf;
      if (off < 0 || off > KCAP) {  // the host-side bound on the delays was wrong
        raise_error(p.err, DEVERR_K3_WINDOW);
        off = max(0, min(off, KCAP));
      }
      add_term_row<H>(row + off, Kf - D, (double)pr.t[k].sign, p.ls);
    }
  }
  __syncthreads();
  if (tid < T && tile0 + tid < n_tiles) {
    rows[(size_t)tid * G::QBUF + G::QFLAG] = split[tid] ? 1.0 : 0.0;
    if (split[tid]) list[1 + atomicAdd(list, 1)] = tile0 + tid;  // for the fix-up pass (list[0] zeroed by the host)
  }
  __syncthreads();
  const int nt = min(T, n_tiles - tile0);
  double* dst = tab + (size_t)tile0 * G::QBUF;
  for (int i = tid; i < nt * G::QBUF; i += K3_TAB_THREADS) dst[i] = rows[i];
}

template <int H, int WIN>
__global__ void __launch_bounds__(K3_THREADS, K3Geom<H, WIN>::BLOCKS_PER_SM)
    k3_tdi_mma(const __grid_constant__ K3Params p, const __grid_constant__ CUtensorMap tmap, const int use_tma,
               const double* __restrict__ tab, const int n_tiles) {
  using G = K3Geom<H, WIN>;
  constexpr int LOW = G::LOW, KSTEPS = G::KSTEPS, TW = G::TW, PAD = G::PAD, QS = G::QS;
  constexpr int NWARPS = K3_THREADS / 32;
  constexpr bool OVERLAP_FILL = G::BLOCKS_PER_SM == 1;  // form the next tile's A fragments under the last chunk's DMMAs
  __shared__ __align__(8) uint64_t ybar[2];    // TMA completion, one per walker-chunk buffer
  __shared__ __align__(8) uint64_t tbar[2];    // TMA completion, one per anchor-table buffer
  extern __shared__ __align__(128) double smem[];
  double* ys = smem;                       // [2][WC][6][TW]
  double* xs = ys + 2 * G::YBUF;           // [2][3][TS][XS]
  double* qtab = xs + G::XBUF;             // [2][12][3][QS]
  const int lane = threadIdx.x & 31;
  const int wid = threadIdx.x >> 5;

  if (threadIdx.x == 0) {
    mbar_init(&ybar[0], 1);
    mbar_init(&ybar[1], 1);
    mbar_init(&tbar[0], 1);
    mbar_init(&tbar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  const int my_tiles = ((int)n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  auto tile_id = [&](int it) { return (long long)blockIdx.x + (long long)it * gridDim.x; };
  auto tile_n0 = [&](int it) { return tile_id(it) * K3_TS; };
  auto fetch_table = [&](int it) {  // thread 0: anchor table of this block's tile `it` into buffer it & 1
    mbar_arrive_expect_tx(&tbar[it & 1], (unsigned)(G::QBUF * sizeof(double)));
    tma_load_1d(qtab + (it & 1) * G::QBUF, tab + (size_t)(tile_id(it) / K3_GT) * G::QBUF, (unsigned)(G::QBUF * sizeof(double)), &tbar[it & 1]);
  };
  if (threadIdx.x == 0 && my_tiles > 0) fetch_table(0);

  // =============================================================== MMA warps
  const int n_chunks = (p.B + K3_WC - 1) / K3_WC;
  // Walker chunks arrive by TMA: ONE 2-D tiled copy per chunk (box = TW samples x 96 rows of the
  // [B*6][N] matrix; parts of the box outside the matrix are zero-filled by the hardware, which
  // covers both the grid edges and a ragged last chunk), completion counted on the buffer's
  // mbarrier.  The tensor map needs 16-byte row strides, so odd N takes the zero-filling
  // cp.async path instead.
  auto prefetch = [&](long long n0, int chunk, int buf) {
    double* dst = ys + (size_t)buf * G::YBUF;
    const long long g0 = n0 + LOW - PAD;
    if (use_tma) {
      if (threadIdx.x == 0) {
        mbar_arrive_expect_tx(&ybar[buf], (unsigned)(G::YBUF * sizeof(double)));
        tma_load_2d(dst, &tmap, (int)g0, chunk * K3_WC * 6, &ybar[buf]);
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
  const int ch = wid / K3_RB, rb = wid % K3_RB;
  const int r = lane >> 2, kk = lane & 3;
  int ser[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) ser[q] = p.pair[ch * 4 + q].series;
  const bool vec = (p.N & 1) == 0;

  // A fragments of (channel ch, row block rb), pair q of tile `it`: KSTEPS values, the quadratic
  // through the group's three anchors at this lane's row (a flagged group gets meaningless
  // fragments: the fix-up pass behind this kernel overwrites its outputs)
  double A[4][KSTEPS];
  auto fill_pair = [&](const int q, const int it) {
    const double* src = qtab + (it & 1) * G::QBUF + (ch * 4 + q) * 3 * QS;
    const double u = (double)((int)(tile_id(it) % K3_GT) * K3_TS + rb * 8 + r) * (1.0 / K3_AH);
    const double w0 = 0.5 * (u - 1.0) * (u - 2.0), w1 = u * (2.0 - u), w2 = 0.5 * u * (u - 1.0);
#pragma unroll
    for (int ks = 0; ks < KSTEPS; ++ks) {
      const int i = 4 * ks + kk - r;
      const bool in = i >= 0 && i < WIN;
      const int ic = in ? i : 0;
      const double v = fma(w2, src[2 * QS + ic], fma(w1, src[QS + ic], w0 * src[ic]));
      A[q][ks] = in ? v : 0.0;
    }
  };

  if (my_tiles > 0) {
    prefetch(tile_n0(0), 0, 0);
    mbar_wait(&tbar[0], 0u);
#pragma unroll
    for (int q = 0; q < 4; ++q) fill_pair(q, 0);
  }
  unsigned g = 0;  // chunks processed so far (y and exchange buffers alternate on it)
  for (int it = 0; it < my_tiles; ++it) {
    const long long n0 = tile_n0(it);
    const bool have_next = it + 1 < my_tiles;
    // the table buffer of the next tile was last read when the fragments of tile it - 1 ... were
    // formed, i.e. before the barriers of the chunks behind us
    if (threadIdx.x == 0 && have_next) fetch_table(it + 1);
    if (!OVERLAP_FILL && it > 0) {  // short stencils (order 1, two blocks per SM): the fill is a few loads, up front
      mbar_wait(&tbar[it & 1], (unsigned)((it >> 1) & 1));
#pragma unroll
      for (int q = 0; q < 4; ++q) fill_pair(q, it);
    }

    // ---- stream the walkers.  In the LAST chunk of a tile the fragments of the NEXT tile are formed
    // pair by pair, each as soon as the DMMAs of that pair have been issued: its 39 shared-memory
    // loads and FMAs run under the DMMAs of the following pairs (and of the other warps) instead of
    // in a phase of their own in which the tensor path idles.
    for (int c = 0; c < n_chunks; ++c, ++g) {
      const int buf = g & 1;
      const bool refill = OVERLAP_FILL && have_next && c == n_chunks - 1;
      // the other y buffer was last read in the previous chunk, which every MMA warp has left
      bool more = true;
      if (c + 1 < n_chunks) prefetch(n0, c + 1, buf ^ 1);
      else if (have_next) prefetch(tile_n0(it + 1), 0, buf ^ 1);
      else more = false;
      if (use_tma) {
        mbar_wait(&ybar[buf], (g >> 1) & 1);
      } else {
        if (more) cp_async_wait<1>();
        else cp_async_wait<0>();
        __syncthreads();  // cp.async path: other threads' copies become visible here
      }
      if (refill) mbar_wait(&tbar[(it + 1) & 1], (unsigned)(((it + 1) >> 1) & 1));
      double* xsc = xs + (size_t)buf * (3 * K3_TS * K3_XS);
      // lane's B element: walker (r | r + 8) of the chunk, time rb*8 + 4 ks + kk
      const double* yb = ys + (size_t)buf * G::YBUF + (size_t)r * 6 * TW + rb * 8 + kk + PAD;
      // four independent accumulator chains per warp (two walker groups x even / odd k-steps): with
      // three warps per scheduler that is twelve DMMAs in flight against the latency of one
      double d00 = 0.0, d01 = 0.0, d10 = 0.0, d11 = 0.0, e00 = 0.0, e01 = 0.0, e10 = 0.0, e11 = 0.0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const double* y0 = yb + ser[q] * TW;
        const double* y1 = y0 + 8 * 6 * TW;
#pragma unroll
        for (int ks = 0; ks < KSTEPS; ++ks) {
          if ((ks & 1) == 0) {
            dmma884(d00, d01, A[q][ks], y0[4 * ks]);
            dmma884(d10, d11, A[q][ks], y1[4 * ks]);
          } else {
            dmma884(e00, e01, A[q][ks], y0[4 * ks]);
            dmma884(e10, e11, A[q][ks], y1[4 * ks]);
          }
        }
        if (refill) fill_pair(q, it + 1);
      }
      d00 += e00; d01 += e01; d10 += e10; d11 += e11;
      {
        double* xr = xsc + (size_t)(ch * K3_TS + rb * 8 + r) * K3_XS + 2 * kk;
        xr[0] = d00; xr[1] = d01; xr[8] = d10; xr[9] = d11;
      }
      __syncthreads();  // X,Y,Z of this chunk complete; every warp is done reading y buffer `buf`
      // thread = (walker, two adjacent samples): X,Y,Z -> the three output channels, one 16-byte
      // store per channel
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

// bytes of workspace run_tdi needs for N samples: the anchor tables (sized for the widest window),
// then the list of flagged tiles
static long long tdi_table_bytes(long long n_groups) {
  return ((n_groups * (long long)K3Geom<16, 48>::QBUF * (long long)sizeof(double)) + 255) / 256 * 256;
}
long long tdi_workspace_bytes(long long N) {
  const long long n_groups = (N + K3_GS - 1) / K3_GS;
  return tdi_table_bytes(n_groups) + ((n_groups + 1) * (long long)sizeof(int) + 255) / 256 * 256;
}

template <int H, int WIN>
static int launch_mma(const K3Params& p, double* tab, cudaStream_t st) {
  using G = K3Geom<H, WIN>;
  static_assert(G::SMEM <= (G::BLOCKS_PER_SM == 2 ? 113 : 227) * 1024, "k3_tdi_mma shared memory");
  static_assert((G::YBUF * sizeof(double)) % 128 == 0, "TMA destination alignment");
  static_assert(G::QBUF <= K3Geom<16, 48>::QBUF, "workspace size");
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  int use_tma = 0;
  EncodeTiledFn enc = encode_tiled_fn();
  if (enc && (p.N & 1) == 0 && p.N < (1LL << 31) - 4096) {
    const cuuint64_t gdim[2] = {(cuuint64_t)p.N, (cuuint64_t)p.B * 6};
    const cuuint64_t gstr[1] = {(cuuint64_t)p.N * sizeof(double)};
    const cuuint32_t box[2] = {(cuuint32_t)G::TW, (cuuint32_t)(K3_WC * 6)};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(p.y), gdim, gstr, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    use_tma = r == CUDA_SUCCESS;
  }
  const long long n_tiles = (p.N + K3_TS - 1) / K3_TS;
  // 1. anchor stencils of every tile (walker-independent)
  const long long n_groups = (p.N + K3_GS - 1) / K3_GS;
  int* list = reinterpret_cast<int*>(reinterpret_cast<char*>(tab) + tdi_table_bytes(n_groups));
  LISA_CUDA(cudaMemsetAsync(list, 0, sizeof(int), st));
  k3_anchor_tables<H, WIN><<<(unsigned)((n_groups + K3_TAB_TILES - 1) / K3_TAB_TILES), K3_TAB_THREADS, 0, st>>>(p, tab, list, (int)n_groups);
  LISA_LAUNCH_CHECK("k3_anchor_tables");
  // 2. persistent MMA blocks: one (two at order 1) per SM, each walking over tiles blockIdx.x + i gridDim.x
  const long long resident = (long long)G::BLOCKS_PER_SM * sm_count();
  const unsigned grid = (unsigned)(n_tiles < resident ? n_tiles : resident);
  LISA_CUDA(cudaFuncSetAttribute(k3_tdi_mma<H, WIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM));
  k3_tdi_mma<H, WIN><<<grid, K3_THREADS, G::SMEM, st>>>(p, tmap, use_tma, tab, (int)n_tiles);
  LISA_LAUNCH_CHECK("k3_tdi_mma");
  // 3. fix-up: the flagged tiles, sample by sample (threads of other tiles leave at once)
  k3_tdi_fixup<H><<<2 * sm_count(), 256, 0, st>>>(p, list, K3_GS);
  LISA_LAUNCH_CHECK("k3_tdi_fixup");
  return LISA_TD_OK;
}

// the merged-stencil path with its workspace: the caller's, or a stream-ordered temporary
template <int H, int WIN>
static int run_mma(const K3Params& p, double* tab_ws, long long tab_ws_bytes, cudaStream_t st) {
  const long long need = tdi_workspace_bytes(p.N);
  if (tab_ws) {
    if (tab_ws_bytes < need) return set_error(LISA_TD_ENOMEM, "tdi: workspace of %lld bytes is smaller than the %lld needed", tab_ws_bytes, need);
    return launch_mma<H, WIN>(p, tab_ws, st);
  }
  // no workspace argument (lisa_td_tdi2): draw it from the device's stream-ordered memory pool and
  // give it back in stream order -- no synchronisation, and the pool keeps the pages for the next call
  static thread_local int pool_dev = -1;
  int dev = 0;
  LISA_CUDA(cudaGetDevice(&dev));
  if (dev != pool_dev) {
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      unsigned long long keep = ~0ULL;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    cudaGetLastError();
    pool_dev = dev;
  }
  void* tmp = nullptr;
  LISA_CUDA(cudaMallocAsync(&tmp, (size_t)need, st));
  const int rc = launch_mma<H, WIN>(p, static_cast<double*>(tmp), st);
  const int rc2 = check_cuda(cudaFreeAsync(tmp, st), "cudaFreeAsync");
  return rc ? rc : rc2;
}

int run_tdi(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
            long long margin_lo, long long margin_hi, const double* y, const OrbitDev& orb,
            double* tdi, cudaStream_t st, double* tab_ws, long long tab_ws_bytes) {
  K3Params p;
  p.B = B; p.N = N; p.t0 = t0; p.dt = dt; p.inv_dt = 1.0 / dt;
  p.half = (order + 1) / 2; p.generation = generation; p.out_kind = out_kind;
  p.margin_lo = margin_lo; p.margin_hi = margin_hi; p.y = y; p.tdi = tdi; p.orb = orb;
  p.err = device_error_words();
  make_lagw(order, &p.lw);
  make_lags(order, &p.ls);
  if (build_pairs(generation, p.pair, p.path))
    return set_error(LISA_TD_EINVAL, "tdi: internal term table does not match the light paths");
  const int nL = generation == 20 ? 7 : 3;
  const int kcap = (int)ceil(nL * orb.max_L / dt);
  p.kcap = kcap;
  const int need = kcap + 2 * p.half;
  if (dispatch_mode() != 1) {
    if (p.half == 16) {
      if (need <= 40) return run_mma<16, 40>(p, tab_ws, tab_ws_bytes, st);
      if (need <= 44) return run_mma<16, 44>(p, tab_ws, tab_ws_bytes, st);
      if (need <= 48) return run_mma<16, 48>(p, tab_ws, tab_ws_bytes, st);
    } else if (p.half == 1) {
      if (need <= 8) return run_mma<1, 8>(p, tab_ws, tab_ws_bytes, st);
      if (need <= 16) return run_mma<1, 16>(p, tab_ws, tab_ws_bytes, st);
    }
  }
  dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
  k3_tdi_generic<<<grid, 256, 0, st>>>(p);
  LISA_LAUNCH_CHECK("k3_tdi_generic");
  return LISA_TD_OK;
}

// ---------------------------------------------------------------- no-allocation variant (lisa_td_tdi2_static)
// Same kernels as run_tdi; the anchor tables and the fix-up list live in a file-scope device array
// instead of a stream-ordered temporary, so the call allocates nothing (callers under CUDA graph
// capture, serving loops or harnesses that forbid cudaMalloc).  Every GPU that loads the library
// holds the array until exit; it is sized for K3_STATIC_MAX_N samples.  Layout:
//   [0, 256)   header: DEVERR_COUNT sticky error words of THIS entry point (device memory; the
//              other entry points use mapped host words, common.cuh, whose first use allocates)
//   [256, ...) anchor tables [groups][12][3][QS] and the list of flagged groups, as tdi_workspace_bytes
// The array keeps the last call's contents: the list count is cleared by every call
// (launch_mma), the tables of the groups a call uses are rewritten by it, the error words stay
// set until a call with check != 0 reads and clears them.  Calls that overlap on the GPU race.
constexpr long long K3_STATIC_MAX_N = LISA_TD_TDI2_STATIC_MAX_N;
constexpr long long K3_STATIC_GROUPS = (K3_STATIC_MAX_N + K3_GS - 1) / K3_GS;
constexpr size_t k3_round256(size_t b) { return (b + 255) / 256 * 256; }
constexpr size_t K3_STATIC_HDR = 256;
constexpr size_t K3_STATIC_BYTES = K3_STATIC_HDR + k3_round256((size_t)K3_STATIC_GROUPS * K3Geom<16, 48>::QBUF * sizeof(double)) +
                                   k3_round256((size_t)(K3_STATIC_GROUPS + 1) * sizeof(int));
static_assert(K3_STATIC_BYTES <= (size_t)8 << 20, "the static scratch is meant to stay modest (8 MiB)");
static_assert(DEVERR_COUNT * sizeof(unsigned int) <= K3_STATIC_HDR, "header holds the error words");
static __device__ __align__(256) unsigned char k3_static_scratch[K3_STATIC_BYTES];

// Device address of the array on the CURRENT device.  In host code `k3_static_scratch` is only a
// handle for the runtime, not a device pointer: the address is looked up once per device.
static int k3_static_base(unsigned char** out) {
  constexpr int MAX_DEV = 64;
  static thread_local unsigned char* addr[MAX_DEV] = {nullptr};
  int dev = 0;
  LISA_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEV) return set_error(LISA_TD_EINVAL, "tdi2_static: device ordinal %d not supported", dev);
  if (!addr[dev]) {
    void* ptr = nullptr;
    LISA_CUDA(cudaGetSymbolAddress(&ptr, k3_static_scratch));
    if (!ptr) return set_error(LISA_TD_ECUDA, "tdi2_static: cudaGetSymbolAddress returned a null address");
    addr[dev] = static_cast<unsigned char*>(ptr);
  }
  *out = addr[dev];
  return LISA_TD_OK;
}

int run_tdi_static(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
                   long long margin_lo, long long margin_hi, const double* y, const OrbitDev& orb,
                   double* tdi, int check, cudaStream_t st) {
  if (N > K3_STATIC_MAX_N)
    return set_error(LISA_TD_EINVAL,
                     "lisa_td_tdi2_static: N=%lld exceeds LISA_TD_TDI2_STATIC_MAX_N=%lld samples (the size of the static "
                     "scratch array); use lisa_td_tdi2 or lisa_td_response_tdi with a workspace",
                     N, K3_STATIC_MAX_N);
  if (tdi_workspace_bytes(N) > (long long)(K3_STATIC_BYTES - K3_STATIC_HDR))
    return set_error(LISA_TD_ENOMEM, "lisa_td_tdi2_static: internal: static scratch smaller than the workspace of N=%lld", N);
  unsigned char* base = nullptr;
  int rc = k3_static_base(&base);
  if (rc != LISA_TD_OK) return rc;
  unsigned int* err = reinterpret_cast<unsigned int*>(base);
  double* tab = reinterpret_cast<double*>(base + K3_STATIC_HDR);
  const long long tab_bytes = (long long)(K3_STATIC_BYTES - K3_STATIC_HDR);

  K3Params p;
  p.B = B; p.N = N; p.t0 = t0; p.dt = dt; p.inv_dt = 1.0 / dt;
  p.half = (order + 1) / 2; p.generation = generation; p.out_kind = out_kind;
  p.margin_lo = margin_lo; p.margin_hi = margin_hi; p.y = y; p.tdi = tdi; p.orb = orb;
  p.err = err;
  make_lagw(order, &p.lw);
  make_lags(order, &p.ls);
  if (build_pairs(generation, p.pair, p.path))
    return set_error(LISA_TD_EINVAL, "tdi: internal term table does not match the light paths");
  const int nL = generation == 20 ? 7 : 3;
  const int kcap = (int)ceil(nL * orb.max_L / dt);
  p.kcap = kcap;
  const int need = kcap + 2 * p.half;
  // run_mma with a workspace argument only launches (no cudaMallocAsync / cudaFreeAsync)
  bool done = false;
  if (dispatch_mode() != 1) {
    if (p.half == 16) {
      if (need <= 40) { rc = run_mma<16, 40>(p, tab, tab_bytes, st); done = true; }
      else if (need <= 44) { rc = run_mma<16, 44>(p, tab, tab_bytes, st); done = true; }
      else if (need <= 48) { rc = run_mma<16, 48>(p, tab, tab_bytes, st); done = true; }
    } else if (p.half == 1) {
      if (need <= 8) { rc = run_mma<1, 8>(p, tab, tab_bytes, st); done = true; }
      else if (need <= 16) { rc = run_mma<1, 16>(p, tab, tab_bytes, st); done = true; }
    }
  }
  if (!done) {  // other orders: one thread per sample, no scratch at all
    dim3 grid((unsigned)((N + 255) / 256), (unsigned)B);
    k3_tdi_generic<<<grid, 256, 0, st>>>(p);
    rc = check_cuda(cudaPeekAtLastError(), "k3_tdi_generic");
  }
  if (rc != LISA_TD_OK || !check) return rc;
  // check != 0: wait for the stream and report the sticky device-side range checks of this entry point
  unsigned int words[DEVERR_COUNT] = {0};
  LISA_CUDA(cudaMemcpyAsync(words, err, sizeof(words), cudaMemcpyDeviceToHost, st));
  LISA_CUDA(cudaStreamSynchronize(st));
  bool any = false;
  for (int i = 0; i < DEVERR_COUNT; ++i) any = any || words[i] != 0;
  if (any) {
    LISA_CUDA(cudaMemsetAsync(err, 0, sizeof(words), st));
    return set_error(LISA_TD_EINVAL,
                     "lisa_td_tdi2_static: a merged TDI stencil left its window on the device (the orbit exceeds the bounds "
                     "the margins were checked against); the output of this or an earlier unchecked call is wrong");
  }
  return LISA_TD_OK;
}

}  // namespace lisa
