// k2_link_response.cu -- S2: h+, hx -> six link responses (Eq. 2.7-2.8, PAPER.md:138-161;
// readings A7, A8, A11 of DESIGN.md), and the link-level laser-noise helper (A12).
//
// One block = one walker x a tile of TILE output samples.  The strain tile with its halo
// (+- margin_y samples) is staged once in shared memory, interleaved as (h+, hx) pairs so
// every stencil tap is one 16-byte LDS.  Each thread owns output samples; for each it
// evaluates the orbit, the nine distinct evaluation times (3 receivers + 6 emitters) and, for
// each of them, one fused "Lagrange coefficient sweep + two dot products" (common.cuh).
#include "common.cuh"

namespace lisa {

struct K2Params {
  int B;
  long long N;
  double t0, dt, inv_dt;
  int half;  // (p+1)/2
  int margin;
  const double* hplus;
  const double* hcross;
  const double* lambda;
  const double* beta_sky;
  double* y;
  OrbitDev orb;
  LagW lw;
};

constexpr int K2_TILE = 512;
constexpr int K2_THREADS = 256;

// One fractional-delay read of (h+, hx) at delay D = Dc + Dl (samples).  The integer part is
// decided from the rounded sum, the fraction is formed as (K - Dc) - Dl so that the common
// 1 AU part (up to ~100 samples) does not cost the differential delays their low bits.
template <int HT>
__device__ __forceinline__ void read_pair(const double2* __restrict__ tile, int tile_len,
                                          int n_rel, double Dc, double Dl, int half,
                                          const LagW& lw, double& vp, double& vc) {
  const double Kf = ceil(Dc + Dl);
  const double eps = (Kf - Dc) - Dl;
  int b = n_rel - (int)Kf;  // tile index of tap j = 0
  // memory safety only (validated margins keep the window inside the tile)
  b = max(half - 1, min(b, tile_len - 1 - half));
  lagrange_dot2<HT>(eps, half, lw, tile + b, vp, vc);
}

template <int HT>
__global__ void __launch_bounds__(K2_THREADS, 2) k2_link_response(const K2Params p) {
  extern __shared__ double2 tile[];  // [TILE + 2*margin]
  __shared__ double sky[9];          // k, u, v of this walker (Eq. 2.7)
  const int b = blockIdx.y;
  const long long n0 = (long long)blockIdx.x * K2_TILE;
  const int R = p.margin;
  const int tile_len = K2_TILE + 2 * R;
  const double* hp = p.hplus + (size_t)b * p.N;
  const double* hc = p.hcross + (size_t)b * p.N;
  for (int i = threadIdx.x; i < tile_len; i += K2_THREADS) {
    long long g = n0 - R + i;
    double2 v = make_double2(0.0, 0.0);
    if (g >= 0 && g < p.N) v = make_double2(hp[g], hc[g]);
    tile[i] = v;
  }
  if (threadIdx.x == 0) {
    double sl, cl, sb, cb;
    sincos_d(p.lambda[b], sl, cl);
    sincos_d(p.beta_sky[b], sb, cb);
    sky[0] = -cb * cl; sky[1] = -cb * sl; sky[2] = -sb;  // k
    sky[3] = sl;       sky[4] = -cl;      sky[5] = 0.0;  // u
    sky[6] = -sb * cl; sky[7] = -sb * sl; sky[8] = cb;   // v
  }
  __syncthreads();
  const double kx = sky[0], ky = sky[1], kz = sky[2];
  const double ux = sky[3], uy = sky[4], uz = sky[5];
  const double vx = sky[6], vy = sky[7], vz = sky[8];
  double* yb = p.y + (size_t)b * 6 * p.N;

  for (int i = threadIdx.x; i < K2_TILE; i += K2_THREADS) {
    const long long n = n0 + i;
    if (n >= p.N) break;
    if (n < R || n >= p.N - R) {
#pragma unroll
      for (int l = 0; l < 6; ++l) yb[(size_t)l * p.N + n] = 0.0;
      continue;
    }
    const double t = fma((double)n, p.dt, p.t0);
    double d[3][3], cM, sM;
    orbit_offsets(p.orb, t, d, cM, sM);
    // delays in samples: common part and per-spacecraft parts
    const double Dc = p.orb.a_over_c * fma(kx, cM, ky * sM) * p.inv_dt;
    double Dk[3];
#pragma unroll
    for (int k = 0; k < 3; ++k)
      Dk[k] = fma(kx, d[k][0], fma(ky, d[k][1], kz * d[k][2])) * (p.inv_dt / C_LIGHT);
    const int n_rel = i + R;
    // the three reception-time reads h(t - k.r_r/c)
    double hpr[3], hcr[3];
#pragma unroll
    for (int k = 0; k < 3; ++k)
      read_pair<HT>(tile, tile_len, n_rel, Dc, Dk[k], p.half, p.lw, hpr[k], hcr[k]);
    // three arms; links l and -l share |d|, x+, xx and have opposite n
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int s = link_s(a), r = link_r(a);
      const double dx = d[r][0] - d[s][0], dy = d[r][1] - d[s][1], dz = d[r][2] - d[s][2];
      const double len = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
      const double inv = 1.0 / len;
      const double nx = dx * inv, ny = dy * inv, nz = dz * inv;
      const double un = fma(ux, nx, fma(uy, ny, uz * nz));
      const double vn = fma(vx, nx, fma(vy, ny, vz * nz));
      const double kn = fma(kx, nx, fma(ky, ny, kz * nz));
      const double xp = fma(un, un, -vn * vn);
      const double xc2 = 2.0 * un * vn;
      double Lp, Lm;
      if (p.orb.kind == 0) {
        Lp = p.orb.L[a];
        Lm = p.orb.L[a + 3];
      } else {
        Lp = Lm = len / C_LIGHT;
      }
      // link +a: s -> r
      {
        double hps, hcs;
        read_pair<HT>(tile, tile_len, n_rel, Dc, fma(Lp, p.inv_dt, Dk[s]), p.half, p.lw, hps, hcs);
        const double num = fma(xp, hps - hpr[r], xc2 * (hcs - hcr[r]));
        yb[(size_t)a * p.N + n] = num / (2.0 * (1.0 - kn));
      }
      // link -a: r -> s (n reversed)
      {
        double hps, hcs;
        read_pair<HT>(tile, tile_len, n_rel, Dc, fma(Lm, p.inv_dt, Dk[r]), p.half, p.lw, hps, hcs);
        const double num = fma(xp, hps - hpr[s], xc2 * (hcs - hcr[s]));
        yb[(size_t)(a + 3) * p.N + n] = num / (2.0 * (1.0 + kn));
      }
    }
  }
}

// A12: y_l[n] = p(n - L_l(t_n)/dt) - p[n].  Small helper kernel, reads p from global memory.
struct LaserParams {
  long long N;
  double t0, dt, inv_dt;
  int half;
  long long margin;
  const double* p;
  double* y;
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
    b = max((long long)(q.half - 1), min(b, q.N - 1 - q.half));
    q.y[(size_t)l * q.N + n] = lagrange_dot1<0>(eps, q.half, q.lw, q.p + b) - q.p[n];
  }
}

template <int HT>
static int launch_k2(const K2Params& p, cudaStream_t st) {
  const size_t smem = (size_t)(K2_TILE + 2 * p.margin) * sizeof(double2);
  if (smem > 200 * 1024) return set_error(LISA_TD_EINVAL, "link_response: margin_y too large for the shared-memory tile");
  if (smem > 48 * 1024)
    LISA_CUDA(cudaFuncSetAttribute(k2_link_response<HT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid((unsigned)((p.N + K2_TILE - 1) / K2_TILE), (unsigned)p.B);
  k2_link_response<HT><<<grid, K2_THREADS, smem, st>>>(p);
  LISA_LAUNCH_CHECK("k2_link_response");
  return LISA_TD_OK;
}

int g_force_generic = 0;  // debug switch (lisa_td_debug_force_generic)

int run_link_response(int B, long long N, double t0, double dt, int order, long long margin_y,
                      const double* hplus, const double* hcross, const double* lambda,
                      const double* beta_sky, const OrbitDev& orb, double* y, cudaStream_t st) {
  K2Params p;
  p.B = B; p.N = N; p.t0 = t0; p.dt = dt; p.inv_dt = 1.0 / dt;
  p.half = (order + 1) / 2; p.margin = (int)margin_y;
  p.hplus = hplus; p.hcross = hcross; p.lambda = lambda; p.beta_sky = beta_sky; p.y = y;
  p.orb = orb;
  make_lagw(order, &p.lw);
  if (!g_force_generic) {
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
  q.margin = margin; q.p = pser; q.y = y; q.orb = orb;
  make_lagw(order, &q.lw);
  k_laser_links<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(q);
  LISA_LAUNCH_CHECK("k_laser_links");
  return LISA_TD_OK;
}

}  // namespace lisa
