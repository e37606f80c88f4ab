// k2_link_response.cu -- S2: h+, hx -> six link responses (Eq. 2.7-2.8, PAPER.md:138-161;
// readings A7, A8, A11 of DESIGN.md), and the link-level laser-noise helper (A12).
//
// One block = K2_T consecutive output samples (one per thread) x a group of up to K2_G walkers.
// The orbit geometry of a sample -- spacecraft offsets, arm unit vectors, light travel times --
// does not depend on the walker: each thread evaluates it ONCE and keeps it in registers
// while the block loops over its walkers.  Per walker the strain tile with its halo
// (+- margin_y samples) is staged in shared memory by cp.async (double buffered), interleaved
// as (h+, hx) pairs so every stencil tap is one 16-byte LDS; the thread then forms the nine
// distinct evaluation times (3 receivers + 6 emitters) and, for each, one fused "Lagrange
// coefficient sweep + two dot products" (common.cuh).
#include "common.cuh"

namespace lisa {

struct K2Params {
  int B;
  long long N;
  double t0, dt, inv_dt;
  int half;  // (p+1)/2
  int margin;
  int group;  // walkers per block
  const double* hplus;
  const double* hcross;
  const double* lambda;
  const double* beta_sky;
  double* y;
  OrbitDev orb;
  LagW lw;   // generic (runtime order) path
  LagS ls;   // compile-time-order path
};

constexpr int K2_T = 256;  // output samples per block = threads per block
constexpr int K2_G = 16;   // walkers per block (upper bound)

__device__ __forceinline__ void k2_cp_async8_zfill(void* smem, const void* gmem, bool valid) {
  unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  int sz = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(sa), "l"(gmem), "r"(sz));
}

// One fractional-delay read of (h+, hx) at delay D = Dc + Dl (samples).  The integer part is
// decided from the rounded sum, the fraction is formed as (K - Dc) - Dl so that the common
// 1 AU part (up to ~100 samples) does not cost the differential delays their low bits.
template <int HT>
__device__ __forceinline__ void read_pair(const double2* __restrict__ tile, int tile_len,
                                          int n_rel, double Dc, double Dl, const K2Params& p,
                                          double& vp, double& vc) {
  const double Kf = ceil(Dc + Dl);
  const double eps = (Kf - Dc) - Dl;
  int b = n_rel - (int)Kf;  // tile index of tap j = 0
  // memory safety only (validated margins keep the window inside the tile)
  b = max(p.half - 1, min(b, tile_len - 1 - p.half));
  lagrange_dot2h<HT>(eps, p.half, p.ls, tile + b, vp, vc);
}

template <int HT, int KIND>
__global__ void __launch_bounds__(K2_T, 3) k2_link_response(const K2Params p) {
  extern __shared__ double2 tiles[];   // [2][K2_T + 2*margin] strain tiles, then geo[26][K2_T]
  __shared__ double sky[K2_G][9];      // k, u, v of the block's walkers (Eq. 2.7)
  const int R = p.margin;
  const int tile_len = K2_T + 2 * R;
  const long long n0 = (long long)blockIdx.x * K2_T;
  const int w0 = blockIdx.y * p.group;
  const int nw = min(p.group, p.B - w0);

  auto prefetch = [&](int w, int buf) {
    const double* hp = p.hplus + (size_t)(w0 + w) * p.N;
    const double* hc = p.hcross + (size_t)(w0 + w) * p.N;
    double2* dst = tiles + (size_t)buf * tile_len;
    for (int i = threadIdx.x; i < tile_len; i += K2_T) {
      const long long g = n0 - R + i;
      const bool ok = g >= 0 && g < p.N;
      const long long src = ok ? g : 0;
      k2_cp_async8_zfill(&dst[i].x, hp + src, ok);
      k2_cp_async8_zfill(&dst[i].y, hc + src, ok);
    }
    asm volatile("cp.async.commit_group;\n" ::);
  };
  prefetch(0, 0);

  if (threadIdx.x < nw) {
    double sl, cl, sb, cb;
    sincos_d(p.lambda[w0 + threadIdx.x], sl, cl);
    sincos_d(p.beta_sky[w0 + threadIdx.x], sb, cb);
    double* s = sky[threadIdx.x];
    s[0] = -cb * cl; s[1] = -cb * sl; s[2] = -sb;  // k
    s[3] = sl;       s[4] = -cl;      s[5] = 0.0;  // u
    s[6] = -sb * cl; s[7] = -sb * sl; s[8] = cb;   // v
  }

  // ---- walker-independent geometry of this thread's sample, kept in registers
  const long long n = n0 + threadIdx.x;
  const bool in_grid = n < p.N;
  const bool active = n >= R && n < p.N - R;
  // geo[f][thread]: 0,1 common 1 AU delay per unit k (samples); 2..10 spacecraft offsets as
  // delays per unit k (samples); 11..19 arm unit vectors (arm a: link_s(a) -> link_r(a));
  // 20..22 / 23..25 light travel times of links +a / -a (samples)
  double* geo = reinterpret_cast<double*>(tiles + 2 * (size_t)tile_len) + threadIdx.x;
#define GEO(f) geo[(f) * K2_T]
  {
    double d[3][3], cM, sM;
    orbit_offsets(p.orb, fma((double)n, p.dt, p.t0), d, cM, sM);
    const double sc = p.inv_dt / C_LIGHT;
    GEO(0) = p.orb.a_over_c * p.inv_dt * cM;
    GEO(1) = p.orb.a_over_c * p.inv_dt * sM;
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int j = 0; j < 3; ++j) GEO(2 + 3 * k + j) = d[k][j] * sc;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int s = link_s(a), r = link_r(a);
      const double dx = d[r][0] - d[s][0], dy = d[r][1] - d[s][1], dz = d[r][2] - d[s][2];
      const double len = sqrt(fma(dx, dx, fma(dy, dy, dz * dz)));
      const double inv = 1.0 / len;
      GEO(11 + 3 * a) = dx * inv; GEO(12 + 3 * a) = dy * inv; GEO(13 + 3 * a) = dz * inv;
      GEO(20 + a) = KIND == 0 ? p.orb.L[a] * p.inv_dt : len * sc;
      GEO(23 + a) = KIND == 0 ? p.orb.L[a + 3] * p.inv_dt : len * sc;
    }
  }
  const int n_rel = threadIdx.x + R;

  for (int w = 0; w < nw; ++w) {
    const int buf = w & 1;
    if (w + 1 < nw) {
      prefetch(w + 1, buf ^ 1);
      asm volatile("cp.async.wait_group 1;\n" ::);
    } else {
      asm volatile("cp.async.wait_group 0;\n" ::);
    }
    __syncthreads();  // tile of walker w (and, first time round, sky[]) visible to everyone
    double* yb = p.y + (size_t)(w0 + w) * 6 * p.N + n;
    if (active) {
      const double2* tile = tiles + (size_t)buf * tile_len;
      const double* s = sky[w];
      const double kx = s[0], ky = s[1], kz = s[2];
      const double ux = s[3], uy = s[4], uz = s[5];
      const double vx = s[6], vy = s[7], vz = s[8];
      const double Dc = fma(kx, GEO(0), ky * GEO(1));
      double Dk[3], hpr[3], hcr[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) Dk[k] = fma(kx, GEO(2 + 3 * k), fma(ky, GEO(3 + 3 * k), kz * GEO(4 + 3 * k)));
      // the three reception-time reads h(t - k.r_r/c)
#pragma unroll
      for (int k = 0; k < 3; ++k) read_pair<HT>(tile, tile_len, n_rel, Dc, Dk[k], p, hpr[k], hcr[k]);
      // three arms; links a and -a share x+, xx and have opposite n
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const int sd = link_s(a), rc = link_r(a);
        const double nx = GEO(11 + 3 * a), ny = GEO(12 + 3 * a), nz = GEO(13 + 3 * a);
        const double un = fma(ux, nx, fma(uy, ny, uz * nz));
        const double vn = fma(vx, nx, fma(vy, ny, vz * nz));
        const double kn = fma(kx, nx, fma(ky, ny, kz * nz));
        const double xp = fma(un, un, -vn * vn);
        const double xc2 = 2.0 * un * vn;
        const double om = 1.0 - kn, opl = 1.0 + kn;
        const double inv = 0.5 / (om * opl);  // 1/(2(1-kn)) = (1+kn) inv, 1/(2(1+kn)) = (1-kn) inv
        double hps, hcs;
        read_pair<HT>(tile, tile_len, n_rel, Dc, GEO(20 + a) + Dk[sd], p, hps, hcs);   // link +a: sd -> rc
        yb[(size_t)a * p.N] = fma(xp, hps - hpr[rc], xc2 * (hcs - hcr[rc])) * (opl * inv);
        read_pair<HT>(tile, tile_len, n_rel, Dc, GEO(23 + a) + Dk[rc], p, hps, hcs);   // link -a: rc -> sd
        yb[(size_t)(a + 3) * p.N] = fma(xp, hps - hpr[sd], xc2 * (hcs - hcr[sd])) * (om * inv);
      }
    } else if (in_grid) {
#pragma unroll
      for (int l = 0; l < 6; ++l) yb[(size_t)l * p.N] = 0.0;
    }
    __syncthreads();  // everyone is done with tiles[buf] before walker w+2 is prefetched into it
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

#undef GEO

template <int HT>
static int launch_k2(const K2Params& p, cudaStream_t st) {
  const size_t smem = (size_t)2 * (K2_T + 2 * p.margin) * sizeof(double2) + (size_t)26 * K2_T * sizeof(double);
  if (smem > 100 * 1024) return set_error(LISA_TD_EINVAL, "link_response: margin_y too large for the shared-memory tile");
  dim3 grid((unsigned)((p.N + K2_T - 1) / K2_T), (unsigned)((p.B + p.group - 1) / p.group));
  if (p.orb.kind == 0) {
    if (smem > 48 * 1024)
      LISA_CUDA(cudaFuncSetAttribute(k2_link_response<HT, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k2_link_response<HT, 0><<<grid, K2_T, smem, st>>>(p);
  } else {
    if (smem > 48 * 1024)
      LISA_CUDA(cudaFuncSetAttribute(k2_link_response<HT, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k2_link_response<HT, 1><<<grid, K2_T, smem, st>>>(p);
  }
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
  p.group = B < K2_G ? B : K2_G;
  make_lagw(order, &p.lw);
  make_lags(order, &p.ls);
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
