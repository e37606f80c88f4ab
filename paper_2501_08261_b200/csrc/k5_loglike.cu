// k5_loglike.cu -- S4 + S5: forward FFT of A,E,T (cuFFT, the one library call on the path,
// PAPER.md:211, 404) and the band-limited noise-weighted inner products -> log L
// (Eq. 2.12-2.13; readings A13, A17; band PAPER.md:243).
//
//   (d|h)_b = sum_c sum_{k=kmin..kmax} w_c[k] Re(D_c[k] conj(H_{b,c}[k]))
//   (h|h)_b = sum_c sum_k w_c[k] |H_{b,c}[k]|^2         log L_b = (d|h)_b - (h|h)_b / 2
//
// FFT: the real series x[0..N) is handed to cuFFT as the complex series z[m] = x[2m] + i x[2m+1]
// of length M = N/2 (one Z2Z pass instead of D2Z's Z2Z + a full-spectrum post-processing pass);
// the real-input spectrum is recovered only where it is used -- inside the band -- by the
// textbook split  X[k] = E[k] + e^{-2 pi i k/N} O[k],  E = (Z[k] + conj Z[M-k])/2,
// O = -i (Z[k] - conj Z[M-k])/2, fused into the reduction kernels (packed_bin below).
//
// Reduction: grid (K5_SLICES, B); each block sums a contiguous slice of the band for the three
// channels of one walker (per-thread partials -> warp shuffles -> one value per warp ->
// first warp), writes one (dh, hh) pair; a second tiny kernel adds the K5_SLICES pairs of
// each walker in a fixed order, so the result is deterministic (no atomics).
#include <cufft.h>

#include <map>

#include "common.cuh"

namespace lisa {

constexpr int K5_SLICES = 32;
constexpr int K5_THREADS = 256;
constexpr int K5_MAX_PLANS = 8;  // cached cuFFT plans per lisa_td_plan (batch sizes a sampler alternates between)
constexpr int K6_MAXD = 32;     // parameters of the Fisher matrix
constexpr int K6_TILE = 128;    // (channel, bin) items staged per pass
constexpr int K6_THREADS = 256;
constexpr int K6_BLOCKS = 296;  // 2 per SM

struct Plan {
  int B;  // capacity (walkers)
  long long N, nf;
  // batched half-length Z2Z plans keyed by (walkers, all channels | one channel); at most
  // K5_MAX_PLANS of them, all sharing ONE work area (cuFFT's own allocation is switched off)
  std::map<int, cufftHandle> fft;
  void* work;
  size_t work_bytes;
  double2* spec;     // [B][3][M] packed half-length spectra Z (M = N/2)
  double2* partial;  // [B][K5_SLICES]
  double* fisher_partial;  // [K6_BLOCKS][K6_MAXD * K6_MAXD], allocated on first use
};

// X[k] of the real series from the packed spectrum Z (row of M = N/2 values), 0 <= k <= M.
// cs = (cos, sin)(2 pi k / N).
__device__ __forceinline__ double2 packed_bin(const double2* __restrict__ Z, long long M, long long k, double c, double s) {
  const double2 a = Z[k == M ? 0 : k];
  const double2 b = Z[k == 0 ? 0 : M - k];
  const double er = 0.5 * (a.x + b.x), ei = 0.5 * (a.y - b.y);
  const double orr = 0.5 * (a.y + b.y), oi = -0.5 * (a.x - b.x);
  return make_double2(er + fma(c, orr, s * oi), ei + fma(c, oi, -s * orr));
}
__device__ __forceinline__ void bin_twiddle(long long k, double two_pi_over_N, double& c, double& s) {
  sincos_d((double)k * two_pi_over_N, s, c);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(K5_THREADS) k5_inner_partial(
    const double2* __restrict__ spec, const double2* __restrict__ data,
    const double* __restrict__ weight, long long nf, long long kmin, long long kmax,
    double two_pi_over_N, double2* __restrict__ partial, int n_ch) {
  const int b = blockIdx.y, slice = blockIdx.x;
  const long long nk = kmax - kmin + 1;
  const long long per = (nk + K5_SLICES - 1) / K5_SLICES;
  const long long k0 = kmin + (long long)slice * per;
  const long long k1 = min(k0 + per, kmax + 1);
  const long long M = nf - 1;
  double dh = 0.0, hh = 0.0;
  for (long long k = k0 + threadIdx.x; k < k1; k += K5_THREADS) {
    double cw, sw;
    bin_twiddle(k, two_pi_over_N, cw, sw);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      if (c >= n_ch) break;  // channel subset A / A,E / A,E,T
      const double2 h = packed_bin(spec + ((size_t)b * 3 + c) * M, M, k, cw, sw);
      const double2 d = data[(size_t)c * nf + k];
      const double w = weight[(size_t)c * nf + k];
      dh = fma(w, fma(d.x, h.x, d.y * h.y), dh);
      hh = fma(w, fma(h.x, h.x, h.y * h.y), hh);
    }
  }
  __shared__ double sdh[K5_THREADS / 32], shh[K5_THREADS / 32];
  dh = warp_sum(dh);
  hh = warp_sum(hh);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) {
    sdh[wid] = dh;
    shh[wid] = hh;
  }
  __syncthreads();
  if (wid == 0) {
    dh = lane < K5_THREADS / 32 ? sdh[lane] : 0.0;
    hh = lane < K5_THREADS / 32 ? shh[lane] : 0.0;
    dh = warp_sum(dh);
    hh = warp_sum(hh);
    if (lane == 0) partial[(size_t)b * K5_SLICES + slice] = make_double2(dh, hh);
  }
}

__global__ void k5_inner_final(const double2* __restrict__ partial, int B, double* loglike,
                               double* dh_out, double* hh_out) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  double dh = 0.0, hh = 0.0;
  for (int s = 0; s < K5_SLICES; ++s) {
    const double2 v = partial[(size_t)b * K5_SLICES + s];
    dh += v.x;
    hh += v.y;
  }
  loglike[b] = fma(-0.5, hh, dh);
  if (dh_out) dh_out[b] = dh;
  if (hh_out) hh_out[b] = hh;
}

// ---------------------------------------------------------------- K6: Fisher matrix
// Gamma_ij = sum_c sum_k w_c[k] Re(d_i H conj d_j H),  d_i H = (H_i - H_0)/delta_i  (PAPER.md:249,
// reading A19).  The (channel, bin) items of the band are dealt to the blocks in tiles of
// K6_TILE: the first K6_TILE threads stage the D derivative values and the weight of one item
// each in shared memory (coalesced reads of the D+1 spectra), then thread = (i, j) pair sums
// the tile.  Per-block partial matrices are added in a fixed order by k6_fisher_final:
// deterministic, no atomics.
struct K6Params {
  int D;
  long long nf, kmin, nk;  // nk = kmax - kmin + 1 bins per channel
  const double2* spec;     // [D+1][3][M] packed
  double two_pi_over_N;
  const double* weight;    // [3][nf]
  double* partial;         // [gridDim.x][D*D]
  double inv_delta[K6_MAXD];
};

__global__ void __launch_bounds__(K6_THREADS) k6_fisher_partial(const K6Params p) {
  extern __shared__ double2 dsh[];               // [D][K6_TILE]
  __shared__ double wsh[K6_TILE];
  const int D = p.D, npairs = D * (D + 1) / 2;
  const long long items = 3 * p.nk;
  const long long ntiles = (items + K6_TILE - 1) / K6_TILE;
  // pairs owned by this thread: p0, p0 + K6_THREADS, ... (at most 3 for D <= 32)
  double acc[3] = {0.0, 0.0, 0.0};
  for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    __syncthreads();  // previous tile fully consumed
    if (threadIdx.x < K6_TILE) {
      const long long it = tile * K6_TILE + threadIdx.x;
      double w = 0.0;
      if (it < items) {
        const int c = (int)(it / p.nk);
        const long long k = p.kmin + (it - (long long)c * p.nk);
        w = p.weight[(size_t)c * p.nf + k];
        const long long M = p.nf - 1;
        double cw, sw;
        bin_twiddle(k, p.two_pi_over_N, cw, sw);
        const double2 h0 = packed_bin(p.spec + (size_t)c * M, M, k, cw, sw);
        for (int i = 0; i < D; ++i) {
          const double2 hi = packed_bin(p.spec + ((size_t)(i + 1) * 3 + c) * M, M, k, cw, sw);
          dsh[i * K6_TILE + threadIdx.x] = make_double2((hi.x - h0.x) * p.inv_delta[i], (hi.y - h0.y) * p.inv_delta[i]);
        }
      } else {
        for (int i = 0; i < D; ++i) dsh[i * K6_TILE + threadIdx.x] = make_double2(0.0, 0.0);
      }
      wsh[threadIdx.x] = w;
    }
    __syncthreads();
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      const int pr = threadIdx.x + s * K6_THREADS;
      if (pr >= npairs) break;
      // pair index -> (i, j), i <= j, row-major upper triangle
      int i = 0, rem = pr;
      while (rem >= D - i) { rem -= D - i; ++i; }
      const int j = i + rem;
      const double2* di = dsh + i * K6_TILE;
      const double2* dj = dsh + j * K6_TILE;
      double sum = 0.0;
      for (int t = 0; t < K6_TILE; ++t) sum = fma(wsh[t], fma(di[t].x, dj[t].x, di[t].y * dj[t].y), sum);
      acc[s] += sum;
    }
  }
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    const int pr = threadIdx.x + s * K6_THREADS;
    if (pr < npairs) p.partial[(size_t)blockIdx.x * (K6_MAXD * K6_MAXD) + pr] = acc[s];
  }
}

__global__ void k6_fisher_final(const double* __restrict__ partial, int nblocks, int D, double* fisher) {
  const int pr = blockIdx.x * blockDim.x + threadIdx.x;
  if (pr >= D * (D + 1) / 2) return;
  double sum = 0.0;
  for (int b = 0; b < nblocks; ++b) sum += partial[(size_t)b * (K6_MAXD * K6_MAXD) + pr];
  int i = 0, rem = pr;
  while (rem >= D - i) { rem -= D - i; ++i; }
  const int j = i + rem;
  fisher[(size_t)i * D + j] = sum;
  fisher[(size_t)j * D + i] = sum;
}

static int check_fft(cufftResult r, const char* what) {
  if (r == CUFFT_SUCCESS) return LISA_TD_OK;
  return set_error(LISA_TD_ECUDA, "%s failed: cufftResult %d", what, (int)r);
}

// single != 0: one channel per walker (input and output strides of three rows), executed once
// per selected channel; otherwise all 3B rows in one batch.
static int get_fft(Plan* pl, int B, cufftHandle* h, int single = 0) {
  const int key = 2 * B + (single ? 1 : 0);
  auto it = pl->fft.find(key);
  if (it != pl->fft.end()) {
    *h = it->second;
    return LISA_TD_OK;
  }
  cufftHandle f;
  int rc = check_fft(cufftCreate(&f), "cufftCreate");
  if (rc != LISA_TD_OK) return rc;
  long long n[1] = {pl->N / 2};
  size_t ws = 0;
  long long embed[1] = {pl->N / 2};
  const long long dist = single ? 3 * (pl->N / 2) : pl->N / 2;
  rc = check_fft(cufftSetAutoAllocation(f, 0), "cufftSetAutoAllocation");
  if (rc == LISA_TD_OK)
    rc = check_fft(cufftMakePlanMany64(f, 1, n, embed, 1, dist, embed, 1, dist, CUFFT_Z2Z, single ? (long long)B : 3LL * B, &ws),
                   "cufftMakePlanMany64");
  if (rc == LISA_TD_OK && ws > pl->work_bytes) {
    // a larger work area than any plan so far needed (normally only the capacity plan made in
    // lisa_td_plan_create gets here): wait for work that may still use the old one, then replace it
    rc = check_cuda(cudaDeviceSynchronize(), "cudaDeviceSynchronize");
    void* nw = nullptr;
    if (rc == LISA_TD_OK) rc = check_cuda(cudaMalloc(&nw, ws), "cudaMalloc(cuFFT work area)");
    if (rc == LISA_TD_OK) {
      cudaFree(pl->work);
      pl->work = nw;
      pl->work_bytes = ws;
      for (auto& kv : pl->fft)
        if (rc == LISA_TD_OK) rc = check_fft(cufftSetWorkArea(kv.second, pl->work), "cufftSetWorkArea");
    }
  }
  if (rc == LISA_TD_OK && ws > 0) rc = check_fft(cufftSetWorkArea(f, pl->work), "cufftSetWorkArea");
  if (rc != LISA_TD_OK) {
    cufftDestroy(f);
    return rc;
  }
  if ((int)pl->fft.size() >= K5_MAX_PLANS) {
    // bounded cache: drop every plan but the capacity plan (key 2 * pl->B); they are re-made on demand
    for (auto it2 = pl->fft.begin(); it2 != pl->fft.end();) {
      if (it2->first != 2 * pl->B) {
        cufftDestroy(it2->second);
        it2 = pl->fft.erase(it2);
      } else {
        ++it2;
      }
    }
  }
  pl->fft[key] = f;
  *h = f;
  return LISA_TD_OK;
}

int plan_destroy(Plan* pl);

int plan_create(Plan** out, int B, long long N) {
  Plan* pl = new Plan();
  pl->B = B; pl->N = N; pl->nf = N / 2 + 1; pl->spec = nullptr; pl->partial = nullptr; pl->fisher_partial = nullptr;
  pl->work = nullptr; pl->work_bytes = 0;
  int rc = check_cuda(cudaMalloc(&pl->spec, sizeof(double2) * (size_t)B * 3 * pl->nf), "cudaMalloc(spec)");
  if (rc == LISA_TD_OK) rc = check_cuda(cudaMalloc(&pl->partial, sizeof(double2) * (size_t)B * K5_SLICES), "cudaMalloc(partial)");
  cufftHandle h;
  if (rc == LISA_TD_OK) rc = get_fft(pl, B, &h);
  if (rc != LISA_TD_OK) {
    plan_destroy(pl);
    return rc;
  }
  *out = pl;
  return LISA_TD_OK;
}

int plan_destroy(Plan* pl) {
  if (!pl) return LISA_TD_OK;
  for (auto& kv : pl->fft) cufftDestroy(kv.second);
  cudaFree(pl->spec);
  cudaFree(pl->partial);
  cudaFree(pl->fisher_partial);
  cudaFree(pl->work);
  delete pl;
  return LISA_TD_OK;
}

// FFT of B <= capacity walkers.  A plan for a batch size not seen before is created on first
// use (host work inside cuFFT; no device allocation unless it needs a larger work area than the
// capacity plan).  The cuFFT handles carry the stream of the last call: a lisa_td_plan must not
// be used from two host threads at once.
static int run_fft(Plan* pl, int B, const double* tdi, double2* spec, cudaStream_t st, int n_ch = 3) {
  if (B > pl->B) return set_error(LISA_TD_EINVAL, "B=%d exceeds the plan's capacity %d", B, pl->B);
  cufftHandle h;
  int rc = get_fft(pl, B, &h, n_ch < 3);
  if (rc != LISA_TD_OK) return rc;
  rc = check_fft(cufftSetStream(h, st), "cufftSetStream");
  if (rc != LISA_TD_OK) return rc;
  if (n_ch < 3) {  // only the selected channels are transformed
    for (int c = 0; c < n_ch; ++c) {
      rc = check_fft(cufftExecZ2Z(h, reinterpret_cast<cufftDoubleComplex*>(const_cast<double*>(tdi)) + (size_t)c * (pl->N / 2),
                                  reinterpret_cast<cufftDoubleComplex*>(spec) + (size_t)c * (pl->N / 2), CUFFT_FORWARD),
                     "cufftExecZ2Z");
      if (rc != LISA_TD_OK) return rc;
    }
    return LISA_TD_OK;
  }
  return check_fft(cufftExecZ2Z(h, reinterpret_cast<cufftDoubleComplex*>(const_cast<double*>(tdi)),
                                reinterpret_cast<cufftDoubleComplex*>(spec), CUFFT_FORWARD),
                   "cufftExecZ2Z");
}
// full real-input spectrum [rows][nf] from the packed spectra [rows][M] (not on the timed path)
__global__ void k5_unpack_spectrum(const double2* __restrict__ Z, long long rows, long long nf, double two_pi_over_N,
                                   double2* __restrict__ out) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nf) return;
  double cw, sw;
  bin_twiddle(k, two_pi_over_N, cw, sw);
  for (long long row = blockIdx.y; row < rows; row += gridDim.y)  // grid.y is capped at 65535
    out[(size_t)row * nf + k] = packed_bin(Z + (size_t)row * (nf - 1), nf - 1, k, cw, sw);
}

int run_spectrum(Plan* pl, int B, long long N, const double* tdi, double* spec, cudaStream_t st) {
  if (N != pl->N) return set_error(LISA_TD_EINVAL, "spectrum: N differs from the plan's");
  int rc = run_fft(pl, B, tdi, pl->spec, st);
  if (rc != LISA_TD_OK) return rc;
  dim3 grid((unsigned)((pl->nf + 255) / 256), (unsigned)(3 * B < 65535 ? 3 * B : 65535));
  k5_unpack_spectrum<<<grid, 256, 0, st>>>(pl->spec, 3LL * B, pl->nf, 6.283185307179586476925 / (double)N,
                                           reinterpret_cast<double2*>(spec));
  LISA_LAUNCH_CHECK("k5_unpack_spectrum");
  return LISA_TD_OK;
}

int run_loglike(Plan* pl, int B, long long N, const double* tdi, const double* data_spec,
                const double* weight, long long kmin, long long kmax, double* loglike, double* dh,
                double* hh, cudaStream_t st, int n_ch) {
  if (N != pl->N) return set_error(LISA_TD_EINVAL, "loglike: N differs from the plan's");
  int rc = run_fft(pl, B, tdi, pl->spec, st, n_ch);
  if (rc != LISA_TD_OK) return rc;
  dim3 grid(K5_SLICES, (unsigned)B);
  k5_inner_partial<<<grid, K5_THREADS, 0, st>>>(pl->spec, reinterpret_cast<const double2*>(data_spec), weight,
                                                pl->nf, kmin, kmax, 6.283185307179586476925 / (double)N, pl->partial, n_ch);
  LISA_LAUNCH_CHECK("k5_inner_partial");
  k5_inner_final<<<(B + 127) / 128, 128, 0, st>>>(pl->partial, B, loglike, dh, hh);
  LISA_LAUNCH_CHECK("k5_inner_final");
  return LISA_TD_OK;
}

// tdi: [D+1][3][N] (walker 0 = centre, walker i = theta + delta_i e_i) -> fisher [D][D]
int run_fisher(Plan* pl, int D, long long N, const double* tdi, const double* delta_host, const double* weight,
               long long kmin, long long kmax, double* fisher, cudaStream_t st) {
  if (N != pl->N) return set_error(LISA_TD_EINVAL, "fisher: N differs from the plan's");
  if (D < 1 || D > K6_MAXD) return set_error(LISA_TD_EINVAL, "fisher: D must be in [1,%d]", K6_MAXD);
  if (D + 1 > pl->B) return set_error(LISA_TD_EINVAL, "fisher: D+1=%d walkers exceed the plan's capacity %d", D + 1, pl->B);
  K6Params p;
  for (int i = 0; i < K6_MAXD; ++i) p.inv_delta[i] = 0.0;
  for (int i = 0; i < D; ++i) {
    if (delta_host[i] == 0.0) return set_error(LISA_TD_EINVAL, "fisher: delta[%d] is zero", i);
    p.inv_delta[i] = 1.0 / delta_host[i];
  }
  if (!pl->fisher_partial)
    LISA_CUDA(cudaMalloc(&pl->fisher_partial, sizeof(double) * (size_t)K6_BLOCKS * K6_MAXD * K6_MAXD));
  int rc = run_fft(pl, D + 1, tdi, pl->spec, st);
  if (rc != LISA_TD_OK) return rc;
  p.D = D; p.nf = pl->nf; p.kmin = kmin; p.nk = kmax - kmin + 1;
  p.spec = pl->spec; p.weight = weight; p.partial = pl->fisher_partial;
  p.two_pi_over_N = 6.283185307179586476925 / (double)N;
  const long long ntiles = (3 * p.nk + K6_TILE - 1) / K6_TILE;
  const int nblocks = (int)(ntiles < K6_BLOCKS ? ntiles : K6_BLOCKS);
  const size_t smem = (size_t)D * K6_TILE * sizeof(double2);
  if (smem > 48 * 1024)
    LISA_CUDA(cudaFuncSetAttribute(k6_fisher_partial, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k6_fisher_partial<<<nblocks, K6_THREADS, smem, st>>>(p);
  LISA_LAUNCH_CHECK("k6_fisher_partial");
  k6_fisher_final<<<(D * (D + 1) / 2 + 127) / 128, 128, 0, st>>>(pl->fisher_partial, nblocks, D, fisher);
  LISA_LAUNCH_CHECK("k6_fisher_final");
  return LISA_TD_OK;
}

}  // namespace lisa
