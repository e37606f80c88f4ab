// k5_loglike.cu -- S4 + S5: forward FFT of A,E,T (cuFFT, the one library call on the path,
// PAPER.md:211, 404) and the band-limited noise-weighted inner products -> log L
// (Eq. 2.12-2.13; readings A13, A17; band PAPER.md:243).
//
//   (d|h)_b = sum_c sum_{k=kmin..kmax} w_c[k] Re(D_c[k] conj(H_{b,c}[k]))
//   (h|h)_b = sum_c sum_k w_c[k] |H_{b,c}[k]|^2         log L_b = (d|h)_b - (h|h)_b / 2
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

struct Plan {
  int B;  // capacity (walkers)
  long long N, nf;
  std::map<int, cufftHandle> fft;  // batched D2Z plans keyed by the number of walkers
  double2* spec;     // [B][3][nf]
  double2* partial;  // [B][K5_SLICES]
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(K5_THREADS) k5_inner_partial(
    const double2* __restrict__ spec, const double2* __restrict__ data,
    const double* __restrict__ weight, long long nf, long long kmin, long long kmax,
    double2* __restrict__ partial) {
  const int b = blockIdx.y, slice = blockIdx.x;
  const long long nk = kmax - kmin + 1;
  const long long per = (nk + K5_SLICES - 1) / K5_SLICES;
  const long long k0 = kmin + (long long)slice * per;
  const long long k1 = min(k0 + per, kmax + 1);
  double dh = 0.0, hh = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double2* H = spec + ((size_t)b * 3 + c) * nf;
    const double2* D = data + (size_t)c * nf;
    const double* W = weight + (size_t)c * nf;
    double dhc = 0.0, hhc = 0.0;
    for (long long k = k0 + threadIdx.x; k < k1; k += K5_THREADS) {
      const double2 h = H[k], d = D[k];
      const double w = W[k];
      dhc = fma(w, fma(d.x, h.x, d.y * h.y), dhc);
      hhc = fma(w, fma(h.x, h.x, h.y * h.y), hhc);
    }
    dh += dhc;
    hh += hhc;
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

static int check_fft(cufftResult r, const char* what) {
  if (r == CUFFT_SUCCESS) return LISA_TD_OK;
  return set_error(LISA_TD_ECUDA, "%s failed: cufftResult %d", what, (int)r);
}

static int get_fft(Plan* pl, int B, cufftHandle* h) {
  auto it = pl->fft.find(B);
  if (it != pl->fft.end()) {
    *h = it->second;
    return LISA_TD_OK;
  }
  cufftHandle f;
  int rc = check_fft(cufftCreate(&f), "cufftCreate");
  if (rc != LISA_TD_OK) return rc;
  long long n[1] = {pl->N};
  size_t ws = 0;
  rc = check_fft(cufftMakePlanMany64(f, 1, n, nullptr, 1, pl->N, nullptr, 1, pl->nf, CUFFT_D2Z, 3LL * B, &ws),
                 "cufftMakePlanMany64");
  if (rc != LISA_TD_OK) {
    cufftDestroy(f);
    return rc;
  }
  pl->fft[B] = f;
  *h = f;
  return LISA_TD_OK;
}

int plan_destroy(Plan* pl);

int plan_create(Plan** out, int B, long long N) {
  Plan* pl = new Plan();
  pl->B = B; pl->N = N; pl->nf = N / 2 + 1; pl->spec = nullptr; pl->partial = nullptr;
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
  delete pl;
  return LISA_TD_OK;
}

// FFT of B <= capacity walkers.  A plan for a batch size not seen before is created on first
// use (that call synchronises inside cuFFT).
static int run_fft(Plan* pl, int B, const double* tdi, double2* spec, cudaStream_t st) {
  if (B > pl->B) return set_error(LISA_TD_EINVAL, "B=%d exceeds the plan's capacity %d", B, pl->B);
  cufftHandle h;
  int rc = get_fft(pl, B, &h);
  if (rc != LISA_TD_OK) return rc;
  rc = check_fft(cufftSetStream(h, st), "cufftSetStream");
  if (rc != LISA_TD_OK) return rc;
  return check_fft(cufftExecD2Z(h, const_cast<double*>(tdi), reinterpret_cast<cufftDoubleComplex*>(spec)), "cufftExecD2Z");
}
int run_spectrum(Plan* pl, int B, long long N, const double* tdi, double* spec, cudaStream_t st) {
  if (N != pl->N) return set_error(LISA_TD_EINVAL, "spectrum: N differs from the plan's");
  return run_fft(pl, B, tdi, reinterpret_cast<double2*>(spec), st);
}

int run_loglike(Plan* pl, int B, long long N, const double* tdi, const double* data_spec,
                const double* weight, long long kmin, long long kmax, double* loglike, double* dh,
                double* hh, cudaStream_t st) {
  if (N != pl->N) return set_error(LISA_TD_EINVAL, "loglike: N differs from the plan's");
  int rc = run_fft(pl, B, tdi, pl->spec, st);
  if (rc != LISA_TD_OK) return rc;
  dim3 grid(K5_SLICES, (unsigned)B);
  k5_inner_partial<<<grid, K5_THREADS, 0, st>>>(pl->spec, reinterpret_cast<const double2*>(data_spec), weight,
                                                pl->nf, kmin, kmax, pl->partial);
  LISA_LAUNCH_CHECK("k5_inner_partial");
  k5_inner_final<<<(B + 127) / 128, 128, 0, st>>>(pl->partial, B, loglike, dh, hh);
  LISA_LAUNCH_CHECK("k5_inner_final");
  return LISA_TD_OK;
}

}  // namespace lisa
