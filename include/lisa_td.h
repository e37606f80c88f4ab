/*
 * lisa_td.h -- C ABI of liblisa_td.so: the per-likelihood hot path of the time-domain LISA
 * pipeline of arXiv:2501.08261 on one NVIDIA B200 (sm_100a).
 *
 *   S1  modes -> h+, hx              Eq. 2.1-2.6   (psi at PAPER.md:306)
 *   S2  h+, hx -> six link responses Eq. 2.7-2.8   (orbits PAPER.md:134)
 *   S3  links -> TDI X,Y,Z -> A,E,T  Eq. 2.9-2.11  (interpolation PAPER.md:209)
 *   S4  FFT of A,E,T (cuFFT)
 *   S5  inner products -> log L      Eq. 2.12-2.13 (band PAPER.md:243)
 *
 * The readings taken where the paper is silent or garbled are listed in DESIGN.md section 2
 * (A1..A22); the comments below name the ones each call depends on.
 *
 * General conventions
 *  - Every array pointer is a DEVICE pointer unless its name ends in _host.  All arrays are
 *    fp64, row-major, time fastest, and must be 16-byte aligned (LISA_TD_EALIGN otherwise).
 *  - The caller owns every buffer.  The library allocates device memory only inside a
 *    lisa_td_plan.  Inputs are never modified.
 *  - Every call only ENQUEUES work on `stream` (a cudaStream_t passed as void*; NULL = the
 *    legacy default stream) and returns without synchronising, except lisa_td_plan_create /
 *    lisa_td_plan_destroy, lisa_td_orbit_table_create, lisa_td_pipeline_host and lisa_td_check,
 *    which synchronise.  The enqueue-only calls may therefore be captured into a CUDA graph and
 *    replayed (tests/test_gpu_graph.py; call lisa_td_loglike once with the batch size before
 *    capturing: the first use of a batch size creates its cuFFT plan).
 *  - Return value: LISA_TD_OK (0) or a negative lisa_td_status.  Argument errors are detected
 *    on the host before any launch.  The library never throws, aborts or falls back to the
 *    CPU.  lisa_td_last_error() returns a thread-local description of the last failure.
 *  - Device-side range checks.  Tile and window sizes of S2 / S3 follow from host-side bounds on the
 *    orbit (max |r|, max L, drift of the common delay; for a TABLE orbit taken from its nodes).  A
 *    kernel that meets a delay outside those bounds does not clamp silently: it raises a sticky
 *    flag, and the next lisa_td_check / lisa_td_pipeline_host returns LISA_TD_EINVAL (the outputs
 *    written since the previous check are then invalid).
 *  - Walkers b = 0..B-1, samples n = 0..N-1 at t_n = t0 + n*dt, `order` p odd in [1,63]
 *    (p+1 Lagrange taps; p = 1 is the paper's linear interpolation).
 *  - Link order everywhere: l = [1,2,3,-1,-2,-3] <-> (sender,receiver) =
 *    [(3,2),(1,3),(2,1),(2,3),(3,1),(1,2)]  (y_{slr} notation of PAPER.md:132).
 *
 * Fractional-delay read (O-I of DESIGN.md): x(n - D) = sum_{j=-h+1..h} c_j(eps) x[n - K + j],
 * K = ceil(D), eps = K - D, h = (p+1)/2, c_j(eps) = prod_{i != j} (eps - i)/(j - i), x = 0
 * outside [0,N).
 */
#ifndef LISA_TD_H
#define LISA_TD_H

#if defined(__GNUC__)
#define LISA_TD_API __attribute__((visibility("default")))
#else
#define LISA_TD_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LISA_TD_OK = 0,
  LISA_TD_EINVAL = -1,   /* bad argument value (sizes, order, margins, NULL where not allowed) */
  LISA_TD_EALIGN = -2,   /* a device pointer is not 16-byte aligned */
  LISA_TD_ENOMEM = -3,   /* allocation failed / workspace too small */
  LISA_TD_ECUDA = -4,    /* a CUDA or cuFFT call failed (see lisa_td_last_error) */
  LISA_TD_ENOTIMPL = -5
} lisa_td_status;

LISA_TD_API const char* lisa_td_last_error(void);
LISA_TD_API int lisa_td_version(void);

/* Synchronises `stream` and reports (then clears) the device-side range checks raised by the
 * kernels since the last check: LISA_TD_OK, LISA_TD_EINVAL (see "Device-side range checks" above)
 * or LISA_TD_ECUDA if the stream itself failed. */
LISA_TD_API int lisa_td_check(void* stream);

/* Orbit description (host struct, copied at call time).
 * kind 0 = STATIC : spacecraft positions r_static[spacecraft][xyz] in metres and the six light
 *                   travel times L_static (seconds, link order) are constants.
 * kind 1 = KEPLER1: reading A8 of DESIGN.md (analytic orbits, first-order solution of Kepler's
 *                   equation, breathing unequal arms; L_l(t) = |r_r(t) - r_s(t)|/c).
 * kind 2 = TABLE  : reading A21 (orbits "tracked over the whole observation period",
 *                   e.g. an ESA orbit file): spacecraft positions tabulated on a uniform time
 *                   grid, held in a lisa_td_orbit_table; per sample they are interpolated with a
 *                   Lagrange polynomial of odd degree q on the q+1 nodes j0..j0+q,
 *                   j0 = floor((t - t_tab0)/dt_tab) - (q-1)/2 clamped to the table;
 *                   L_l(t) = |r_r(t) - r_s(t)|/c.  The table must cover [t0, t0 + N dt].
 *
 * Delay model (reading A22 of DESIGN.md):
 * tt_order   0: L_l(t) = |r_r(t) - r_s(t)|/c as above.
 *            1: first order in v/c of  c L = |r_r(t) - r_s(t - L)|:
 *               L_l(t) = (d/c)(1 + n.v_s/c), d = |r_r - r_s|, n = (r_r - r_s)/d, v_s = velocity of the
 *               sender (analytic for KEPLER1, derivative of the interpolant for TABLE), all at the
 *               reception time t, so that L_l != L_{-l}.  Used by S2, S3 and the laser helper.
 *               STATIC ignores it (its six L are given).
 * tdi_nested 0: every TDI delay is the SUM of the listed L_l(t_n), all at the output time (A10).
 *            1: every TDI delay is CHAINED along the light path traced back from the output time:
 *               tau_0 = 0, tau_{i+1} = tau_i + L_{l_i}(t_n - tau_i), labels in the order of the two
 *               paths 1<-2<-1<-3<-1<-3<-1<-2<-1 and 1<-3<-1<-2<-1<-2<-1<-3<-1 (for X; Y, Z cyclic),
 *               of which every delay of Eq. 2.9 / 2.10 is a leading piece.  S3 only. */
typedef struct lisa_td_orbit_table lisa_td_orbit_table;
typedef struct {
  int kind;
  double L_m, a_m, year_s, phase0, t_ref;
  double r_static[3][3];
  double L_static[6];
  const lisa_td_orbit_table* table; /* kind 2 only */
  int tt_order;                     /* 0 | 1 */
  int tdi_nested;                   /* 0 | 1 */
} lisa_td_orbit;

/* Owns a device copy of the table (the only device memory the library holds besides plans).
 * r_host: [n_tab][3][3] = [node][spacecraft][xyz] in metres at t_tab0 + j dt_tab; interp_order q
 * odd in [1,15], n_tab > q.  create synchronises (one host-to-device copy). */
LISA_TD_API int lisa_td_orbit_table_create(lisa_td_orbit_table** out, int n_tab, double t_tab0, double dt_tab,
                               int interp_order, const double* r_host);
LISA_TD_API int lisa_td_orbit_table_destroy(lisa_td_orbit_table* table);

/* S1 -- Eq. 2.4-2.6 (single-sum form; readings A1-A6).
 *   h+ - i hx = e^{2 i psi} sum_k [ h_k frakD^l_{m,2}(R) + (-1)^l conj(h_k) frakD^l_{-m,2}(R) ] sqrt((2l+1)/4pi)
 *   h_k = amp_k e^{-i phase_k},  R = R(alpha,beta,gamma)(t) . R(euler0) . R(phi, iota, 0)
 * l_host/m_host: n_modes (<= 16) mode labels, 2 <= l <= 8, 0 <= m <= l (the -m partner is implied).
 * amp, phase: [B][n_modes][N].  alpha,beta,gamma: [B][N] each, or all three NULL (aligned spin).
 * |phase|, |alpha|, |gamma| must stay below 2^30 rad (1e9): the kernels reduce arguments with a
 * two-constant Cody-Waite step that is good to 6e-17 up to there (a months-long chirp reaches 1e6).
 * iota, phi, psi: [B].  euler0: [B][3] constant J->L0 angles or NULL.  hplus, hcross: [B][N]. */
LISA_TD_API int lisa_td_modes_to_pol(int B, long long N, int n_modes, const int* l_host, const int* m_host,
                         const double* amp, const double* phase, const double* alpha,
                         const double* beta, const double* gamma, const double* iota,
                         const double* phi, const double* psi, const double* euler0,
                         double* hplus, double* hcross, void* stream);

/* S2 -- Eq. 2.7-2.8 (readings A7, A8, A11).  For every link (s,l,r) and sample n, with r_i, L_l
 * at the reception time t_n:
 *   y = [ x+ (h+(n-Ds) - h+(n-Dr)) + 2 xx (hx(n-Ds) - hx(n-Dr)) ] / ( 2 (1 - k.n) ),
 *   Ds = (L_l + k.r_s/c)/dt, Dr = (k.r_r/c)/dt, fractional-delay reads of order p.
 * hplus, hcross: [B][N] on the output grid.  lambda, beta_sky: [B] ecliptic longitude/latitude.
 * y: [B][6][N]; samples outside [margin_y, N - margin_y) are written as exact zeros.
 * margin_y must cover the stencil reach: margin_y >= ceil(max|D|) + (p+1)/2 for the given orbit
 * (LISA_TD_EINVAL otherwise; the bound used is max_i |r_i|/c + max_l L_l). */
LISA_TD_API int lisa_td_link_response(int B, long long N, double t0, double dt, int order, long long margin_y,
                          const double* hplus, const double* hcross, const double* lambda,
                          const double* beta_sky, const lisa_td_orbit* orbit_host, double* y,
                          void* stream);

/* S2 with the paper's 10 s -> 5 s trick (the waveforms are sampled "every
 * Delta t = 10 s and then linearly interpolate[d] ... to generate the arm and TDI responses with
 * a sampling time of 5 s"; reading A20 of DESIGN.md).  hplus_c, hcross_c: [B][N/2+1] on the grid
 * t0 + i (2 dt) (e.g. lisa_td_modes_to_pol run on N/2+1 samples of the coarse modes); the strain
 * on the dt grid is x[2i] = c[i], x[2i+1] = (c[i] + c[i+1])/2, formed while the tile is staged
 * (never materialised).  N must be even; everything else as lisa_td_link_response.  Note the
 * row stride N/2+1: rows need not be 16-byte aligned, only the base pointers. */
LISA_TD_API int lisa_td_link_response_up2(int B, long long N, double t0, double dt, int order,
                              long long margin_y, const double* hplus_c, const double* hcross_c,
                              const double* lambda, const double* beta_sky,
                              const lisa_td_orbit* orbit_host, double* y, void* stream);

/* A12 -- link-level common laser noise y_l[n] = p(n - L_l(t_n)/dt) - p[n] (zero outside
 * [margin, N - margin)); p: [N], y: [6][N].  Used to check TDI laser-noise suppression. */
LISA_TD_API int lisa_td_laser_links(long long N, double t0, double dt, int order, long long margin,
                        const double* p, const lisa_td_orbit* orbit_host, double* y, void* stream);

/* S3 -- Eq. 2.9 (generation 15) / Eq. 2.10 with the y123 block corrected (generation 20, reading
 * A9), Y and Z by cyclic permutation, optionally A,E,T of Eq. 2.11.  Every delayed read is a
 * fractional-delay read of one y series at D = (sum of the listed L_l(t_n))/dt (A10: summed, all
 * L at the output time).  y: [B][6][N].  tdi: [B][3][N], out_kind 0 = X,Y,Z, 1 = A,E,T; samples
 * outside [margin_lo, N - margin_hi) are exact zeros.  Requires margin_lo >= ceil(7 Lmax/dt) +
 * (p+1)/2 (3 Lmax for generation 15) and margin_hi >= (p+1)/2.  If y came from
 * lisa_td_link_response with margin_y, the caller must ADD margin_y to both (reading A7: TDI must
 * not interpolate across the zeroed edge of y); this call cannot know margin_y and does not check
 * that, lisa_td_response_tdi and lisa_td_pipeline_host do.
 * Temporary memory: at orders 1 and 31 the walker-independent merged stencils of the call (13 KB
 * per 128 samples, plus a list of sample groups to recompute one by one) are drawn from the device's
 * stream-ordered memory pool (cudaMallocAsync / cudaFreeAsync on `stream`): no synchronisation, the
 * memory is released in stream order and the pool keeps the pages for the next call.  The call stays
 * capturable into a CUDA graph.  lisa_td_response_tdi keeps them in the caller's workspace instead. */
LISA_TD_API int lisa_td_tdi2(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
                 long long margin_lo, long long margin_hi, const double* y,
                 const lisa_td_orbit* orbit_host, double* tdi, void* stream);

/* S3 without any allocation -- lisa_td_tdi2 (same arguments, same kernels, same output) for callers
 * that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  The merged-stencil tables and the fix-up list that lisa_td_tdi2 draws from the memory
 * pool live in ONE file-scope device array of the library instead (about 7 MiB, held by every GPU
 * that loads the library until the process exits), sized for N <= LISA_TD_TDI2_STATIC_MAX_N samples;
 * a larger N is rejected with LISA_TD_EINVAL before anything is launched.  The call makes no
 * cudaMalloc / cudaFree / cudaMallocAsync and no allocating library call; the first call on each
 * device looks the array's address up (cudaGetSymbolAddress), so make that call before capturing.
 * Every call shares the array: it clears what must start at zero itself, and two calls that overlap
 * on the GPU (different streams without an ordering between them, or two host threads) RACE.
 * Device-side range checks of this entry point are kept in the array too, not in the words
 * lisa_td_check reads: check != 0 makes the call wait for `stream` and return LISA_TD_EINVAL if a
 * stencil left its window in this call or in an earlier call with check == 0 (then cleared);
 * check == 0 only enqueues (use this under capture). */
#define LISA_TD_TDI2_STATIC_MAX_N 65536
LISA_TD_API int lisa_td_tdi2_static(int B, long long N, double t0, double dt, int order, int generation, int out_kind,
                 long long margin_lo, long long margin_hi, const double* y,
                 const lisa_td_orbit* orbit_host, double* tdi, int check, void* stream);

/* S2+S3 in one call: h+,hx -> tdi.  This is lisa_td_link_response into `workspace` followed by
 * lisa_td_tdi2 from it: all six links of all B walkers make one round trip through HBM ([B][6][N]
 * doubles = 48 B N bytes; lisa_td_response_tdi_workspace_bytes returns that plus the anchor
 * tables of S3, ~100 B per sample), they just never appear in a caller array.  An on-chip fusion was prototyped and measured slower (DESIGN.md
 * section 9, profiles/r2_s1.md): both kernels are bound by fp64 arithmetic, not by the
 * round trip.  Requires margin_lo >= margin_y + reach and margin_hi >= margin_y + (p+1)/2. */
LISA_TD_API long long lisa_td_response_tdi_workspace_bytes(int B, long long N);
LISA_TD_API int lisa_td_response_tdi(int B, long long N, double t0, double dt, int order, long long margin_y,
                         int generation, int out_kind, long long margin_lo, long long margin_hi,
                         const double* hplus, const double* hcross, const double* lambda,
                         const double* beta_sky, const lisa_td_orbit* orbit_host, double* tdi,
                         void* workspace, long long workspace_bytes, void* stream);

/* S4+S5 plan: owns the cuFFT plans (batched complex-to-complex of length N/2 on the packed real
 * series, one per batch size seen, at most 8, sharing one work area), the spectrum scratch and the
 * partial-sum scratch for up to B walkers.  Not thread-safe: one host thread per plan at a time. */
typedef struct lisa_td_plan lisa_td_plan;
LISA_TD_API int lisa_td_plan_create(lisa_td_plan** out, int B, long long N);
LISA_TD_API int lisa_td_plan_destroy(lisa_td_plan* plan);

/* S4+S5 -- Eq. 2.12-2.13 (readings A13, A17):  H_c[k] = sum_n tdi_c[n] e^{-2 pi i k n/N},
 *   (d|h)_b = sum_c sum_{k=kmin..kmax} w_c[k] Re( D_c[k] conj(H_{b,c}[k]) ),
 *   (h|h)_b = sum_c sum_k w_c[k] |H_{b,c}[k]|^2,   log L_b = (d|h)_b - (h|h)_b / 2.
 * tdi: [B][3][N] (A,E,T); data_spec: [3][N/2+1][2] (re,im); weight: [3][N/2+1] =
 * 4 df dt^2 / S_c(f_k); 0 <= kmin <= kmax <= N/2.  loglike: [B]; dh, hh: [B] or NULL. */
LISA_TD_API int lisa_td_loglike(lisa_td_plan* plan, int B, long long N, const double* tdi,
                    const double* data_spec, const double* weight, long long kmin, long long kmax,
                    double* loglike, double* dh, double* hh, void* stream);

/* The same with a subset of the channels ("injections and recoveries were performed
 * using one (A), two (AE) and three (AET) TDI channels"): the sums over c run over the first
 * n_channels (1, 2 or 3) of A,E,T; the other channels of tdi are neither transformed nor read.
 * Layouts as above (tdi stays [B][3][N], data_spec and weight stay [3][...]). */
LISA_TD_API int lisa_td_loglike_channels(lisa_td_plan* plan, int B, long long N, int n_channels, const double* tdi,
                             const double* data_spec, const double* weight, long long kmin, long long kmax,
                             double* loglike, double* dh, double* hh, void* stream);

/* S1..S5 in one call from DEVICE inputs (the call a sampler makes per batch of walkers): modes ->
 * h+,hx -> six links -> TDI A,E,T of the given generation -> FFT -> log L, enqueued on `stream`
 * without synchronising.  Arguments as in lisa_td_modes_to_pol (no euler0), lisa_td_link_response,
 * lisa_td_tdi2 and lisa_td_loglike; margins as in lisa_td_response_tdi.  Every intermediate lives in
 * `workspace` (device, >= lisa_td_loglike_from_modes_workspace_bytes(B, N) bytes = 88 B N plus the
 * anchor tables of S3; 5.9 GB at B = 64, N = 2^20).  The stages run one after the other on the one
 * stream: every compute kernel of the path fills the register file of every SM, so chunking the
 * batch over a second stream to hide the FFT was measured and does not pay. */
LISA_TD_API long long lisa_td_loglike_from_modes_workspace_bytes(int B, long long N);
LISA_TD_API int lisa_td_loglike_from_modes(lisa_td_plan* plan, int B, long long N, int n_modes, const int* l_host,
                               const int* m_host, const double* amp, const double* phase, const double* alpha,
                               const double* beta, const double* gamma, const double* iota, const double* phi,
                               const double* psi, const double* lambda, const double* beta_sky, double t0,
                               double dt, int order, long long margin_y, int generation, long long margin_lo,
                               long long margin_hi, const lisa_td_orbit* orbit_host, const double* data_spec,
                               const double* weight, long long kmin, long long kmax, double* loglike, double* dh,
                               double* hh, void* workspace, long long workspace_bytes, void* stream);

/* Fisher matrix by first-order finite differences ("The Fisher matrix is computed
 * from the derivatives of the likelihood function, using first-order finite differences";
 * reading A19 of DESIGN.md).  tdi: [D+1][3][N] (A,E,T): walker 0 is the centre theta, walker
 * i = 1..D is theta + delta_i e_i, all run through S1..S3 by the caller.  With
 * d_i H = (H_i - H_0)/delta_i on the Fourier transforms,
 *   fisher[i][j] = (d_i h | d_j h) = sum_c sum_{k=kmin..kmax} w_c[k] Re(d_i H_c[k] conj(d_j H_c[k])).
 * delta_host: [D] host array, no zero entries.  1 <= D <= 32, D + 1 <= plan capacity.
 * fisher: [D][D] device, symmetric, written in full.  Deterministic (fixed summation order). */
LISA_TD_API int lisa_td_fisher(lisa_td_plan* plan, int D, long long N, const double* tdi,
                   const double* delta_host, const double* weight, long long kmin, long long kmax,
                   double* fisher, void* stream);

/* Spectrum only (used to build the zero-noise injection): tdi [B][3][N] ->
 * spec [B][3][N/2+1][2]. */
LISA_TD_API int lisa_td_spectrum(lisa_td_plan* plan, int B, long long N, const double* tdi, double* spec,
                     void* stream);

/* Host helper, outside the timed path: Eq. 2.14-2.15 with readings A14, A15, A17.
 * weight_host: [3][N/2+1] (A,E,T) = 4 df dt^2 / S_c(k df), 0 at k = 0; generation 20 multiplies
 * the PSDs by 4 sin^2(4 pi f arm_s). */
LISA_TD_API int lisa_td_psd_weights(long long N, double dt, double acc_noise, double oms_noise, double arm_s,
                        int generation, double* weight_host);

/* Whole path S1..S5 from HOST buffers (the end-to-end call).  All *_host arrays are host memory
 * (pinned for full copy bandwidth); layouts as in the calls above.  Walkers are processed in
 * chunks of the plan's capacity; host->device copies of chunk i+1 overlap the kernels of chunk
 * i on two internal streams.  Synchronises before returning.  alpha/beta/gamma_host may all be
 * NULL.  loglike_host: [B]; dh_host, hh_host: [B] or NULL. */
typedef struct lisa_td_pipeline lisa_td_pipeline;
LISA_TD_API int lisa_td_pipeline_create(lisa_td_pipeline** out, int chunk_B, long long N, int n_modes,
                            int twisted);
LISA_TD_API int lisa_td_pipeline_destroy(lisa_td_pipeline* p);
LISA_TD_API int lisa_td_pipeline_host(lisa_td_pipeline* p, int B, long long N, int n_modes, const int* l_host,
                          const int* m_host, const double* amp_host, const double* phase_host,
                          const double* alpha_host, const double* beta_host,
                          const double* gamma_host, const double* iota_host,
                          const double* phi_host, const double* psi_host,
                          const double* lambda_host, const double* beta_sky_host, double t0,
                          double dt, int order, long long margin_y, int generation,
                          long long margin_lo, long long margin_hi,
                          const lisa_td_orbit* orbit_host, const double* data_spec_host,
                          const double* weight_host, long long kmin, long long kmax,
                          double* loglike_host, double* dh_host, double* hh_host);

/* The same with the paper's 10 s -> 5 s trick (reading A20): amp/phase_host are
 * [B][n_modes][N/2+1] and alpha/beta/gamma_host [B][N/2+1], sampled on the grid t0 + i (2 dt); S1 runs
 * on that grid and S2 interpolates h+, hx linearly to the dt grid (lisa_td_link_response_up2).  Half
 * the bytes cross PCIe.  Everything else (N, margins, data, weights, outputs) as above. */
LISA_TD_API int lisa_td_pipeline_host_up2(lisa_td_pipeline* p, int B, long long N, int n_modes, const int* l_host,
                              const int* m_host, const double* amp_host, const double* phase_host,
                              const double* alpha_host, const double* beta_host,
                              const double* gamma_host, const double* iota_host,
                              const double* phi_host, const double* psi_host,
                              const double* lambda_host, const double* beta_sky_host, double t0,
                              double dt, int order, long long margin_y, int generation,
                              long long margin_lo, long long margin_hi,
                              const lisa_td_orbit* orbit_host, const double* data_spec_host,
                              const double* weight_host, long long kmin, long long kmax,
                              double* loglike_host, double* dh_host, double* hh_host);

#ifdef __cplusplus
}
#endif
#endif /* LISA_TD_H */
