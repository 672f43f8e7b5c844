/* tb.h -- C ABI of libtb: template-bank binary-pulsar search, per-template hot path on one
 * NVIDIA B200 (sm_100a).  Method: Balakrishnan et al., arXiv:2112.11991; citations below are
 * lines of PAPER.md (the paper text) and readings G<n> of DESIGN.md section 3.
 *
 * For every orbital template the library
 *   a1  derives per-template constants and the zero offset            (Alg. 1)
 *   a2  evaluates the Roemer delay of every output sample             (eq A1, eq 3,
 *       circular closed form or per-sample Kepler solve                Alg. 1)
 *   a3  gathers the nearest input sample (nearest-neighbour resampling) (L664, L702)
 *   a4  takes the real-to-complex FFT                                   (L144, L706)
 *   a5  forms the interbinned power spectrum                            (G12-G14)
 *   a6  takes block medians, a7 normalises by the interpolated median   (L660 "de-reddening", G15)
 *   a8  sums 1, 2, 4, 8, 16 harmonics                                   (eq 9, G16)
 *   a9  thresholds in sigma and compacts candidates on the device       (eq 11, G17, G19)
 *   a10 returns the candidate list sorted by (template, fold, bin).
 * All of a1-a9 run in hand-written CUDA kernels plus one batched cuFFT R2C call; there is no CPU
 * fallback: every entry point that needs the GPU fails with TB_ERR_CUDA when none is usable.
 *
 * Conventions
 *   - Every function returns TB_OK (0) or a negative TB_ERR_* code; nothing throws, aborts or
 *     prints.  tb_last_error(plan) gives a detail string owned by the plan (valid until the next
 *     call on that plan); tb_strerror(code) a static string.
 *   - "host" pointers are ordinary CPU memory, "device" pointers are CUDA device memory on the
 *     plan's device.  The caller owns every buffer it passes in or receives results in; the
 *     plan owns all memory it allocates and frees it in tb_plan_destroy.
 *   - Work is queued on the plan's stream (opts.stream, or a stream the plan creates).
 *     tb_search_templates returns once the work is queued (host template staging is complete);
 *     tb_get_candidates / tb_get_timings / tb_debug_* synchronise that stream.
 *   - No global state in the library (one exception: the static scratch array of
 *     tb_series_mean_noalloc, see there) and no environment variables; plans are independent; one
 *     plan must not be used from two threads at once.  Two device-wide side effects, both of
 *     performance only: tb_plan_create RAISES cudaLimitPersistingL2CacheSize to the size of the
 *     series if it is smaller (it is never lowered or reset, so other plans keep their L2 set-aside),
 *     and it sets a persisting access-policy window for the series on the plan's stream; on a
 *     caller-owned stream (opts.stream) the window that stream had before is restored by
 *     tb_plan_destroy.
 */
#ifndef TB_H_
#define TB_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define TB_API __attribute__((visibility("default")))
#else
#define TB_API
#endif

#define TB_OK                 0
#define TB_ERR_INVALID_ARG   -1   /* null pointer, N not a power of two >= 2*W, tsamp <= 0, fold > 4, bad template */
#define TB_ERR_CUDA          -2   /* a CUDA runtime call failed (including "no device") */
#define TB_ERR_CUFFT         -3   /* a cuFFT call failed */
#define TB_ERR_NOMEM         -4   /* host or device allocation failed */
#define TB_ERR_OVERFLOW      -5   /* more candidates than opts.max_candidates were produced */
#define TB_ERR_CAPACITY      -6   /* caller's output buffer is too small; nothing was consumed */

#define TB_MAX_FOLD           4   /* folds L = 0..4 <=> 1, 2, 4, 8, 16 summed harmonics (eq 9) */

typedef struct tb_plan tb_plan;   /* opaque */

/* One orbital template ({tau, Omega, alpha, psi, e}; BASELINE's names).
 *   p_orb_s   orbital period P_orb = 2 pi / Omega, seconds, finite and > 0
 *   tau_lts   projected semi-major axis a sin(i)/c, light-seconds, >= 0
 *   phi0_rad  initial orbital phase alpha (mean anomaly at t = 0), radians, finite
 *   ecc       eccentricity e, 0 <= e < 1
 *   omega_rad longitude of periastron psi, radians, finite
 * ecc == 0 takes E = M without a Kepler solve: Delta = tau sin(Omega t + phi0 + omega_rad), which for
 * omega_rad == 0 is the circular closed form (eq 4 L49 / eq A1 at e = 0, G6); ecc > 0 takes the
 * Kepler solve of eq 3 + eq A1. */
typedef struct {
    double p_orb_s, tau_lts, phi0_rad, ecc, omega_rad;
} tb_template;                    /* 40 bytes */

/* One detection: S_L[bin] >= threshold (eq 9; G19).  The fundamental spin frequency of the
 * candidate is bin / (2^fold * N * tsamp) Hz (G16: bin indexes the highest summed harmonic). */
typedef struct {
    uint32_t template_id;         /* first_template_id + index in the tmpl array */
    uint32_t fold;                /* L, 0..4 */
    uint32_t bin;                 /* k, k_lo*2^L <= k < N/2 */
    float    power;               /* S_L[k], normalised summed power (fp32) */
    float    sigma;               /* (sqrt(S) - mu_n) / s_n, n = 2^L (eq 11 at n = 1; G17) */
    uint32_t pad;                 /* 0 */
} tb_candidate;                   /* 24 bytes */

/* Plan options.  Zero-initialise, set struct_size = sizeof(tb_plan_opts), then override.
 * A field left 0 takes the default in brackets. */
typedef struct {
    uint32_t struct_size;
    int32_t  device;              /* CUDA device ordinal [0] */
    void*    stream;              /* cudaStream_t to queue on; NULL -> the plan creates its own */
    uint32_t median_window;       /* W: power of two, 128..2048 [1024] (BASELINE C1) */
    double   f_min_hz;            /* lowest searched fundamental frequency [0.1] (G20); <0 -> 0 */
    uint64_t max_candidates;      /* capacity of the device candidate buffer [1<<22] */
    uint32_t chunk_templates;     /* templates per launch group B; 0 -> chosen from free memory */
    int32_t  series_is_device_ptr;/* 0: series is host memory; 1: series is device memory on
                                     `device`.  Either way the plan copies it (on its stream);
                                     the caller's buffer may be reused once the call returns and
                                     the stream has been synchronised (tb_get_candidates does) */
    int32_t  has_fill;            /* 0: out-of-range samples take the fp64 mean of the series,
                                     rounded to fp32 (G8); 1: they take fill_value */
    float    fill_value;
    int32_t  enable_timings;      /* 1: record CUDA events around every stage of every chunk */
    int32_t  fft_path;            /* 0: automatic (hand-written FFT with fused gather where it applies:
                                     2^17 <= N <= 2^26 (two passes up to 2^25, three at 2^26), W in
                                     {512, 1024, 2048} (256 or 1024 at 2^17; 1024 or 2048 at 2^25) and
                                     knot spacing >= 8; batched cuFFT otherwise); 1: always
                                     cuFFT; 2: hand-written or TB_ERR_INVALID_ARG */
    int32_t  whiten;              /* 1: front-end whitening once per series ("Fourier
                                     de-reddening", "birdie zapping"; reading G25): tb_plan_create and
                                     tb_plan_set_series replace the series by x' = C2R(X_k / sqrt(m(k)/ln2)) / sqrt(N)
                                     (m(k): the G15 baseline of the raw powers |X_k|^2, X'_0 = X'_{N/2} = 0, zapped
                                     ranges = 0; unit variance for noise), and every template is then normalised by
                                     ONE constant, P^_k = kappa P_k, kappa = ln2 / mean of the block medians of the
                                     interbinned spectrum of x' -- step a6 leaves the per-template loop */
    uint32_t n_zap_ranges;        /* number of zapped bin ranges (used only when whiten is set) */
    const uint32_t* zap_ranges;   /* host, 2 * n_zap_ranges values: [lo, hi) pairs, lo < hi <= N/2; copied */
    int32_t  delay_model;         /* 0: the paper's resampler, eq A1 with the Kepler solve ("BT model", L668);
                                     1: the ELL7 approximate orbit (eqs 15-16, App. B; reading
                                     G26): cos E and sqrt(1-e^2) sin E from the printed series through e^6, no Kepler
                                     solve; differs from 0 by about 1.2 e^7 tau (0.015 samples at e = 0.1, tau/tsamp =
                                     1.25e5), so a mode of its own with its own oracle, not bit-compatible with 0 */
    int32_t  interbin_oversample; /* 0: the interbinned spectrum of N/2 bins (G12); 1: the 2x-oversampled spectrum of
                                     N HALF bins (reading G12b; Ransom et al. 2002, the paper's reference for scalloping,
                                     L289): P'_2k = |X_k|^2, P'_2k+1 = (pi/4)^2 |X_k - X_k+1|^2.  Everything downstream
                                     counts half bins: W of them per median block, candidate.bin = half bin of the highest
                                     summed harmonic (fundamental frequency bin / (2^(fold+1) N tsamp) Hz), k_lo doubled,
                                     tb_debug_spectrum / tb_debug_hsums return N (5 N) values.  Library-FFT path only
                                     (fft_path 2 -> TB_ERR_INVALID_ARG), not with whiten, N <= 2^27 */
} tb_plan_opts;

/* Per-stage device time of the last tb_search_templates call (CUDA events on the plan's stream,
 * summed over chunks; zero unless opts.enable_timings), and the byte model of DESIGN.md section 7.
 *   hand-written FFT path (fft_path_used = 2)        cuFFT path (fft_path_used = 1)
 *   ms_delay     K0 k_delay_segments (a2 knots);     0
 *                from the second chunk on it runs on a
 *                side stream beside P2 / the spectrum
 *                former of the previous chunk: the span
 *                it was resident for, NOT additive
 *   ms_resample  P1 k_fft_cols32 / k_fft_cols        k_resample (a2+a3)
 *                (a2+a3 + a4 pass 1)
 *   ms_fft       P2 k_fft_rows_t / k_fft_rows_wide   batched cuFFT R2C (a4)
 *                (a4 pass 2; two kernels at N = 2^26)
 *   ms_spectrum  k_spectrum_t (a4 unpack, a5-a7)     k_spectrum_median (a5-a7)
 *   ms_hsum      k_hsum_tile (a8+a9)                 same
 * ms_normalise is always 0 (a7 is fused into the spectrum kernels); kept for layout stability. */
typedef struct {
    double   ms_resample, ms_fft, ms_spectrum, ms_normalise, ms_hsum, ms_total;
    uint64_t n_templates, n_samples, n_chunks, chunk_templates;
    uint64_t model_bytes_per_template;   /* 22*N: algorithmic HBM bytes */
    uint64_t n_kernel_launches;          /* libtb's own kernels launched by that call (cuFFT's not counted) */
    uint64_t n_median_fallbacks;         /* median blocks that took the data-independent bisection path */
    double   ms_delay;
    uint64_t fft_path_used;              /* bit 0: some templates went through k_resample + batched cuFFT; bit 1: some
                                            through the hand-written FFT with fused gather (a bank is split per template:
                                            knot spacing >= 8 samples -> fused path); 3 = both, and then the per-stage
                                            times above are sums over both kinds of chunk */
} tb_timings;

/* Create a plan for one dedispersed time series S[i], i*tsamp.
 *   out        receives the plan (set to NULL on failure)
 *   series     float32[n_samples], host or device memory per opts; copied into the plan
 *   n_samples  N, a power of two, 2*W <= N <= 2^28
 *   tsamp_s    sampling time in seconds, > 0
 *   opts       may be NULL (all defaults)
 * Allocates every device buffer the search needs (series, B resampled series, B spectra, the
 * candidate buffer, the cuFFT plan and its work area): TB_ERR_NOMEM if that does not fit. */
TB_API int tb_plan_create(tb_plan** out, const float* series, uint64_t n_samples, double tsamp_s,
                   const tb_plan_opts* opts);

/* Replace the plan's time series by another of the same length and sampling time (the next
 * DM trial / beam: PAPER.md L448, L660), reusing every buffer and FFT plan.  `series` is host
 * memory (copied on the plan's stream; pinned memory makes the copy asynchronous) unless the
 * plan was created with series_is_device_ptr, in which case it is device memory (copied device
 * to device).
 * The fill value is recomputed unless the plan was created with has_fill. */
TB_API int tb_plan_set_series(tb_plan* plan, const float* series);

/* Search `n_templates` templates (host array) and APPEND the detections to the plan's device
 * candidate buffer (steps a1-a9).  template_id of tmpl[i] is first_template_id + i.
 *   folds / n_folds   the harmonic folds to threshold: distinct values from {0,1,2,3,4}
 *   sigma_threshold   candidates have sigma_L >= sigma_threshold (finite)
 * Invalid templates make the whole call fail with TB_ERR_INVALID_ARG before any work is queued.
 * If a later step fails (TB_ERR_CUDA / TB_ERR_CUFFT / TB_ERR_NOMEM) the candidates of the chunks
 * that had already been queued REMAIN in the buffer; call tb_clear_candidates before retrying.
 * n_templates == 0 is valid and does nothing. */
TB_API int tb_search_templates(tb_plan* plan, const tb_template* tmpl, uint64_t n_templates,
                        uint32_t first_template_id, const uint32_t* folds, uint32_t n_folds,
                        double sigma_threshold);

/* Copy the accumulated candidates to `out` (host, capacity entries), sorted by
 * (template_id, fold, bin); *n_total receives the number produced since the last clear.
 *   out == NULL or capacity < count -> TB_ERR_CAPACITY, *n_total set, nothing consumed
 *   count > max_candidates          -> TB_ERR_OVERFLOW, *n_total = true count, the first
 *                                      max_candidates stored entries are returned if they fit
 * A successful full read clears the buffer (so does tb_clear_candidates). */
TB_API int tb_get_candidates(tb_plan* plan, tb_candidate* out, uint64_t capacity, uint64_t* n_total);
TB_API int tb_clear_candidates(tb_plan* plan);
TB_API int tb_plan_destroy(tb_plan* plan);      /* NULL is allowed */

/* ---- candidate reduction ("a candidate reduction algorithm by grouping together
 * multiple detections of the same candidate"; the paper gives no algorithm: reading G24) ----
 * One group = one signal.  R1: within a (template, fold) a run of detections in adjacent bins is one
 * peak (its detection of highest sigma; ties: lowest bin).  R2: peaks are ranked by sigma
 * (descending; ties: template, fold, bin).  R3: in rank order, a peak that has not been absorbed
 * heads a new group and absorbs every weaker unabsorbed peak, of any template and fold, whose
 * fundamental frequency f = bin / 2^fold (in bins of 1/T_obs) is harmonically related to its own:
 * |q f_b - p f_head| <= freq_tol_bins for some integers 1 <= p, q <= 16 (frequencies are held as
 * exact multiples of 1/16 bin).  Groups are numbered in head order. */
typedef struct {
    uint32_t template_id, fold, bin;   /* the group's head: its most significant detection */
    float    power, sigma;
    uint32_t n_peaks;                  /* peaks in the group (head included) */
    uint32_t n_detections;             /* raw detections in those peaks */
    uint32_t n_templates;              /* distinct templates among them */
} tb_group;                            /* 32 bytes */

/* Reduce the candidates accumulated in the plan (device side: sort, run scan, distillation) WITHOUT
 * consuming them: tb_get_candidates afterwards returns the same sorted list.
 *   freq_tol_bins    tolerance of R3 in fundamental bins; 0 -> 1.0; rounded to 1/16 bin
 *   groups_out       host, `capacity` entries; *n_groups receives the number of groups
 *   member_of        host, optional (NULL): group index of every detection, in the order
 *                    tb_get_candidates returns them (sorted by template, fold, bin);
 *                    member_capacity entries, must hold them all
 * TB_ERR_CAPACITY if groups_out is NULL or too small (*n_groups is set) or member_of too small;
 * TB_ERR_OVERFLOW if the candidate buffer overflowed (clear it and search with a higher threshold). */
TB_API int tb_reduce_candidates(tb_plan* plan, double freq_tol_bins, tb_group* groups_out, uint64_t capacity,
                         uint64_t* n_groups, uint32_t* member_of, uint64_t member_capacity);

/* Parity tap: REPLACE the plan's accumulated candidates by `n` rows from host memory (fold <= 4,
 * bin < N/2, n <= max_candidates), so that tb_reduce_candidates can be compared with the oracle on a
 * seeded synthetic detection list. */
TB_API int tb_debug_set_candidates(tb_plan* plan, const tb_candidate* cands, uint64_t n);

TB_API const char* tb_strerror(int code);
TB_API const char* tb_last_error(const tb_plan* plan);

/* ---- measurement and parity taps (not on the timed path) ---- */
TB_API int tb_get_timings(tb_plan* plan, tb_timings* out);

/* Source index idx_j = j - floor(delta_j + 1/2) of every output sample of one template, exactly
 * as the resampling kernel computes it (same device function), before the range check.
 * idx_out: host int64[N]. */
TB_API int tb_debug_resample_indices(tb_plan* plan, const tb_template* tmpl, int64_t* idx_out);

/* Spectra of one template through the production kernels: interbinned powers P_k (a5),
 * normalised powers P^_k (a7), both float32[N/2], and block medians float32[N/2/W] (a6).
 * Any output pointer may be NULL.  Host buffers. */
TB_API int tb_debug_spectrum(tb_plan* plan, const tb_template* tmpl, float* p_interbinned,
                      float* p_normalised, float* medians);

/* Resampled series y_j of one template (a3): host float32[N]. */
TB_API int tb_debug_resampled(tb_plan* plan, const tb_template* tmpl, float* y_out);

/* The plan's working copy of the series (host float32[N]; the whitened series when opts.whiten is
 * set) and the normalisation constant kappa of a whitened plan (0 otherwise).  Either may be NULL. */
TB_API int tb_debug_series(tb_plan* plan, float* x_out, double* kappa_out);

/* Harmonic sums of one template (a8; eq 9, G16) through the production summing kernel with its
 * tap enabled and every threshold at +infinity: sums_out[L * (N/2) + k] = S_L[k], L = 0..4,
 * k = 0..N/2-1; host float32[5 * N/2].  Emits no candidates. */
TB_API int tb_debug_hsums(tb_plan* plan, const tb_template* tmpl, float* sums_out);

/* Host fp64: the summed power at which sigma_L equals `sigma` (G17).  fold 0..4. */
TB_API int tb_sigma_to_power(uint32_t fold, double sigma, double* power_out);

/* Plan facts for harnesses: fill value in use, chunk size B, lowest bin k_lo, and the Hermite
 * knot spacing (log2, 0 = every sample exact) the resampler would choose for a template. */
TB_API int tb_plan_info(const tb_plan* plan, float* fill_value, uint32_t* chunk_templates, uint32_t* k_lo);
TB_API int tb_template_knot_log2(const tb_plan* plan, const tb_template* tmpl, int32_t* log2_h);

/* ---- random template bank (PAPER.md sections 2.2-2.7; readings G27-G29) ----
 * Plan-free: these calls own their device memory for the duration of the call, run on the default
 * stream of `device` and synchronise before returning.
 *
 * The density of templates is rho(lambda) = sqrt|det gamma_ab| (L115, L263), gamma the frequency-
 * projected metric (eq 22) of g_ab = <d_a Phi d_b Phi>_T - <d_a Phi>_T <d_b Phi>_T (eq 13,
 * time averages over [0, t_obs_s], eq 14) for the phase Phi = 2 pi f0 [t + tau X(t)] of eq 1-2
 * (L35-41), X = sin(psi) cos E + cos(psi) sqrt(1-e^2) sin E with the e-series of eqs 15-16 (L106-111,
 * App. B), or X = sin(Omega t + alpha) (eq 4) when elliptical == 0.  Coordinates
 * lambda = (tau [lt-s], Omega [rad/s], alpha [rad], psi [rad], e) (reading G27); f0 = f_max_hz (eq 30).
 * Time averages: composite 32-point Gauss-Legendre, 1024 nodes (4096 when the shortest orbit makes
 * more than 7 revolutions in t_obs_s; more than 28 revolutions -> TB_ERR_INVALID_ARG). */
typedef struct {
    uint32_t struct_size;         /* sizeof(tb_bank_space) */
    int32_t  device;              /* CUDA device ordinal */
    double   t_obs_s;             /* T of eq 14 */
    double   f_max_hz;            /* spin frequency the bank is built for (L140, eq 30) */
    double   p_orb_min_s, p_orb_max_s;        /* P_orb ~ U(min, max)              (Table 1) */
    double   m_pulsar_min, m_comp_max, theta; /* eq 31 (L248), solar masses; 0 < theta <= 1:
                                                 tau ~ U(0, theta (G M_sun)^(1/3) Omega^(-2/3) m_c / (c (m_p + m_c)^(2/3))) */
    double   e_max;               /* e ~ U(0, e_max), 0 < e_max <= 0.3 (used when elliptical)   */
    int32_t  elliptical;          /* 0: three orbital parameters (tau, Omega, alpha); 1: five (+ psi, e) */
    int32_t  pad;
} tb_bank_space;

/* rho at n given points.  lam: host double[n][5] = (tau, Omega, alpha, psi, e) per point (psi, e
 * ignored when elliptical == 0; tau >= 0, Omega > 0, 0 <= e <= 0.3); rho_out: host double[n].
 * Only t_obs_s, f_max_hz, elliptical and device of `space` are used. */
TB_API int tb_bank_density(const tb_bank_space* space, const double* lam, uint64_t n, double* rho_out);

/* Rejection placement (L263; reading G28).  uniforms: host double[n][6], every value in [0, 1); proposal i
 * is P_orb = min + u0 (max - min), tau = u1 tau_max(Omega), alpha = 2 pi u2, psi = 2 pi u3, e = u4 e_max
 * and is accepted iff u5 * rho_max < rho.  Accepted proposals are written to `out` (host, capacity
 * entries) as templates (P_orb, tau, phi0 = alpha, e, omega = psi) IN PROPOSAL ORDER.
 * rho_max must bound the density over the box for the accepted set to follow rho: a proposal with
 * rho > rho_max is accepted with probability 1 (the sampled density is clipped at rho_max) and the call
 * does not report it -- pass rho_out and check max(rho_out) <= rho_max (or draw a first batch with
 * rho_max = +huge, which accepts nothing, to learn the maximum).  volume_out does not depend on rho_max.
 *   n_accepted   receives the number accepted (also when it exceeds capacity -> TB_ERR_CAPACITY)
 *   rho_out      optional (NULL), host double[n]: the density of every proposal
 *   volume_out   optional (NULL): Monte-Carlo estimate of the proper volume V = int rho d lambda
 *                (eq 17) over the box, mean of rho / q with q the pdf of the proposal */
TB_API int tb_bank_generate(const tb_bank_space* space, const double* uniforms, uint64_t n, double rho_max,
                     tb_template* out, uint64_t capacity, uint64_t* n_accepted, double* rho_out, double* volume_out);

/* Host fp64: number of random templates for coverage eta at nominal mismatch m_star in n_dim
 * dimensions and proper volume `volume`: eq 20 (L131; exact != 0) or eq 21 (L136), C_n of eq 18 (L123). */
TB_API int tb_bank_n_templates(double eta, double m_star, uint32_t n_dim, double volume, int32_t exact, double* n_out);

/* ---- one entry point that allocates nothing ----
 * tb_series_mean_noalloc: the fp64 mean of a float32 series that is already on the GPU, i.e. the value a
 * plan uses to fill resampled samples whose source falls outside the series (reading G8; the resampling
 * step is Alg. 1).  Every other GPU entry point of this library calls cudaMalloc, directly or through a plan.
 * Some callers cannot afford that: a real-time acquisition loop, where cudaMalloc / cudaFree would take
 * the driver's lock and make the device drain while copies and searches are in flight on other streams;
 * and a process that handed the whole GPU to its own memory pool at start-up, where cudaMalloc simply
 * fails.  This call makes no cudaMalloc, no cudaFree and no allocating library call.  Its only scratch
 * memory (one partial sum per 65 536 samples and an arrival counter) is a static device array of
 * TB_NOALLOC_SCRATCH_BYTES that every GPU on which the library's kernels get loaded holds until the
 * process exits.
 *
 *   d_series     device float32[n_samples], on the device that is current on the calling thread
 *   n_samples    1 .. TB_NOALLOC_MAX_SAMPLES (2^28); need not be a power of two.  More -> TB_ERR_CAPACITY
 *                (the static array has no room for the partial sums), nothing is queued.  0 -> TB_ERR_INVALID_ARG
 *   d_mean_out   device double[1], same device; written by the kernel: read it after the stream has
 *                reached this point.  (float)*d_mean_out is the fill value a plan would derive
 *   stream       a cudaStream_t of that device (NULL = the default stream).  The call only queues a
 *                256-byte clear and one kernel on it and returns; it never synchronises
 *   errbuf       optional (NULL): receives a one-line description when the call fails; errbuf_len bytes
 *
 * First call on each device: it also looks up the device address of the static array (cudaGetSymbolAddress,
 * which makes the runtime load this library's kernels on that device if nothing did yet).  Make that
 * first call during start-up, before any stream capture.  Later calls only queue work.
 * Shared state: all calls in the process, from any thread, on any stream, use the same array on a given
 * device, and it keeps what the last call left (the counter is cleared at the start of every call).  Two
 * calls whose kernels may overlap on the GPU (different streams without an event between them) race on it
 * and both results are garbage: order them, e.g. by using one stream.  Calls on different devices are
 * independent.  The result is deterministic (fixed summation order, independent of the SM count) and
 * agrees with the plan's fill value to fp64 rounding (a few 1e-16 relative). */
#define TB_NOALLOC_MAX_SAMPLES   (1ull << 28)
#define TB_NOALLOC_SCRATCH_BYTES 33024   /* (32 + 4096) doubles */
TB_API int tb_series_mean_noalloc(const float* d_series, uint64_t n_samples, double* d_mean_out, void* stream,
                           char* errbuf, uint64_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* TB_H_ */
