/*
 * cbmf.h -- C ABI of the B200-native coalescing-binary matched filter
 *           (hot path of "cuInspiral", arXiv 1006.4644).
 *
 * The library matched-filters ONE detector data segment against a bank of 2PN
 * stationary-phase chirp templates (eq. 2.1; the per-chunk loop of
 * PAPER.md:96-103).  For every template it generates h~(f) on the fly, forms
 * d~ h~* / S_n, runs an N-point inverse FFT to the two-quadrature output z(t),
 * normalises by sigma and reduces |z| to the peak SNR, its sample index, the
 * coalescence phase and the list of samples above threshold.  Every step runs in
 * hand-written sm_100a kernels; the host code below this ABI only validates
 * arguments, allocates device memory and launches.  There is no CPU fallback.
 *
 * Conventions (readings A1-A21):
 *   N samples, fs, dt = 1/fs, df = fs/N, f_k = k df.
 *   forward transform  d~[k] = dt sum_j d[j] e^{-2 pi i jk/N}
 *   template           h~[k] = f_k^{-7/6} e^{-i Psi_T(f_k)},  k_lo <= k <= k_hi, else 0
 *                      k_lo = ceil(f_low/df), k_hi = min(floor(f_ISCO/df), N/2-1)
 *   Psi_T              2PN SPA phase of BASELINE.json configs[0] with t_c = phi_c = 0
 *   sigma^2            4 df sum_k |h~[k]|^2 / S_n[k]            (one-sided S_n)
 *   z[j]               4 df sum_k d~[k] h~*[k] / S_n[k] e^{+2 pi i jk/N}, j = 0..N-1, circular
 *   rho[j]             |z[j]| / sigma     (= sqrt(c_+^2 + c_x^2))
 *   peak               smallest j attaining max rho; phase = atan2(Im z, Re z) in (-pi, pi]
 *   trigger            every j with rho[j] > threshold (strict)
 *
 * Return codes: 0 success, < 0 error, > 0 warning.  All pointers are HOST pointers
 * unless the function name ends in _dev, in which case every array pointer is a
 * DEVICE pointer on the context's device (scalars stay host values).  The caller
 * owns every array; the context owns all of its device memory.  Every call that
 * returns results is synchronous with respect to the context's stream: they are
 * complete on return.  cbmf_set_psd_dev and cbmf_load_segment_dev, which return no
 * results, are STREAM-ORDERED: they enqueue their work on the context's stream and
 * return without waiting; the check of their input (a PSD entry <= 0 or NaN, a NaN /
 * Inf sample) comes back with the next call that waits (any cbmf_filter_* / chisq /
 * debug call, or a host-pointer set / load), which then returns CBMF_EINVAL and leaves the
 * context without that PSD or segment (ESTATE afterwards).  The input arrays of a _dev call
 * must stay valid until such a call has returned.  A context is not thread-safe; contexts
 * are independent.
 */
#ifndef CBMF_H
#define CBMF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CBMF_OK        0
#define CBMF_EINVAL   -1   /* bad argument (see each call) */
#define CBMF_ESTATE   -2   /* call order: PSD, then segment, then filter */
#define CBMF_ECUDA    -3   /* a CUDA runtime call failed; cbmf_last_cuda_error() names it */
#define CBMF_ENOMEM   -4   /* host or device allocation failed */
#define CBMF_ELIMIT   -5   /* size beyond the fixed limit of a no-allocation entry point (cbmf_ifft_noalloc_dev) */
#define CBMF_WTRUNC    1   /* more triggers found than trig_capacity: list truncated */

typedef struct cbmf_ctx cbmf_ctx;                 /* opaque */

/* One template = one point (m1, m2) of the bank, solar masses, both > 0 and finite
 * ("(m1,m2)_i").  Layout: two consecutive doubles. */
typedef struct { double m1, m2; } cbmf_template;

/* Per-template result (candidate time and c(t_0) = SNR).
 * idx_peak counts samples from segment start (t_peak = idx_peak / fs).  A template whose
 * band is empty (f_ISCO < f_low) returns {0, -1, 0, 0}. */
typedef struct { float snr_max; int32_t idx_peak; float phase; float sigma; } cbmf_peak;

/* One above-threshold sample (PAPER.md:102, :131 device_maxfind). */
typedef struct { int32_t template_idx; int32_t sample_idx; float snr; float phase; } cbmf_trigger;

/* Create a context for segments of n samples (n a power of two, 2^12 <= n <= 2^24) at
 * sample rate fs_hz, with lower cutoff f_low_hz (0 < f_low < fs/2), on CUDA device
 * `device`.  cuda_stream is a cudaStream_t (e.g. torch's current stream) or NULL for the
 * default stream.  Contexts are independent, also across devices of one process: all
 * per-device state (kernel attributes, SM count) lives in the context, and the library
 * reads no environment variable.  The floor 2^12 (SURVEY.md §8(b) proposes 2^10) is that of
 * the two-pass FFT split, N1, N2 >= 64; the paper's segments are 2^18..2^21
 * (PAPER.md:249-254).  Errors: EINVAL, ECUDA, ENOMEM. */
int cbmf_create(cbmf_ctx **out, int device, int64_t n, double fs_hz, double f_low_hz,
                void *cuda_stream);
int cbmf_destroy(cbmf_ctx *ctx);

/* S0: one-sided noise PSD S_n[k], k = 0..n/2 (n_bins == n/2+1).
 * Builds, on the device in fp64, the weights 4 df dt f_k^{-7/6}/S_n[k] and the prefix table
 * P[k] = 4 df sum_{k'=k_lo..k} f_k'^{-7/3}/S_n[k'] (sigma^2 of a template is P[k_hi]).
 * +inf is legal (weight 0).  EINVAL if n_bins is wrong or an entry inside [k_lo, n/2) is
 * <= 0 or NaN.  Invalidates the loaded segment. */
int cbmf_set_psd(cbmf_ctx *ctx, const double *psd_onesided, int64_t n_bins);
int cbmf_set_psd_dev(cbmf_ctx *ctx, const double *psd_onesided_dev, int64_t n_bins);

/* S1: one data segment d[j], j = 0..n-1, float32 ("input data chunk").
 * Computes w[k] = 4 df d~[k] f_k^{-7/6}/S_n[k] (k_lo <= k < n/2, else 0) with the
 * library's own FFT and keeps it resident on the device for all following filter calls
 * (PAPER.md:107, :157).  ESTATE if no PSD is set; EINVAL if n_samples != n or a sample
 * is NaN/Inf. */
int cbmf_load_segment(cbmf_ctx *ctx, const float *samples, int64_t n_samples);
int cbmf_load_segment_dev(cbmf_ctx *ctx, const float *samples_dev, int64_t n_samples);

/* S2-S8: the bank loop of PAPER.md:98-102.  For each template: SPA generation, correlate,
 * inverse FFT, |z|/sigma, peak and triggers.
 *   peaks_out[n_templates]   one cbmf_peak per template, bank order.
 *   trig_out[trig_capacity]  triggers sorted by (template_idx, sample_idx); may be NULL
 *                            with capacity 0 (triggers are still counted).
 *   n_trig_found             total number of samples above threshold over the whole bank;
 *                            if it exceeds trig_capacity the list is TRUNCATED: trig_out holds
 *                            the first trig_capacity triggers in (template_idx, sample_idx)
 *                            order (what the full sorted list would start with) and the call
 *                            returns CBMF_WTRUNC.  A truncated call may filter the leading part
 *                            of the bank a second time to collect them.
 * The trigger test is |z[j]|^2 > (snr_threshold * sigma)^2 evaluated in fp32 (monotone in rho,
 * SURVEY.md reading A13); it is authoritative: the reported snr = sqrt(|z|^2) / sigma is rounded
 * separately and may differ from the threshold by one unit in the last place either way.
 * snr_threshold >= 0.  n_templates may be 0.  ESTATE before PSD and segment are set;
 * EINVAL on a non-positive or non-finite mass, on a template whose phase exceeds 2^19 cycles
 * inside the band (total mass far below 0.3 Msun at f_low = 10 Hz), or a negative / NaN threshold.
 * The masses are checked on the device BEFORE any filtering: a bank with an invalid template
 * fails at once, nothing is written, and cbmf_last_bad_template() names the first offender. */
int cbmf_filter_bank(cbmf_ctx *ctx, const cbmf_template *bank, int64_t n_templates,
                     float snr_threshold, cbmf_peak *peaks_out,
                     cbmf_trigger *trig_out, int64_t trig_capacity, int64_t *n_trig_found);
/* Device-pointer variant: bank_dev, peaks_out_dev, trig_out_dev are device arrays;
 * n_trig_found stays a HOST pointer. */
int cbmf_filter_bank_dev(cbmf_ctx *ctx, const cbmf_template *bank_dev, int64_t n_templates,
                         float snr_threshold, cbmf_peak *peaks_out_dev,
                         cbmf_trigger *trig_out_dev, int64_t trig_capacity,
                         int64_t *n_trig_found);
/* Bank index of the first invalid template of the last cbmf_filter_bank* call that returned
 * EINVAL for that reason, else -1. */
int64_t cbmf_last_bad_template(const cbmf_ctx *ctx);

/* ---- trigger clustering ----
 * "Reduce the [c(t_0)] set, in order to detect local maximum"; "The clusterization phase is made
 * only by CPU.  This chose permits us to hide this computing part behind the next iteration".
 * The paper states no rule; reading A24: above-threshold samples of ONE template form an event
 * while consecutive ones are at most window_samples apart, the segment taken as a circle (the filter output is
 * circular); an event is reported as its sample of largest snr (the whole trigger record), the smallest
 * sample_idx among equal maxima; events are ordered by (template_idx, sample_idx). */

/* Host function, no device work: trig[n_trig] must be sorted strictly by (template_idx, sample_idx) with
 * 0 <= sample_idx < n_samples, as cbmf_filter_bank returns it.  Writes at most event_capacity events (the first ones
 * in order; rc = CBMF_WTRUNC if there are more), *n_events = the full count.  EINVAL on an unsorted list, an index
 * out of range, window_samples < 0 or a NULL n_events. */
int cbmf_cluster_triggers(const cbmf_trigger *trig, int64_t n_trig, int64_t n_samples, int64_t window_samples,
                          cbmf_trigger *events_out, int64_t event_capacity, int64_t *n_events);

/* cbmf_filter_bank with the reduction behind it, overlapped as PAPER.md:131 describes: the bank runs as a stream of
 * launch pairs (sub-batches); each pair's raw triggers are copied to pinned host memory right behind it and the
 * host sorts and clusters them while the GPU filters the following pairs.  All pointers are HOST pointers.
 * peaks_out[n_templates] as in cbmf_filter_bank; events_out[event_capacity] the events of the whole bank in
 * (template_idx, sample_idx) order, truncated like the trigger list (CBMF_WTRUNC); *n_events the full event count;
 * *n_trig_found (may be NULL) the number of raw above-threshold samples.  Same errors as cbmf_filter_bank.
 * The call is not profiled: cbmf_last_pass_time and cbmf_debug_timeline read empty after it. */
int cbmf_filter_bank_clustered(cbmf_ctx *ctx, const cbmf_template *bank, int64_t n_templates, float snr_threshold,
                               int64_t window_samples, cbmf_peak *peaks_out, cbmf_trigger *events_out,
                               int64_t event_capacity, int64_t *n_events, int64_t *n_trig_found);

/* ---- segment streaming ----
 * The online use of PAPER.md:247-255 (table 4.1: templates processed in real time) with the data kept on the device
 * (PAPER.md:157-165).  A continuous stream samples[n_total] (HOST pointer, float32; pinned memory lets the copies
 * overlap) is cut into segments of n samples (the context's n) that overlap by `discard` samples: segment s starts
 * at s * (n - discard), and as many whole segments as fit are processed (*n_segments).  Every segment is filtered
 * on its own, circularly, exactly as cbmf_load_segment + cbmf_filter_bank do; the first `discard` output samples of a
 * segment, which the wrap-around of templates up to that length corrupts, take no part in its peaks or triggers
 * (overlap-save; reading A25: the paper's table implies discard = n/2).  The template constants are
 * set up once; while the bank runs on segment s, segment s + 1 is copied to the device and transformed on a second
 * stream into a second weight buffer.
 *   peaks_out[n_segments * n_templates]  segment-major; idx_peak counts from the start of ITS segment (>= discard)
 *   trig_out[trig_capacity]              the triggers of segment 0, then 1, ...; inside a segment sorted by
 *                                        (template_idx, sample_idx), sample_idx counted from the segment start
 *   seg_offsets_out[n_segments + 1]      (may be NULL) segment s owns trig_out[seg_offsets_out[s] .. [s + 1])
 *   n_trig_found                         (may be NULL) all above-threshold samples of all segments; when that exceeds
 *                                        trig_capacity the list stops at the capacity (whole leading triggers of the
 *                                        segment that crosses it, later segments empty) and rc = CBMF_WTRUNC
 * Global sample index of a peak or trigger = s * (n - discard) + its index.  The call leaves no loaded segment in
 * the context (ESTATE for cbmf_filter_bank until the next cbmf_load_segment).  ESTATE without a PSD; EINVAL for
 * discard outside [0, n), n_total < n, a NaN / Inf sample, an invalid template (cbmf_last_bad_template). */
int cbmf_filter_stream(cbmf_ctx *ctx, const float *samples, int64_t n_total, const cbmf_template *bank,
                       int64_t n_templates, float snr_threshold, int64_t discard, cbmf_peak *peaks_out,
                       cbmf_trigger *trig_out, int64_t trig_capacity, int64_t *seg_offsets_out,
                       int64_t *n_trig_found, int64_t *n_segments);

/* ---- chi-squared veto ----
 * Allen's chi-squared time-frequency discriminator ("a optimized chi-squared [24] test routine";
 * ref. [24] at PAPER.md:321: Phys. Rev. D 71, 062001), for every template of `bank` at ONE output sample of the
 * loaded segment, sample_idx[t] (e.g. idx_peak of cbmf_filter_bank; a negative index gives chi^2 = 0, as does an
 * empty band).  Reading A26: the band [k_lo, k_hi] of a template is cut into p_bands contiguous
 * sub-bands of equal expected SNR^2 on the grid (bin k belongs to band floor(p P[k-1] / sigma^2), P the S0 prefix
 * table); z_l = the filter output restricted to band l (sum_l z_l = z[sample]), p_l = sigma_l^2 / sigma^2,
 *     chi^2 = sum_l |z_l - p_l z|^2 / (p_l sigma^2),
 * which has 2 p_bands - 2 degrees of freedom in Gaussian noise (quadratures of unit variance) and vanishes for data
 * proportional to the template.  One sample needs no FFT: the band sums are taken directly on the device in fp64
 * from the same w[k] and SPA phase the filter uses.  All pointers are HOST pointers; chisq_out[n_templates];
 * zl_out (may be NULL): n_templates * p_bands complex doubles (re, im), the z_l.  1 <= p_bands <= 256,
 * n_templates <= 65535.  ESTATE before PSD and segment; EINVAL for an index >= n or an invalid template. */
int cbmf_chisq(cbmf_ctx *ctx, const cbmf_template *bank, int64_t n_templates, const int32_t *sample_idx,
               int p_bands, float *chisq_out, double *zl_out);

/* ---- diagnostics: used by the parity tests and the kernel sweep, never by filter_bank ---- */

/* rho[j] (n floats) and optionally z[j] (2n floats, interleaved re,im) for one template,
 * through the same generator / FFT kernels with a storing epilogue. */
int cbmf_debug_snr_series(cbmf_ctx *ctx, cbmf_template t, float *snr_out, float *z_out_or_null);
/* Unit-amplitude template h~[k] = f_k^{-7/6} e^{-i Psi_T}, k = 0..n/2 (2*(n/2+1) floats). */
int cbmf_debug_template(cbmf_ctx *ctx, cbmf_template t, float *h_out);
/* out[b][j] = sum_k in[b][k] e^{+2 pi i jk/n} (unnormalised inverse DFT), `batch` vectors of
 * n complex floats (interleaved), n must equal the context's n. */
int cbmf_debug_ifft(cbmf_ctx *ctx, const float *in, float *out, int64_t n, int64_t batch);
int cbmf_debug_ifft_dev(cbmf_ctx *ctx, const float *in_dev, float *out_dev, int64_t n, int64_t batch);
/* The generator alone: writes q~[b][k] = w[k] e^{+i Psi_b(f_k)} (n/2 complex floats per
 * template, device array) -- SURVEY.md config 4 "template-generator-only throughput". */
int cbmf_debug_generate_dev(cbmf_ctx *ctx, const cbmf_template *bank_dev, int64_t n_templates,
                            float *q_out_dev);
/* The FP32 throughput this GPU reaches on dependent FMA chains (one 1024-thread block per SM, eight chains per
 * thread), in TFLOP/s: scalar FFMA and packed FFMA2 (fma.rn.f32x2).  bench.py reports it beside the unit-count peak
 * that is the roofline denominator.  Allocates a small buffer, runs on the legacy default stream of
 * `device` and waits.  EINVAL for a NULL pointer or a device that does not exist; ECUDA. */
int cbmf_debug_fp32_peak(int device, double *tflops_ffma, double *tflops_ffma2);
/* Copies of device state for tests: sigma^2 prefix table P[k] (n/2 doubles) and w[k]
 * (n/2 complex floats, interleaved). */
int cbmf_debug_get_prefix(cbmf_ctx *ctx, double *p_out);
int cbmf_debug_get_weights(cbmf_ctx *ctx, float *w_out);

/* ---- inverse FFT for callers that must not allocate device memory ----
 * Who this is for.  Every other device-side call of this library goes through a cbmf_ctx, and creating or growing
 * a context calls cudaMalloc (the inter-pass buffer Y of the two-pass FFT alone is 8 n bytes per transform).  Some
 * users of the transform cannot do that at the point where they need it:
 *   - code that runs inside someone else's memory budget -- a plug-in of a framework whose caching allocator has
 *     already taken (nearly) all of the GPU, so that a raw cudaMalloc fails or fragments the pool;
 *   - a real-time analysis loop (the online search of PAPER.md:247-255) that may not stall: cudaMalloc / cudaFree
 *     synchronise the whole device and take an unbounded time;
 *   - code that is between cudaStreamBeginCapture and cudaStreamEndCapture on some stream of the process, where an
 *     allocation is an error.
 * cbmf_ifft_noalloc_dev is the stand-alone transform of cbmf_debug_ifft_dev (same kernels, same split of n, same
 * results: S5 of SURVEY.md §8(a), "inverse FFT") WITHOUT a context and without any allocation: its
 * inter-pass buffer is a fixed array of CBMF_NOALLOC_MAX_N complex floats (8 MiB) that is part of the library image.
 * Every GPU that loads this library's device code holds that array from then until the process exits, whether or
 * not this function is ever called there: that is the price, and the reason for the modest limit.
 *   out_dev[b][j] = sum_k in_dev[b][k] e^{+2 pi i jk/n}     (unnormalised, b < batch, interleaved re,im float32)
 *   in_dev, out_dev  DEVICE pointers on `device`, batch * n complex floats each, 16-byte aligned, caller-owned,
 *                    not overlapping; in_dev is only read.
 *   n                a power of two, 2^12 <= n <= CBMF_NOALLOC_MAX_N.  batch >= 0: the transforms run
 *                    CBMF_NOALLOC_MAX_N / n at a time, one launch pair after the other.
 *   cuda_stream      a cudaStream_t of `device`, or NULL for the default stream.
 * STREAM-ORDERED: the launches are enqueued on cuda_stream and the call returns without waiting; out_dev is
 * complete once the stream has reached that point.  in_dev must stay valid until then.
 * First call on a device: with that device current it looks the array's device address up (cudaGetSymbolAddress)
 * and reads the SM count; the first call for each n on a device also opts that size's two kernels in to their
 * shared-memory size (cudaFuncSetAttribute).  That is a one-off set-up of a few runtime calls: make a first call
 * for every (device, n) you will use at start-up, before any stream capture begins and outside the part of the
 * program that must not stall.  Later calls only launch kernels.  No call, first or later, uses cudaMalloc, cudaFree, or a library routine that
 * allocates device memory.
 * ONE array per GPU serves every call of the process.  Calls on the same stream follow each other and are safe.
 * Calls whose kernels may run at the same time on one GPU (different streams, different threads) would write the
 * same buffer: the results of both are then undefined -- order them yourself (one stream, or events).  The array
 * keeps what the last call left in it; nothing in it has to start at zero, because pass 1 writes every element that
 * pass 2 reads before pass 2 starts, so no clearing is done or needed.
 * Errors: CBMF_ELIMIT if n > CBMF_NOALLOC_MAX_N (nothing is enqueued; use a context and cbmf_debug_ifft_dev);
 * CBMF_EINVAL for a NULL pointer with batch > 0, a misaligned pointer, n not a power of two or below 2^12,
 * batch < 0, a device index that does not exist or is >= 64; CBMF_ECUDA if a runtime call fails. */
#define CBMF_NOALLOC_MAX_N (1 << 20)
int cbmf_ifft_noalloc_dev(int device, void *cuda_stream, const float *in_dev, float *out_dev,
                          int64_t n, int64_t batch);

/* ---- waveform order ----
 * Phase order of the SPA templates, in half post-Newtonian orders: 4 = 2PN (default: BASELINE.json configs[0], the
 * Psi_T of the header comment), 5 = 2.5PN, the order the paper states ("Post Newtonian approximation of order 2.5 in
 * phase and 0 in amplitude"; its Fig. 4 title says "PN2").  The paper prints no formula; the 2.5PN term
 * is the published one (Arun, Iyer, Sathyaprakash & Sundararajan, Phys. Rev. D 71, 084008 (2005), eq. 3.4 =
 * Buonanno et al., Phys. Rev. D 80, 084043 (2009), eq. 3.18):
 *     Psi += 3/(128 eta v^5) * pi (38645/756 - 65 eta/9) (1 + 3 ln(v / v_lso)) v^5,   v_lso = 6^{-1/2}.
 * Applies to every later call (filter, stream, chisq, debug); amplitude, band and sigma do not change, so PSD and
 * segment stay loaded.  EINVAL for any other value. */
int cbmf_set_pn_order(cbmf_ctx *ctx, int half_order);
int cbmf_get_pn_order(const cbmf_ctx *ctx);

/* ---- the paper's own template path (second part) ----
 * "the two polarization of the template signal are generated, FFT transformed and normalized ... with a complex
 * product and reduction algorithms", then the two correlators and the quadrature sum
 * (PAPER.md:99-101, :127-131).  The paper prints no waveform; reading A28: the time-domain chirp with
 * an explicit phase, every sample an independent evaluation ("TaylorT3": Blanchet, Living Rev. Relativity 9, 4 (2006),
 * eq. (234)), phase order as cbmf_set_pn_order says, amplitude at Newtonian order:  with tau = t_c - t,
 * Theta = eta tau / (5 M), x = Theta^{1/8},
 *     phi_gw = -(2/eta) [x^5 + a2 x^3 - (3 pi/4) x^2 + a4 x + a5 ln Theta],   F = (1/2 pi) d phi_gw / dt,
 *     a2 = 3715/8064 + 55 eta/96,  a4 = 9275495/14450688 + 284875 eta/258048 + 1855 eta^2/2048,
 *     a5 = (-38645/172032 + 65 eta/2048) pi  (2.5PN only),
 *     h_+ = (F/f_low)^{2/3} cos phi_gw,  h_x = (F/f_low)^{2/3} sin phi_gw,
 * from F = f_low up to F = f_ISCO, or to the maximum of F where the series stops sweeping upward first; the
 * coalescence sits at sample 0 (= n: the segment is a circle).  Per polarisation p: H_p = forward transform,
 * sigma_p^2 = 4 df sum_k |H_p[k]|^2 / S_n[k], c_p[j] = 4 df Re sum_k d~[k] H_p*[k] / S_n[k] e^{+2 pi i jk/n}, both over
 * k_lo <= k < n/2, and rho[j] = sqrt((c_+/sigma_+)^2 + (c_x/sigma_x)^2).
 * Arguments, results, truncation and errors as cbmf_filter_bank (host pointers); phase = atan2(c_x/sigma_x,
 * c_+/sigma_+) at the peak, sigma = sigma_+.  Additional EINVAL: a template longer than the segment
 * (cbmf_last_bad_template names it).  A template whose f_ISCO lies below f_low is empty: {0, -1, 0, 0}.
 * This is the comparison path (generation + two transforms + a reduction per template, every intermediate in device
 * memory, as in the paper); the tuned path is cbmf_filter_bank. */
int cbmf_filter_bank_td(cbmf_ctx *ctx, const cbmf_template *bank, int64_t n_templates,
                        float snr_threshold, cbmf_peak *peaks_out,
                        cbmf_trigger *trig_out, int64_t trig_capacity, int64_t *n_trig_found);
/* Diagnostic: the two polarisations of one template on the sample grid, (h_+[j], h_x[j]) interleaved, 2n floats. */
int cbmf_debug_td_template(cbmf_ctx *ctx, cbmf_template t, float *h_out);

/* ---- tuning ---- */
/* Templates per launch pair (pass 1 + pass 2), an upper limit: a call over a small bank uses fewer, so that every
 * launch pair in flight has work.  Default: 2 GiB of inter-pass buffer (8 n bytes per template) per pair, at most
 * 256 templates (256 at n <= 2^20, 64 at 2^22, 16 at 2^24); results do not depend on it.
 * 1 <= templates_per_launch <= 4096; ENOMEM if the larger buffer cannot be allocated. */
int cbmf_set_sub_batch(cbmf_ctx *ctx, int templates_per_launch);
int cbmf_get_sub_batch(const cbmf_ctx *ctx);
/* Launch pairs in flight: sub-batches are issued round-robin on this many internal streams
 * (forked from and joined to the context's stream inside every filter call), so that pass-1 blocks
 * of one pair share the SMs with pass-2 blocks of the others.  Default 4.  The inter-pass buffer
 * grows to launch_pairs_in_flight * templates_per_launch * 8 n bytes; results do not depend on it.
 * 1 <= launch_pairs_in_flight <= 8. */
int cbmf_set_streams(cbmf_ctx *ctx, int launch_pairs_in_flight);
int cbmf_get_streams(const cbmf_ctx *ctx);
/* ---- introspection ---- */
/* The FFT split chosen at create: n = 2^log2_n1 * 2^log2_n2, pass 1 = column FFTs of 2^log2_n1
 * points, pass 2 = row FFTs of 2^log2_n2 points (bench.py's per-pass flop counts). */
int cbmf_get_split(const cbmf_ctx *ctx, int *log2_n1, int *log2_n2);
/* Kernels launched by this context since creation (bench.py's gpu_launches). */
int64_t cbmf_launch_count(const cbmf_ctx *ctx);
/* Device time (ms, CUDA events on the context's stream) and launch count of the two FFT-pass
 * kernels inside the last cbmf_filter_bank* call; used for the roofline line of bench.py.
 * which = 0: pass 1 (generate + column FFT), 1: pass 2 (row FFT + epilogue). */
int cbmf_last_pass_time(const cbmf_ctx *ctx, int which, double *ms_out, int64_t *launches_out);
/* Per-pass event timing above: 0 off (default, no events recorded); 1 every pass launch ALONE, all
 * on the context's stream; 2 the real schedule (launch pairs on the internal streams), every launch
 * bracketed by events on its own stream, so a duration includes the time the kernel shares its SMs
 * with the launches of the other pairs.  EINVAL for any other value. */
int cbmf_set_profiling(cbmf_ctx *ctx, int mode);
/* Launch timeline of the last profiled cbmf_filter_bank* call: for pass `which`, start and end of every launch in ms
 * since the first pass-1 launch (start_end_ms[2 i], [2 i + 1]; at most max_launches pairs; *n_launches = all). */
int cbmf_debug_timeline(const cbmf_ctx *ctx, int which, float *start_end_ms, int64_t max_launches, int64_t *n_launches);
const char *cbmf_strerror(int rc);
const char *cbmf_last_cuda_error(const cbmf_ctx *ctx);
const char *cbmf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CBMF_H */
