/* sft.h - C ABI of libsft_b200.so: the SFT inner product of arXiv:2502.11823 on one B200.
 *
 * Citations "P:NNN" are line numbers of the paper text; "DESIGN" is DESIGN.md in
 * this repository (readings of the paper where it is silent or garbled).
 *
 * What the library computes (Eq.(20)-(35); discretised Eq.(1)):
 *
 *   ([x,h]) = 4 df Re sum_{c,a,k in B_a} conj(x~_{c,a,k}) h~_{c,a,k} / S_{c,a}(f_k)
 *   ([h,h]) = 4 df    sum_{c,a,k in B_a} |h~_{c,a,k}|^2            / S_{c,a}(f_k)
 *   h~_{c,a,k} = 1/2 T A_a R_{c,a} e^{i phi_a} F((f_a - f_k) T, fdot_a T^2)
 *   F(a,b)     = int_0^1 exp(i pi (2 a s + b s^2)) ds          (Eq.(28), dimensionless)
 *
 * c = channel, a = SFT index (start t_a = t0 + a T), k = frequency bin (f_k = k/T,
 * P:191), B_a = {k_c-K .. k_c+K} the truncated band around the signal, {A, phi, f,
 * fdot}_a the four numbers per SFT of P:164 from a restricted TaylorT3 inspiral (0PN or
 * 0PN+1PN; DESIGN W1), R_{c,a} the per-SFT complex detector response with
 * Lambda z = Re[R z] (Eq.(5)-(6) P:80-85), S_{c,a}(f_k) = s_{c,a} S_c(f_k) the per-SFT noise
 * PSD, gaps = missing SFTs.  Every step runs in CUDA kernels on the plan's
 * device; there is no CPU fallback.
 *
 * Conventions: all functions return an sft_status and never throw, abort or touch errno.
 * On error the outputs are untouched and sft_last_error(plan) describes the failure.
 * The caller owns every pointer it passes; the plan copies what it keeps.  A plan is not
 * thread-safe; distinct plans are independent.  Work is ordered on the plan's stream; calls
 * with host pointers return after the results are on the host, calls with device pointers
 * return after enqueueing (call sft_plan_sync or synchronise the stream yourself).
 */
#ifndef SFT_B200_H
#define SFT_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SFT_MAX_CHANNELS 4
#define SFT_NPARAM 8   /* doubles per template row, see sft_inner_products */
#define SFT_MAX_K 128  /* largest accepted half-width of the band */

typedef struct sft_plan sft_plan; /* opaque; owns all its device memory */

typedef enum {
  SFT_OK = 0,
  SFT_EINVAL = 1,       /* NULL pointer or out-of-range argument            */
  SFT_ESHAPE = 2,       /* inconsistent sizes (t_sft*fs not an integer, ..) */
  SFT_ENODATA = 3,      /* a channel has not been loaded yet                */
  SFT_EUNSUPPORTED = 4, /* valid request this build does not implement      */
  SFT_ECUDA = 5,        /* CUDA runtime error (message in sft_last_error)   */
  SFT_ENOMEM = 6        /* host or device allocation failed                 */
} sft_status;

enum { SFT_KERNEL_DIRICHLET = 0, /* F(a,0) = e^{i pi a} sinc(a), Eq.(B2)          */
       SFT_KERNEL_FRESNEL = 1 }; /* F(a,b), Eq.(28)-(32) P:215-236                      */
enum { SFT_WF_PN0 = 0,           /* Newtonian restricted TaylorT3 inspiral              */
       SFT_WF_PN1 = 1,           /* + 1PN phase and frequency terms                     */
       SFT_WF_PN15 = 2 };        /* + 1.5PN (tail) terms: phase -(3 pi/4) Theta^(1/4), frequency -(3 pi/10) Theta^(-3/4)  */
enum { SFT_PHASE_FP64 = 0,       /* phase/frequency track evaluated in fp64             */
       SFT_PHASE_SPLIT32 = 1 };  /* track evaluated in double-float (2 x fp32) arithmetic: same bins,
                                    phases to ~1e-7 rad; slower on B200       */
enum { SFT_RESP_NONE = 0,        /* R = 1                                               */
       SFT_RESP_TABLE = 1,       /* R_{c,a} from sft_load_data's `response`             */
       SFT_RESP_ANNUAL = 2 };    /* R_{c,a} = [1 + depth cos(2 pi t_a/period + psi_c + lambda)]
                                    e^{i (chi_c + beta)}, (lambda, beta) per template    */
enum { SFT_EVAL_AUTO = 0,        /* moment tables when they fit in device memory, else direct     */
       SFT_EVAL_DIRECT = 1,      /* evaluate the 2K+1 kernel coefficients per (template, SFT)      */
       SFT_EVAL_TABLE = 2 };     /* insist on the moment tables (SFT_ENOMEM if they do not fit)    */
enum { SFT_MEM_HOST = 0, SFT_MEM_DEVICE = 1 };

/* Analysis set-up.  Zero-initialise, then fill. */
typedef struct {
  int32_t n_channels;  /* 1..SFT_MAX_CHANNELS                                            */
  int64_t n_sft;       /* SFT slots per channel, gaps included                   */
  double t_sft;        /* T_SFT [s]; t_sft*fs must be an integer n (samples per SFT)     */
  double fs;           /* sampling rate [Hz]; bins k<1 and k>=n/2 never contribute (DESIGN A6) */
  double t0;           /* start time of SFT 0 [s]                                        */
  int32_t k_lo, k_hi;  /* stored band: bins k_lo <= k < k_hi                             */
  int32_t K;           /* band half-width, 2K+1 bins per SFT; 0..SFT_MAX_K       */
  int32_t kernel;      /* SFT_KERNEL_*                                                   */
  int32_t waveform;    /* SFT_WF_*                                                       */
  int32_t phase_path;  /* SFT_PHASE_*                                                    */
  int32_t response;    /* SFT_RESP_*                                                     */
  double f_lo, f_hi;   /* pair active iff f_lo <= f_a, f_a + fdot_a T <= f_hi, t_a + T < t_c (DESIGN A12) */
  double f_ref;        /* amplitude reference: A_a = amp (f_a/f_ref)^(2/3)       */
  double resp_period;  /* SFT_RESP_ANNUAL: modulation period [s]                          */
  double resp_depth;   /* SFT_RESP_ANNUAL: modulation depth                               */
  double resp_psi[SFT_MAX_CHANNELS]; /* SFT_RESP_ANNUAL: amplitude-modulation phase per channel */
  double resp_chi[SFT_MAX_CHANNELS]; /* SFT_RESP_ANNUAL: response phase per channel             */
  int32_t evaluator;   /* SFT_EVAL_*: how sum_k conj(x~) F / S and sum_k |F|^2 / S are evaluated for
                          |fdot| T^2 <= 1; results agree to ~1e-6 */
  int32_t include_dc;  /* 0: bins k < 1 never contribute (DESIGN A6: int_0^inf of Eq.(1), PSDs diverging at f = 0);
                          1: the bin k = 0 counts at full weight, as in the paper's sums ("d~[k] = 0 for k < 0") -
                          needed by signals below the first bin (edge effects, section IV.D)    */
  int32_t device;      /* CUDA device ordinal                                             */
  void *stream;        /* cudaStream_t to order work on, or NULL for the legacy default stream */
} sft_plan_desc;

/* Creates a plan: validates `desc`, selects the device, allocates the (empty) data-SFT store
 * [n_channels][n_sft][k_hi-k_lo] complex64 + weight tables in device memory (SFTs are
 * "computed once ... reused") and, unless SFT_EVAL_DIRECT, the moment tables of the
 * table evaluator (128 bytes per SFT, window position k_c and quarter bin).
 * *out is set only on SFT_OK. */
sft_status sft_plan_create(const sft_plan_desc *desc, sft_plan **out);

/* Frees the plan and all device memory it owns.  NULL is accepted. */
sft_status sft_plan_destroy(sft_plan *plan);

/* Loads one channel of data SFTs (Eq.(26)) and its noise description, and whitens it
 * on the device (Eq.(15) P:153 moves 1/S onto the data):
 *   sft_bins   complex64 interleaved (re,im), [n_sft][k_hi-k_lo], bin fastest, units strain*s
 *   psd_scale  [n_sft] s_{c,a} of S_{c,a}(f_k) = s_{c,a} S_c(f_k); <= 0 or non-finite => gap
 *   psd_shape  [k_hi-k_lo] S_c(f_k) > 0 (one-sided PSD); NULL => 1
 *   response   complex64 interleaved [n_sft] R_{c,a}; required iff plan response == SFT_RESP_TABLE, else ignored/NULL
 *   mem        SFT_MEM_HOST or SFT_MEM_DEVICE: where ALL the non-NULL pointers of this call live
 * Also (re)builds the channel's moment tables.  May be called again for the same channel to replace
 * its data. */
sft_status sft_load_data(sft_plan *plan, int32_t channel, const float *sft_bins,
                         const double *psd_scale, const double *psd_shape,
                         const float *response, int32_t mem);

/* Streaming ("SFTs ... can be computed online and in parallel as data arrives", section V.A): replaces the SFT slots
 * first_sft <= a < first_sft + n_new of a channel that sft_load_data has loaded before (typically with the slots still to come
 * marked as gaps), in place: the rows of the whitened store and of the moment tables of these slots only.  The channel keeps the
 * PSD shape S_c(f_k) of its sft_load_data call.
 *   sft_bins   complex64 [n_new][k_hi-k_lo], psd_scale [n_new] (<= 0 or non-finite => gap), response complex64 [n_new] (iff
 *   SFT_RESP_TABLE); `mem` as in sft_load_data.  SFT_ESHAPE if the slots do not fit the plan, SFT_ENODATA before sft_load_data. */
sft_status sft_append_sfts(sft_plan *plan, int32_t channel, int64_t first_sft, int64_t n_new,
                           const float *sft_bins, const double *psd_scale, const float *response, int32_t mem);

/* Data SFTs from a time series (Eq.(26), section V.A): for each of n_sft disjoint segments of n
 * samples (a trailing partial segment is ignored, DESIGN A13)
 *     bins[a][k - k_lo] = dt sum_{j<n} x[a n + j] exp(-2 pi i j k / n),   k_lo <= k < k_hi,
 * as complex64 interleaved [n_sft][k_hi-k_lo].  x holds n_sft*n doubles (16-byte aligned if on the device).
 * n = 64 .. 16384 a power of two: one shared-memory FFT per segment, the series is read once; other n: direct
 * summation over the band.  No plan needed; `stream` is a cudaStream_t or NULL; blocks until done. */
sft_status sft_compute_sfts(int32_t device, void *stream, const double *x, int64_t n_sft, int32_t n,
                            double dt, int32_t k_lo, int32_t k_hi, float *bins, int32_t mem);

/* Per-SFT noise level from the data themselves ("whitening data on a per-SFT basis"): with S_a(f_k) = s_a S(f_k)
 * (DESIGN A9) and Gaussian noise, |x~_{a,k}|^2 / (S(f_k) T_SFT / 2) is s_a times a unit exponential variate (median ln 2), so
 *     psd_scale[a] = median{ |x~_{a',k}|^2 / (S(f_k) T_SFT/2) : |a' - a| <= half_window, a' not a gap, 1 <= k <= n_samp/2 - 1 } / ln 2
 * - a median over the band (and 2 half_window + 1 neighbouring SFTs), insensitive to a narrow signal crossing it.  An SFT whose
 * bins are all exactly zero is a gap: psd_scale = 0, and it does not enter its neighbours' pools.
 *   sft_bins complex64 [n_sft][k_hi-k_lo]; psd_shape [k_hi-k_lo] or NULL (= 1); psd_scale [n_sft] out; `mem` for all three.
 * No plan needed; blocks until done.  At most 8192 pooled values per SFT (SFT_EUNSUPPORTED beyond). */
sft_status sft_estimate_psd_scale(int32_t device, void *stream, const float *sft_bins, int64_t n_sft, int32_t k_lo,
                                  int32_t k_hi, int32_t n_samp, double t_sft, const double *psd_shape,
                                  int32_t half_window, double *psd_scale, int32_t mem);

/* sft_compute_sfts + sft_load_data in one call: channel `channel` of the plan from its strain time series
 * x[n_samples] (n_samples >= n_sft * t_sft * fs; sample j of SFT a is x[a n + j], t = t0 + (a n + j)/fs).
 * The SFT bins never leave the device.  Noise description and `mem` as in sft_load_data, except that psd_scale may be NULL:
 * the per-SFT noise levels are then estimated from the data (sft_estimate_psd_scale with half_window = 0) and segments whose
 * samples are all zero become gaps. */
sft_status sft_ingest_timeseries(sft_plan *plan, int32_t channel, const double *x, int64_t n_samples,
                                 const double *psd_scale, const double *psd_shape,
                                 const float *response, int32_t mem);

/* ([x,h]) and ([h,h]) for n_templates templates (Eq.(35) P:259 with ONE df, DESIGN A1).
 *   params  [n_templates][SFT_NPARAM] doubles, row-major:
 *           m_chirp [Msun], eta, t_c [s], phi_c [rad], amp, lambda [rad], beta [rad], reserved(0)
 *   xh, hh  [n_templates] doubles (required)
 *   xh_im   [n_templates] or NULL: imaginary part of the complex sum (for the phase-maximised
 *           statistic Eq.(7)-(9) P:97-101)
 *   kc_out  [n_templates][n_channels][n_sft] int32 or NULL: the selected central bin k_c of
 *           every active pair whose SFT is present, -1 otherwise (DESIGN A5)
 *   mem     where params and all outputs live (SFT_MEM_HOST / SFT_MEM_DEVICE)
 * n_templates == 0 is SFT_OK and touches nothing.  SFT_ENODATA unless every channel is loaded. */
sft_status sft_inner_products(sft_plan *plan, int64_t n_templates, const double *params,
                              double *xh, double *hh, double *xh_im, int32_t *kc_out,
                              int32_t mem);

/* sft_inner_products for callers that may not allocate device memory inside the call (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same kernels and the same results (Eq.(35)), but the scratch
 * of the call - per-template constants, the per-chunk totals that the final reduction sums, the work-unit counter - lives in
 * one file-scope device array of SFT_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds
 * until the process exits.  The call issues no cudaMalloc / cudaFree / allocating library routine, whatever the plan did
 * before.
 *   params, xh, hh, xh_im (nullable): DEVICE pointers, shapes as in sft_inner_products; results are complete when the
 *           plan's stream reaches this point (the call returns after enqueueing; sft_plan_sync to wait).
 *   n_templates <= SFT_STATIC_MAX_TEMPLATES, else SFT_EUNSUPPORTED (outputs untouched); 0 is SFT_OK.  Larger banks: several
 *           calls on slices, or sft_inner_products.
 * The SFT axis is cut into fewer, longer chunks than sft_inner_products uses when the scratch would not hold its chunk
 * totals; the fp64 sums are then taken in a different order (differences at the 1e-15 relative level).
 * The scratch is SHARED by every plan and every call on a device and keeps the previous call's contents; the call itself
 * clears the one word that must start at zero.  Calls that overlap on the GPU (two plans on different streams, or two
 * host threads) race on it: order them on one stream or with events.  sft_static_setup(device, &bytes) resolves the
 * array's address on that device ahead of time (the first call on a device does it otherwise; do it before a capture
 * begins) and reports the size; it allocates nothing either. */
#define SFT_STATIC_MAX_TEMPLATES 4096
#define SFT_STATIC_SCRATCH_BYTES 8388608
sft_status sft_static_setup(int32_t device, int64_t *scratch_bytes /* nullable */);
sft_status sft_inner_products_static(sft_plan *plan, int64_t n_templates, const double *params,
                                     double *xh, double *hh, double *xh_im);

/* Early-warning variant ("accumulating the result over time"): inclusive prefix
 * sums over the SFT index of the per-SFT terms (summed over channels; gaps and inactive SFTs
 * add 0), carried in fp64 and stored in fp32:
 *   snr     [n_templates][n_sft] floats, SFT index fastest: cum_xh / sqrt(cum_hh), 0 where cum_hh == 0
 *   cum_xh, cum_hh  same shape, or NULL
 * At least one of the three outputs must be non-NULL. */
sft_status sft_cumulative_snr(sft_plan *plan, int64_t n_templates, const double *params,
                              float *snr, float *cum_xh, float *cum_hh, int32_t mem);

/* Statistics on top of sft_inner_products' outputs (all arrays [n_templates] doubles, `mem` as above):
 *   loglike         L = <x,h> - <h,h>/2                                   (Eq.(2)), nullable
 *   rho2_phase_max  (<x,h_c>^2 + <x,h_s>^2) / <h_c,h_c> = (xh^2 + xh_im^2) / hh, the detection statistic maximised
 *                   over distance and initial phase (Eq.(7)-(9) P:97-101; 0 where hh == 0), nullable */
sft_status sft_statistics(sft_plan *plan, int64_t n_templates, const double *xh, const double *xh_im,
                          const double *hh, double *loglike, double *rho2_phase_max, int32_t mem);

/* Validity of the per-SFT signal model for each template (Eq.(33)-(34) P:244-248): the quadratic phase model of Eq.(17) is good
 * over one SFT while 1/2 T_SFT^2 max fddot <= delta df; per template
 *   delta_eff [n_templates] doubles or NULL: 1/2 T_SFT^3 fddot at the template's last active SFT (DESIGN A12), where fddot is
 *             largest - the delta at which Eq.(33) holds with equality on this plan's T_SFT; 0 for a template with no active SFT
 *   flags     [n_templates] bytes or NULL: 1 where delta_eff > delta_max (the template leaves the regime the plan's SFT length
 *             was chosen for: expect a loss r, Eq.(36), above the one of the paper's Fig. 3/4 at that delta), else 0
 * Needs no data (channels may be unloaded).  At least one output must be non-NULL. */
sft_status sft_validity(sft_plan *plan, int64_t n_templates, const double *params, double delta_max,
                        double *delta_eff, uint8_t *flags, int32_t mem);

/* F-statistic (Eq.(10)-(13) P:107-122) for long signals whose two polarisations are resolved by the amplitude modulation of the
 * detector: h = sum_nu c_nu h_nu with the four basis waveforms h_nu = A(t) [a cos(phi), b cos(phi), a sin(phi), b sin(phi)]
 * (Eq.(11)); 2F = x^T M^-1 x with x_nu = ([x,h_nu]), M_numu = ([h_nu,h_mu]) is twice the log-likelihood Eq.(2) maximised over
 * the four amplitudes c_nu (Eq.(13)).  Needs a plan with SFT_RESP_TABLE whose table holds, per (channel, SFT), the pair of
 * antenna-pattern functions (a, b) at the SFT start (constant over the SFT) in the (re, im) slots of sft_load_data's
 * `response`; at most 2 channels.  One pass of the fused kernel accumulates the 4 + 3 sums per template; in the SFT framework
 * the products between a cos and a sin quadrature vanish and ([h_0,h_0]) = ([h_2,h_2]), ([h_1,h_1]) = ([h_3,h_3]),
 * ([h_0,h_1]) = ([h_2,h_3]), so that M has three distinct entries.
 *   twoF  [n_templates] (required); 0 where M is singular (no active SFT, or a and b proportional)
 *   xnu   [4][n_templates] or NULL: ([x,h_nu]), nu = 0..3
 *   mnu   [3][n_templates] or NULL: ([h_0,h_0]), ([h_1,h_1]), ([h_0,h_1])
 * `params`, `mem` as in sft_inner_products (phi_c enters 2F only through rounding). */
sft_status sft_fstat(sft_plan *plan, int64_t n_templates, const double *params, double *twoF,
                     double *xnu, double *mnu, int32_t mem);

/* Blocks until all work enqueued on the plan's stream has finished. */
sft_status sft_plan_sync(sft_plan *plan);

/* Number of kernels this plan has launched so far (for launch accounting in benchmarks). */
int64_t sft_plan_launch_count(const sft_plan *plan);

/* Duration [ms] of the most recent main (fused waveform+coefficient+contraction) kernel launch
 * of this plan, from CUDA events recorded on the plan's stream around that launch; blocks
 * until that launch has finished.  < 0 if nothing has been launched. */
double sft_plan_last_kernel_ms(sft_plan *plan);

/* Diagnostic: how the coefficient evaluator (rows A4/A6 of the hot path) was used by the most recent
 * sft_inner_products call that had kc_out != NULL: the number of active (template, SFT, channel) pairs
 * evaluated with the series in b = fdot T^2 about the Dirichlet kernel at order 0, 1, 2, 3 (out[0..3])
 * with the closed Fresnel form Eq.(29) P:219 (out[4]) and through the moment tables (out[5]: tier 1,
 * |b| <= 0.12; out[6]: tier 2, |b| <= 1).  The path is chosen per warp of 32 templates from the largest
 * |b| in the warp.  Blocks until that call finished.  Writes min(n_out, 7) values;
 * host pointer. */
sft_status sft_plan_path_counts(sft_plan *plan, int64_t *out, int32_t n_out);

/* SFT-length rule Eq.(33)-(34) P:244-248: the longest T_SFT for which the quadratic per-SFT phase model Eq.(17) is off by
 * at most ~delta radians, T_SFT(delta) = (2 delta / max fddot)^(1/3), for this library's inspiral waveform (DESIGN W1) up to
 * GW frequency f_max [Hz], where fddot = d^2 f/dt^2 is largest.  Host arithmetic only (no device needed).  *fddot_max
 * (nullable) receives max fddot [Hz/s^2].  Paper's Table I (1.4+1.4 Msun to 10 Hz): delta = 1 -> 73 s. */
sft_status sft_tsft_rule(double m_chirp, double eta, int32_t waveform, double f_max, double delta,
                         double *t_sft, double *fddot_max);

/* Moment tables for a bank around a known track ("Fourier transforms of the data will be computed once and will be valid for any
 * template within a given parameter-space region").  By default the tables of the table evaluator cover every window
 * position k_c of the stored band at every SFT (128 bytes x 4 nodes x (k_hi - k_lo + 2K) x n_sft per channel: 1.1 GB for
 * config 2, and out of reach for wide bands).  With a fiducial template (one parameter row, host pointer) they cover, per block
 * of 32 SFT slots, only the positions its k_c sweeps in that block +- half_width bins: templates whose windows stay inside take
 * the tables, all others the direct evaluator for those SFTs (same results within the evaluators' ~1e-6).  NULL restores the full
 * tables.  Replaces the tables: every channel must be loaded (again) afterwards.  SFT_ENOMEM if SFT_EVAL_TABLE was asked for and
 * the tables still do not fit. */
sft_status sft_plan_set_table_track(sft_plan *plan, const double *fiducial_params, int32_t half_width);

/* Bytes of device memory held by the data-moment tables (0: the plan uses the direct evaluator). */
int64_t sft_plan_table_bytes(const sft_plan *plan);

/* Tuning knob: SFTs per work unit along the time axis (0 = automatic).  Results do not depend on it
 * beyond fp64 summation order. */
sft_status sft_plan_set_chunk(sft_plan *plan, int32_t sfts_per_unit);

/* Tuning knob of sft_cumulative_snr with HOST outputs: the bank is processed in slabs of `templates_per_slab` templates
 * (rounded down to a multiple of 32, at least 32) and the matrices of a finished slab are copied to the host on a second
 * stream while the next slab is computed, so that the copy - 4 n_sft bytes per template and matrix, the part that bounds
 * the call end to end - starts after the first slab instead of after the whole bank.  0 = automatic (about 64 MB per
 * matrix and slab).  Results do not depend on it.  The copies overlap only if the host matrices are pinned
 * (cudaHostAlloc / cudaHostRegister); pageable memory works, without overlap.  If the call fails half-way, slabs already
 * finished may have been written to the host matrices. */
sft_status sft_plan_set_host_slab(sft_plan *plan, int64_t templates_per_slab);

/* Diagnostic: measures the plain-ALU pipe rates of `device` that bound this path (the
 * data store is L2 resident, so FP32 / FP64 / XU issue rates, not HBM, are the roofline).  Writes up
 * to 6 doubles, in 1e9 lane-operations per second (one FMA = one operation):
 *   out[0] fma.rn.f32, out[1] fma.rn.f32x2 (2 lanes per instruction), out[2] fma.rn.f64,
 *   out[3] rcp.approx.f32 (XU/MUFU), out[4] a 4:1 FFMA:MUFU mix (all its operations counted);
 *   out[5] (not Gop/s) warp instructions per clock and scheduler sustained on the instruction mix of the
 *   moment-table kernel with all dependencies and memory stalls removed: the ceiling for that mix.
 * Runs a few ms of synthetic kernels on the device's default stream; touches no plan.  Errors are
 * reported through sft_last_error(NULL). */
sft_status sft_measure_alu_peaks(int32_t device, double *out_gops, int32_t n_out);

/* Message for the last error of this plan ("" if none).  With plan == NULL: the message of the
 * last failed sft_plan_create in this thread.  The pointer stays valid until the next call. */
const char *sft_last_error(const sft_plan *plan);

/* Library version string. */
const char *sft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SFT_B200_H */
