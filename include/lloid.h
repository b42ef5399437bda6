/* lloid.h -- C ABI of the B200-native LLOID multirate SVD matched-filter hot path.
 *
 * The operations are those of arxiv/paper_2511_04730 (SGNL), Sec. II.C-II.D.1; citations are
 * /root/reference/PAPER.md:<line>.  Symbols follow the paper: f0 strain rate, slice s with rate f^s,
 * N^s taps, L^s orthonormal basis filters u_l^s (Eq. 3), reconstruction matrix
 * sigma_l nu_il (Eq. 6), M complex templates = 2M real rows.
 *
 * One push of a strain buffer runs, entirely in CUDA kernels on the caller's stream:
 *   a1 decimate   d_r[j] = sqrt(D) sum_k ghat_D[k] d[jD + c - k], c = n_down*D      (Eq. 4)
 *   a2 correlate  Y^s[l,j] = sum_n u_l^s[n] d_{f^s}[j - delay_s - N^s + 1 + n]     (Eq. 5; Eq. 9, 167-185)
 *   a3 reconstruct + a4 combine   rho = sum_s Up(...Up(R^s Y^s))                    (Eqs. 6-9, Fig. 4)
 *   a5 peaks      per template j: first k maximising rho_2j[k]^2 + rho_2j+1[k]^2
 * SNR sample k of a push is stream sample n0+k (n0 = samples pushed before); it reads strain <= n0+k only.
 *
 * All pointers are plain host or device pointers as stated per argument; no C++/torch types cross this
 * boundary.  Every function returns 0 (LLOID_OK) or a negative lloid_status and lloid_last_error()
 * (thread-local) describes the reason.  Argument/state errors (EINVAL, ELATENCY, ESTATE, ENOMEM) change nothing.
 * LLOID_ECUDA from lloid_stream_push means a kernel launch failed part-way: the stream's device state is then
 * inconsistent and every further push returns LLOID_ESTATE until lloid_state_reset.  There is no CPU fallback: every call that
 * computes needs a CUDA device of compute capability 10.0 (sm_100a).
 */
#ifndef LLOID_H_
#define LLOID_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LLOID_OK = 0,
  LLOID_EINVAL = -1,   /* null pointer, bad size, rate not a power-of-two divisor of f0, rates increasing with s,
                          slices that do not abut, delay[0] != 0, buffer_len not a multiple of max D_s */
  LLOID_ELATENCY = -2, /* a slice with f^s < f0 whose delay is shorter than the look-ahead of its decimator and
                          upsample chain: delay_s < n_down + H_g (PAPER.md:161-163 causality condition) */
  LLOID_ENOMEM = -3,   /* host or device allocation failed */
  LLOID_ECUDA = -4,    /* a CUDA runtime/driver call failed, or the device is not sm_100 */
  LLOID_ESTATE = -5    /* call not valid in this state (debug_bank out of range; push after a failed push) */
} lloid_status;

typedef enum {
  LLOID_PREC_FP32_FFMA = 0, /* every contraction in fp32 on the CUDA cores (gate 1e-4 of SNR rms)              */
  LLOID_PREC_F16 = 1,       /* tcgen05 kind::f16, operands rounded once to fp16, fp32 accumulate in TMEM         */
  LLOID_PREC_F16_SPLIT = 2  /* default (gate 2e-3, measured 2e-4): fp16 main product + one fp8 (e4m3 x e5m2) MMA that
                               carries both hi/lo cross terms a_hi b_lo + a_lo b_hi: 2 MMAs per product            */
} lloid_precision;

/* One time slice of an SVD bank.  Arrays may be host or device memory; create copies them. */
typedef struct {
  int32_t rate_hz;     /* f^s: power of two, divides strain_rate_hz, non-increasing with s, rate_hz[0] = f0  */
  int32_t n_taps;      /* N^s, samples at rate_hz                                                            */
  int32_t n_basis;     /* L^s >= 1                                                                           */
  int64_t delay;       /* t^s * rate_hz: samples (at rate_hz) between the merger and this slice's newest tap;
                          delay[0] = 0; slices abut: (delay_s + n_taps_s)/rate_s = delay_{s+1}/rate_{s+1}     */
  const float *basis;  /* U^s [n_basis][n_taps] row-major, orthonormal rows, oldest tap first                 */
  const float *recon;  /* R^s [2*M][n_basis] row-major = V diag(sigma); row 2j = real, 2j+1 = imaginary part  */
} lloid_slice;

/* Per-template, per-buffer trigger (time, SNR, phase; integer sample). */
typedef struct {
  float snr;           /* max_k |rho_2j[k] + i rho_2j+1[k]| over the pushed buffer                            */
  int32_t sample;      /* first k of the trigger window attaining it: in [0, buffer_len), or in [-trigger_overlap, 0)
                          when the peak lies in the overlap with the previous buffer; LLOID_NO_TRIGGER if snr is
                          below options.threshold                                                              */
  float phase;         /* atan2(rho_2j+1[k], rho_2j[k]) at that k                                             */
} lloid_peak;

typedef struct {
  int32_t n_down;      /* decimator half length in output samples; default 32                  */
  int32_t n_up;        /* upsampler half length in input samples; default 8 (only 8 supported) */
  int32_t precision;   /* lloid_precision; default LLOID_PREC_F16_SPLIT                                      */
  float threshold;     /* report only peaks with snr >= threshold; 0 = report every template's peak          */
  int32_t trigger_overlap; /* samples by which the trigger window of a push extends back into the previous buffer
                          (Fig. 5: light travel time + 0.005 s, e.g. 67 at 2048 Hz); default 0.
                          0 <= trigger_overlap < buffer_len; needs a tensor-core precision                       */
} lloid_options;
#define LLOID_NO_TRIGGER (-2147483647 - 1)

/* One coincident event of a bank in one trigger window. */
#define LLOID_MAX_DET 4
typedef struct {
  int32_t template_index; /* template (index in the stream's peak order) of the event, -1 = no coincidence in this bank */
  int32_t det_mask;       /* bit a set: detector a takes part                                                     */
  float net_snr;          /* sqrt(sum over participating detectors of snr^2)                                       */
  int32_t reserved;
  float snr[LLOID_MAX_DET]; int32_t sample[LLOID_MAX_DET]; float phase[LLOID_MAX_DET]; /* the participating triggers */
} lloid_event;

typedef struct lloid_bank lloid_bank;      /* opaque, immutable after create; owns host+device copies of U, R */
typedef struct lloid_stream lloid_stream;  /* opaque; owns the device rings / state of (banks x detectors)    */

/* Fill *opt with the defaults above. */
void lloid_options_default(lloid_options *opt);

/* Build one SVD bank of M complex templates from its slice table ("during
 * initialization").  `slices[s].basis/recon` may be host or device pointers and may be freed on return.
 * opt == NULL means defaults.  Errors: EINVAL, ELATENCY, ENOMEM, ECUDA. */
int lloid_bank_create(lloid_bank **out, int32_t strain_rate_hz, int32_t n_templates, int32_t n_slices,
                      const lloid_slice *slices, const lloid_options *opt);
void lloid_bank_destroy(lloid_bank *bank);

/* A stream filters n_detectors independent strain series against every bank (same banks for all
 * detectors: flat-PSD synthetic case; per-detector banks = one stream per detector).
 * buffer_len (f0 samples per push) must be a multiple of every bank's largest decimation factor.
 * cuda_stream is a cudaStream_t (NULL = legacy default stream); all work of push/reset is enqueued on it.
 * All banks must use the same precision, n_down and threshold (EINVAL otherwise) and must outlive the stream. */
int lloid_stream_create(lloid_stream **out, const lloid_bank *const *banks, int32_t n_banks,
                        int32_t n_detectors, int32_t buffer_len, void *cuda_stream);
void lloid_stream_destroy(lloid_stream *stream);

/* Push one buffer.  Asynchronous on the stream's cuda_stream; no host synchronisation inside.
 *   strain     DEVICE, [n_detectors][buffer_len] fp32 whitened strain (gaps = zeros)
 *   peaks      DEVICE, [n_detectors][sum_b M_b] lloid_peak, banks in creation order
 *   snr_debug  DEVICE or NULL: [n_detectors][2*M_debug][buffer_len] fp32, the full SNR series of bank
 *              `debug_bank` (row 2j real, 2j+1 imaginary).  NULL in production: SNR never reaches HBM.
 * Buffers are caller-owned and must stay valid until the stream reaches the end of this push. */
int lloid_stream_push(lloid_stream *stream, const float *strain, lloid_peak *peaks, float *snr_debug,
                      int32_t debug_bank);

/* Coincidence formation and clustering on the triggers of one push, asynchronous on the stream's
 * cuda_stream.  A trigger exists where peaks[det][j].sample != LLOID_NO_TRIGGER.  For every template the detector set
 * (>= 2 detectors of the SAME template, every pair within its window) with the largest network SNR is its candidate;
 * each bank keeps the candidate with the highest network SNR (ties: lower bit mask, lower template index).
 *   peaks       DEVICE, [n_detectors][sum_b M_b] as written by lloid_stream_push (n_detectors <= LLOID_MAX_DET)
 *   dt_samples  HOST, [n_detectors][n_detectors] symmetric coincidence windows in strain samples, inclusive
 *               (light travel time + 0.005 s; e.g. ceil(0.0150 * f0) for H-L)
 *   events      DEVICE, [n_banks] lloid_event
 * Errors: EINVAL (null pointer, more than LLOID_MAX_DET detectors, negative window), ECUDA. */
int lloid_stream_events(lloid_stream *stream, const lloid_peak *peaks, const int32_t *dt_samples, lloid_event *events);

/* SVD bank construction on the GPU (Eq. 3): truncated singular value decomposition of one time slice's
 * template matrix, the inputs lloid_bank_create takes.  One-sided Jacobi in float64 (own kernels, no library); synchronous.
 *   H            HOST or DEVICE, [n_rows][n_taps] float64 row-major: the 2M real template rows of the slice
 *   energy       keep the smallest L with sum_{l<L} sigma_l^2 >= energy * sum sigma^2 (0.9999 in BASELINE.json)
 *   basis_out    DEVICE, capacity [max_basis][n_taps] fp32: U, L orthonormal rows written compactly as [L][n_taps]
 *   recon_out    DEVICE, capacity [n_rows][max_basis] fp32: R = V diag(sigma), written compactly as [n_rows][L]
 *   n_basis_out  HOST: L;  singular_out HOST [max_basis] or NULL: sigma_0 >= sigma_1 >= ...;  kept_energy_out HOST or NULL
 * H ~= R U with relative residual energy 1 - kept_energy.  Singular vectors are defined up to sign (and up to a rotation
 * inside a cluster of equal singular values); the product R U is unique.  Errors: EINVAL (sizes, L > max_basis), ENOMEM, ECUDA. */
int lloid_svd_slice(const double *H, int32_t n_rows, int32_t n_taps, double energy, int32_t max_basis, int32_t *n_basis_out,
                    float *basis_out, float *recon_out, double *singular_out, double *kept_energy_out, void *cuda_stream);

/* The same decomposition for callers that may not allocate device memory (a tight serving loop, a harness that forbids
 * cudaMalloc): calls no cudaMalloc / cudaFree or allocating library routine.  The working set lives in a fixed device array
 * inside the library (2.13 MiB, held by every GPU that loads the library until exit), hence the limits
 *   n_rows <= 128 and n_taps <= 2048   (LLOID_SVD_NOALLOC_MAX_ROWS / _TAPS; larger -> EINVAL, use lloid_svd_slice)
 * and H must be a DEVICE pointer (a host pointer is rejected with EINVAL: no staging buffer exists).  All other arguments,
 * the results and the error codes are those of lloid_svd_slice (never ENOMEM).  Synchronous.  Every call on a device shares
 * the array: calls that overlap on one GPU (two streams, two host threads) race and return garbage -- serialise them. */
#define LLOID_SVD_NOALLOC_MAX_ROWS 128
#define LLOID_SVD_NOALLOC_MAX_TAPS 2048
int lloid_svd_slice_noalloc(const double *H, int32_t n_rows, int32_t n_taps, double energy, int32_t max_basis,
                            int32_t *n_basis_out, float *basis_out, float *recon_out, double *singular_out,
                            double *kept_energy_out, void *cuda_stream);

/* xi^2 in the stream (Eq. 10).  lloid_bank_set_autocorrelation attaches the bank's template
 * autocorrelations (before lloid_stream_create): acorr [n_templates][2*delta+1][2] fp32 (re, im), host or device, R_j(t) for
 * t = -delta..delta with R_j(0) = 1 (definition below).  When EVERY bank of a stream carries autocorrelations of one delta
 * (and the stream is LLOID_PREC_F16_SPLIT with buffer_len a multiple of 128 and > delta) every push also keeps its
 * upsampled basis outputs in a three-buffer history ring, and lloid_stream_xi2 evaluates Eq. 10 for the triggers of the push
 * BEFORE the last one (their windows reach delta samples into the last push: the padding / latency of Fig. 5) with a second
 * reconstruction pass over [-delta, buffer_len + delta) whose epilogue accumulates |z - z(0) R_j|^2 over each template's own
 * window; the SNR is still never written to HBM.
 *   xi2_out  DEVICE, [n_detectors][sum_b M_b] fp32, aligned with the peaks of that push; -1 where it reported no trigger.
 * Samples before the start of the stream count as zero.  Errors: EINVAL, ESTATE (not enabled / fewer than two pushes), ECUDA. */
int lloid_bank_set_autocorrelation(lloid_bank *bank, const float *acorr, int32_t delta);
int lloid_stream_xi2(lloid_stream *stream, float *xi2_out);

/* Signal-based consistency statistic xi^2 of Eq. 10 for the triggers of ONE bank whose SNR series is
 * materialised in device memory (the snr_debug output of lloid_stream_push; the caller keeps consecutive buffers side by
 * side so that the +-delta samples around a trigger are present -- the padding of Fig. 5 -- and calls this one buffer
 * later).  Asynchronous on cuda_stream.
 *   snr             DEVICE, [2*n_templates][n_samples] fp32, row 2j real, 2j+1 imaginary part of z_j
 *   trigger_sample  DEVICE, [n_templates] index of the trigger in [0, n_samples), LLOID_NO_TRIGGER = none
 *   acorr           DEVICE, [n_templates][2*delta+1][2] fp32 (re, im): R_j(t), t = -delta..delta, R_j(0) = 1,
 *                   R_j(t) = sum_m g[m] conj(g[m+t]) / sum |g|^2 for the complex template g = h_2j + i h_2j+1
 *   delta           half width in samples: (autocorrelation length - 1) / 2, 175 or 350 in the paper
 *   xi2_out         DEVICE, [n_templates] fp32; -1 where there is no trigger.  Samples outside [0, n_samples) count as 0.
 * Errors: EINVAL, ECUDA. */
int lloid_xi2_series(const float *snr, int32_t n_templates, int64_t n_samples, const int32_t *trigger_sample,
                     const float *acorr, int32_t delta, float *xi2_out, void *cuda_stream);

/* PSD estimation + whitening front end (Figs. 2-3), the step before the path.  Per detector and push:
 * the newest fft_len - 2 zero_pad input samples times a Hann window, zero padded to fft_len -> FFT -> per bin the median of
 * the last n_median instantaneous PSDs updates a running geometric mean over n_average blocks (PSD = its arithmetic-mean
 * equivalent) -> divide by sqrt(PSD), drop the bins above rate_out / 2 (frequency-domain downsampling) -> inverse FFT ->
 * Tukey window (tapers of zero_pad) -> overlap-add.  One push takes hop_in = fft_len / 2 - zero_pad samples at rate_in and
 * returns hop_out = hop_in * rate_out / rate_in samples at rate_out of unit variance, lagging the input by fft_len / 2
 * input samples.  Paper values: rate_in 16384, rate_out 2048, fft_len 4 s, zero_pad 1 s, n_median 7.  Zero history at
 * start; gaps and gating are not handled.  The FFTs are cuFFT transforms (libcufft.so.11 is loaded at create).
 *   strain_in  DEVICE [n_detectors][hop_in] fp32        white_out  DEVICE [n_detectors][hop_out] fp32
 *   psd_out    DEVICE [n_detectors][psd_bins] fp32 one-sided PSD per Hz at bin k * rate_in / fft_len, or NULL
 * Errors: EINVAL (sizes), ENOMEM, ECUDA (cuFFT missing or failing, launch failure). */
typedef struct lloid_whitener lloid_whitener;
int lloid_whitener_create(lloid_whitener **out, int32_t n_detectors, int32_t rate_in, int32_t rate_out, int32_t fft_len,
                          int32_t zero_pad, int32_t n_median, int32_t n_average, void *cuda_stream);
int lloid_whitener_push(lloid_whitener *w, const float *strain_in, float *white_out, float *psd_out);
int lloid_whitener_reset(lloid_whitener *w);
void lloid_whitener_destroy(lloid_whitener *w);
int32_t lloid_whitener_hop_in(const lloid_whitener *w);
int32_t lloid_whitener_hop_out(const lloid_whitener *w);
int32_t lloid_whitener_psd_bins(const lloid_whitener *w);

/* Same through HOST buffers: copies strain host->device, pushes, copies peaks device->host and waits for
 * the stream.  strain_host [n_detectors][buffer_len], peaks_host [n_detectors][sum_b M_b]; pinned memory
 * makes the copies asynchronous but is not required. */
int lloid_stream_push_host(lloid_stream *stream, const float *strain_host, lloid_peak *peaks_host);

/* Pipelined form of lloid_stream_push_host for a caller that pushes buffer after buffer: returns as soon as the copies and
 * kernels are queued; a second CUDA stream copies the peaks of call n to peaks_host while call n + 1 computes (two device
 * peak buffers).  Ownership: strain_host and peaks_host of call n belong to the library until call n + 2 has returned or
 * lloid_stream_host_sync has -- alternate between two pairs of PINNED buffers (pageable memory makes the copies
 * synchronous and the call pointless).  The peaks of call n are complete at the same moment.  lloid_stream_host_sync waits
 * for everything queued.  Do not mix with lloid_stream_push_host / lloid_stream_push on the same stream object without a
 * lloid_stream_host_sync in between.  Errors: EINVAL (null pointer), ESTATE (stream failed earlier), ECUDA. */
int lloid_stream_push_host_async(lloid_stream *stream, const float *strain_host, lloid_peak *peaks_host);
int lloid_stream_host_sync(lloid_stream *stream);

/* Zero all rings and the stream clock: the next push is stream sample 0 (zero history). */
int lloid_state_reset(lloid_stream *stream);

/* Introspection (host values, no device work). */
int64_t lloid_stream_samples_pushed(const lloid_stream *stream);
int32_t lloid_stream_total_templates(const lloid_stream *stream);
int32_t lloid_stream_launches_per_push(const lloid_stream *stream); /* kernels this library launches per push */
/* Executed and algorithmic work of one push, for roofline accounting:
 * out[0] a2 flop executed (padded tiles, x3 for the hi/lo split), out[1] a3 flop executed,
 * out[2] a2 algorithmic flop 2 sum_s L^s N^s f^s (Eq. 5), out[3] a3 algorithmic flop 2 sum_s 2M L^s f^s (Eq. 6, the
 * paper's order), out[4] a4 algorithmic flop 16*2M*sum_stages f_out (Eqs. 7-9), out[5] bytes of operands (U, R)
 * one push reads, out[6] bytes of Y / upsampled-Y intermediates written + read, out[7] reserved (0). */
int lloid_stream_work_per_push(const lloid_stream *stream, double out[8]);

/* Per-stage device timing (bench / roofline evidence).  When enabled, every push records CUDA events on the
 * stream between its kernels: stage 0 a1 decimate, 1 a2 correlate, 2 basis-domain upsample, 3 a3 reconstruct +
 * a5 peaks, 4 peak finalisation.  lloid_stream_stage_times synchronises the stream, adds the elapsed
 * milliseconds of every push since the last call into ms[0..LLOID_N_STAGES), returns the number of pushes
 * covered (or a negative status) and clears the record. */
#define LLOID_N_STAGES 5
int lloid_stream_set_stage_timing(lloid_stream *stream, int32_t enable);
int lloid_stream_stage_times(lloid_stream *stream, float ms[LLOID_N_STAGES]);
const char *lloid_stage_name(int32_t stage);

const char *lloid_last_error(void);
const char *lloid_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LLOID_H_ */
