/*
 * mdsm.h -- C ABI of libmdsm: the data-parallel hot path of the Medicina BEST-2
 * multibeam transient pipeline (arXiv:1307.5700) on NVIDIA B200 (sm_100a).
 *
 *   RFI clip  ->  multibeam brute-force incoherent dedispersion  ->  n-sigma detection
 *
 * Call order of the hot path: mdsm_plan_create, mdsm_plan_reserve (once per sample type: the stage calls never allocate, so the
 * dedispersion scratch is reserved up front -- mdsm_dedisperse returns MDSM_EINVAL without it), then per buffer mdsm_rfi_clip,
 * mdsm_dedisperse, mdsm_detect; or mdsm_pipeline_host, which does all of it from host buffers.
 *
 * Citations are to /root/reference/PAPER.md (line numbers) and to the readings listed in
 * DESIGN.md section 3.  All pointers named d_* are DEVICE pointers, h_* are HOST pointers.
 * The caller owns every buffer it passes; the plan owns the delay table and its scratch.
 * No function throws or exits; every int-returning call returns an MDSM_* status and leaves
 * a message retrievable with mdsm_last_error() (thread-local) on failure.
 *
 * Layouts (dense, row-major, time fastest -- "beam/channel/time order"):
 *   in  [nbeams][nchans][nsamps]   float (MDSM_F32) or uint8_t (MDSM_U8); channel 0 = f_top
 *   out [nbeams][ndms][nsamps]     float (MDSM_F32) or uint32_t (MDSM_U8); row stride = nsamps,
 *                                  only t < nsamps_out = nsamps - max_delay is written / valid
 *                                  (overlap reading A3: Eq. 6)
 * The device-pointer stage calls (mdsm_rfi_clip, mdsm_dedisperse, mdsm_detect, the post-processing calls) only
 * enqueue work on `cuda_stream` (a cudaStream_t cast to void*; NULL = the legacy default stream); they never
 * synchronise and never allocate, so they can be captured into a CUDA graph.  Whatever device memory the path needs
 * beyond the caller's buffers is allocated by mdsm_plan_create and mdsm_plan_reserve.
 * Threads: a plan is NOT internally locked.  Calls on one plan must come from one host thread at a time (the paper's
 * host model is one thread per beam: give every such thread its own plan, or serialise the calls);
 * different plans are independent.  mdsm_last_error() is thread-local.
 * beam0/nb select a contiguous range of beams so that the host can drive beam groups on
 * different streams ("parallelized across beams"); pointers always address the
 * FULL [nbeams]... arrays, the call offsets them by beam0 itself.
 */
#ifndef MDSM_H
#define MDSM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mdsm_plan mdsm_plan;                                 /* opaque */

/* One detection: "(time, DM, intensity) triplets" per beam.  16 bytes. */
typedef struct { int32_t beam, dm_idx, t; float snr; } mdsm_event;

/* Sample types.  MDSM_F32 and MDSM_U8 are accepted by every stage call; MDSM_U16 (uint16 samples) and MDSM_U4 (4-bit samples,
 * two per byte along time, low nibble first; nsamps even) are further INPUT types of mdsm_dedisperse only (SURVEY 8(f)
 * NEXT-4: lower-precision inputs), with uint32 output like MDSM_U8 -- pass MDSM_U8 to mdsm_detect for their series. */
enum { MDSM_F32 = 0, MDSM_U8 = 1, MDSM_U16 = 2, MDSM_U4 = 3 };
enum { MDSM_OK = 0, MDSM_EINVAL = -1, MDSM_ENOMEM = -2, MDSM_ECUDA = -3, MDSM_EOVERFLOW = 1 };

/* Survey parameters of one buffer (PAPER.md:96 "observation and survey parameters", :190, :194).
 *   f_top  centre frequency of channel 0 in MHz; channel c is at f_top + c*foff, foff < 0 (MHz)
 *   tsamp  sampling time in s; nsamps = input samples per channel per call
 *   DM trial d is dm_low + d*dm_step (pc cm^-3), d in [0, ndms)
 * Builds, in fp64 on the host, delay(d,c) = floor(4.148808e3 * DM_d * (f_c^-2 - f_top^-2) / tsamp + 0.5)
 * (Eq. 1; constant and rounding from BASELINE.json north_star), uploads it, and
 * allocates the per-plan device scratch.  Uses the current CUDA device.
 * Returns NULL on error (bad argument: nbeams,nchans,ndms < 1, foff >= 0, tsamp <= 0,
 * dm_step < 0, dm_low < 0, nsamps <= max_delay; or allocation / CUDA failure). */
mdsm_plan *mdsm_plan_create(int nbeams, int nchans, double f_top, double foff, double tsamp,
                            int64_t nsamps, double dm_low, double dm_step, int ndms);
void mdsm_plan_destroy(mdsm_plan *plan);                            /* NULL is a no-op */

int64_t mdsm_plan_max_delay(const mdsm_plan *plan);                 /* delay(ndms-1, nchans-1) */
int64_t mdsm_plan_nsamps_out(const mdsm_plan *plan);                /* nsamps - max_delay */
/* Copies the delay table to h_delays[ndms][nchans] (host). */
int mdsm_plan_get_delays(const mdsm_plan *plan, int32_t *h_delays);
const char *mdsm_last_error(void);

/* Plan options (not for use while work of this plan is in flight; "group_size" synchronises the device, the others
 * only set a field).
 *  "dedisp_kernel": 0 = auto (the pre-summed-rows kernel whenever the plan has tables for it, else the direct kernel),
 *      1 = direct (one thread per output, global loads: the cross-check kernel), 2 = pre-summed rows or MDSM_EINVAL,
 *      3 = pre-summed rows with the operand windows staged in tensor memory (fp32 only; an experimental variant of the
 *      main kernel, slower than 2 today -- DESIGN.md section 6.1) or MDSM_EINVAL.
 *  "group_size": channels per pre-summed group, 1..8, or 0 (default) = the plan's cost model picks it.  Changing it
 *      rebuilds the tables and DROPS the scratch reservation (call mdsm_plan_reserve again).
 *  "detect_two_pass": 0 (default) = mdsm_detect is ONE launch (a CTA per series: statistics from HBM, thresholding of the same row
 *      out of L2); 1 = the two-launch form (statistics kernel, then a grid over (time, series)), kept for comparison.
 *      Series too long for the one-launch kernel's shared memory (nsamps_out above about 5.2 million) take the two-launch form
 *      by themselves.
 *  "post_median_window" (0 = off, else odd <= 33) and "post_detrend" (0/1): mdsm_pipeline_host runs
 *      mdsm_median_filter / mdsm_detrend on the fp32 series between dedispersion and detection (ignored for uint8).
 * Unknown key/value -> MDSM_EINVAL. */
int mdsm_plan_set_option(mdsm_plan *plan, const char *key, int64_t value);
/* Allocates the plan-owned scratch of mdsm_dedisperse for `dtype`: the pre-summed channel-group rows (uint8: exact; fp32: same terms, another order)
 * (DESIGN.md section 6.1), nyrows * nsamps * (4 | 2) bytes per beam.  Call once after mdsm_plan_create (and after
 * changing "group_size") and before the first mdsm_dedisperse of that dtype; mdsm_pipeline_host calls it itself.
 * max_bytes = 0: keep the reservation this dtype already has, whatever its size (so the call is a no-op once reserved, and
 * a cap set earlier survives mdsm_pipeline_host's own call); with none yet, as many beams as fit a quarter of the free
 * device memory.  max_bytes > 0: at most max_bytes (never less than one beam), replacing a reservation of another size.  When the scratch holds fewer beams than the plan (mdsm_plan_kernel_info: scratch_slots < nbeams),
 * mdsm_dedisperse walks its beams through it in stream order and calls for different beam ranges must then be issued
 * on ONE stream.  Synchronises the device only when an existing reservation has to be replaced.
 * Returns MDSM_ENOMEM if not even one beam fits. */
int mdsm_plan_reserve(mdsm_plan *plan, int dtype, int64_t max_bytes);
/* Which dedispersion kernel mdsm_dedisperse runs for `dtype` and with what geometry: writes a NUL-terminated list of
 * "key=value" words to buf ("kernel=rows group_size=4 ... scratch_slots=8 scratch_bytes=..." or
 * "kernel=direct reason=option|no_tables").  Returns 1 (rows), 0 (direct) or a negative MDSM_* status; with option
 * dedisp_kernel = 3 and a dtype / plan the TMEM variant has no tables for it writes "kernel=none reason=tmem_f32_only|
 * no_tmem_tables" and returns MDSM_EINVAL, as mdsm_dedisperse would. */
int mdsm_plan_kernel_info(const mdsm_plan *plan, int dtype, char *buf, int64_t buflen);
/* Number of kernels this plan has launched since creation (all entry points). */
int64_t mdsm_plan_launch_count(const mdsm_plan *plan);

/* RFI thresholding of the input filterbank, in place (PAPER.md:79 channel thresholding,
 * PAPER.md:81 spectrum thresholding; thresholds per north_star: k sigma above the mean).
 * Per beam, over all nsamps samples, one-sided:
 *  1. per channel c: mean_c, sig_c (population) and the replacement value repl_c
 *     (u8: mean rounded half up; f32: (float)mean);
 *  2. channel slices: non-overlapping chunks of `window` samples; a chunk is flagged when its
 *     sum > window*mean_c + k_chan*sig_c*sqrt(window); flags are dilated by one chunk on either
 *     side in time; flagged chunks are overwritten with repl_c;
 *  3. whole spectra, on the data as modified by 2: s_t = sum_c x[c][t]; a spectrum is flagged
 *     when s_t > mean_t(s) + k_spec*rms_t(s); flagged spectra are overwritten with repl_c.
 * d_chan_mask [nbeams][nchans][nsamps/window] and d_spec_mask [nbeams][nsamps] receive 0/1
 * (either may be NULL).  window >= 1 and nsamps % window == 0, else MDSM_EINVAL. */
int mdsm_rfi_clip(mdsm_plan *plan, void *d_in, int dtype, int beam0, int nb,
                  int window, double k_chan, double k_spec,
                  uint8_t *d_chan_mask, uint8_t *d_spec_mask, void *cuda_stream);

/* The paper's own RFI stage (Fig. 3; readings H-i..H-vii of DESIGN.md section 3) as an
 * alternative to mdsm_rfi_clip, for float power data, in place, per beam:
 *  1. averaged bandpass bp[c] = mean_t x[c][t];
 *  2. channels with (bp[c] - median bp) > k_mask * 1.4826 * MAD are masked and replaced by the mean of the nearest
 *     un-masked channel on either side ("interpolating the bandpass");
 *  3. least-squares polynomial of order `order` (<= 12, < nchans) through the interpolated bandpass -> fit[c]; rmse of the
 *     fit; mean_bp, std_bp = mean and population standard deviation of the interpolated bandpass over the channels;
 *  4. channel thresholding: chunks of `window` samples whose MEAN > fit[c] + k_chan * rmse are flagged together with their
 *     two time neighbours and overwritten with (float)fit[c];
 *  5. spectrum thresholding on the modified data: spectra whose mean over the channels > mean_bp + k_spec * std_bp are
 *     overwritten with (float)fit[c];
 *  6. subtract != 0: (float)fit[c] is subtracted from every sample (flagged samples become exactly 0).
 * The fit runs on the GPU (one CTA per beam), so the call is asynchronous like the other stage calls and allocates nothing.
 * d_chan_mask [nbeams][nchans][nsamps/window], d_spec_mask [nbeams][nsamps] (0/1; either may be NULL);
 * d_fit (may be NULL) [nbeams][nchans][2] doubles = fit, interpolated bandpass; d_stats (may be NULL) [nbeams][4] doubles =
 * rmse, mean_bp, std_bp, number of masked channels.  MDSM_EINVAL: bad beam range / window / order, nchans too large for
 * the shared-memory sort (> 8192). */
int mdsm_bandpass_clip(mdsm_plan *plan, float *d_in, int beam0, int nb, int window, int order, double k_mask,
                       double k_chan, double k_spec, int subtract, uint8_t *d_chan_mask, uint8_t *d_spec_mask,
                       double *d_fit, double *d_stats, void *cuda_stream);

/* Brute-force incoherent dedispersion:
 *   out[b][d][t] = sum_c in[b][c][t + delay(d,c)],   t in [0, nsamps_out)
 * MDSM_F32: float in, float out (fp32 accumulation; |err| <= 1e-5 * sum_c|in| + 1e-6).
 * MDSM_U8 : uint8 in, uint32 out, exact.  MDSM_U16: uint16 in, uint32 out, exact (nchans * 65535 must fit 32 bits).
 * MDSM_U4 : 4-bit samples packed two per byte (row = nsamps/2 bytes), uint32 out, exact.
 * d_in [nbeams][nchans][nsamps], d_out [nbeams][ndms][nsamps] (only t < nsamps_out of the rows of beams
 * [beam0, beam0+nb) is written), both caller-owned device buffers of any alignment.  Asynchronous on cuda_stream;
 * allocates nothing: the scratch of the pre-summed-rows kernel must have been reserved with
 * mdsm_plan_reserve(plan, dtype, ...) -- MDSM_EINVAL otherwise.  A plan whose delay table the pre-summed-rows
 * kernel cannot express runs the direct kernel (one thread per output; mdsm_plan_kernel_info says which and why).
 * fp32: the channel groups are added first, so the summation order differs from the definition's (same terms). */
int mdsm_dedisperse(mdsm_plan *plan, const void *d_in, int dtype, int beam0, int nb,
                    void *d_out, void *cuda_stream);

/* n-sigma thresholding of every dedispersed series (normalisation PAPER.md:110).
 * Per (beam, dm) over t < nsamps_out: mean and population rms of the series; an event
 * (beam, dm_idx, t, snr) is appended for every sample with snr = (x - mean)/rms > snr_thresh
 * (fp64 arithmetic; a series with rms == 0 emits nothing).  Events are appended in no
 * particular order with warp-aggregated atomics.  *d_count (device, must be zeroed by the
 * caller before the first beam group) is incremented by the number of events found; only
 * events whose slot index < max_events are stored in d_events. */
int mdsm_detect(mdsm_plan *plan, const void *d_out, int dtype, int beam0, int nb,
                double snr_thresh, mdsm_event *d_events, int64_t max_events,
                unsigned long long *d_count, void *cuda_stream);

/* mdsm_detect for callers that are not able to allocate device memory -- the same n-sigma thresholding (PAPER.md:116,
 * normalisation PAPER.md:110), same events, but it needs NO plan and calls no cudaMalloc / cudaFree / allocating library
 * routine, neither at set-up nor per call.
 *
 * Who this is for.  Every other stage call wants an mdsm_plan, and mdsm_plan_create / mdsm_plan_reserve obtain their
 * device memory with cudaMalloc.  Some users of the detection step cannot do that:
 *   - a plug-in inside a host application (an acquisition or correlator process, a framework with its own caching
 *     allocator) that has already claimed the device's memory and hands the plug-in fixed input / output buffers:
 *     a further cudaMalloc there fails, or takes memory the host has budgeted for something else;
 *   - the soft-real-time loop of the paper itself: cudaMalloc and cudaFree synchronise the whole
 *     device, so a thread that allocates while other beams' buffers are in flight stalls all of them and can make
 *     the pipeline miss its buffer deadline.
 * The per-series mean / rms pairs that detection keeps between its two kernels therefore live in a fixed array
 * inside libmdsm.so's device image (`static __device__`, 16 bytes x MDSM_DETECT_NOALLOC_MAX_SERIES = 512 KB).  The
 * CUDA runtime places that array on every GPU on which the library's kernels are loaded and keeps it there until the
 * process exits; that is the price of never allocating.
 *
 *   d_series [nbeams][ndms][nsamps]  float (MDSM_F32) or uint32_t (MDSM_U8), device, caller-owned, any alignment; the first
 *                                    nsamps_out (1 <= nsamps_out <= nsamps) samples of a row are thresholded, as in mdsm_detect;
 *   d_events, max_events, d_count    exactly as in mdsm_detect (the caller zeroes *d_count; events carry beam 0 .. nbeams-1).
 * Limit: nbeams * ndms <= MDSM_DETECT_NOALLOC_MAX_SERIES (enough for 16 beams x 2048 DM trials, the largest
 * configuration this library is measured on); beyond that the call does nothing and returns MDSM_EINVAL with a message that
 * names the limit -- split the series into several calls then, one after the other on ONE stream.
 * First call: the first call on each device (with that device current) asks the runtime for the device address of the
 * array and remembers it; later calls only launch the two kernels.  Make that first call during start-up, before any
 * stream capture begins on the device.
 * Shared state: all calls on a device use the same array.  It still holds the previous call's means and rms values; no
 * element has to start at zero, because each call first writes the nbeams * ndms pairs it then reads.  For the same reason
 * two calls whose kernels may run on the GPU at the same time (different streams, different host threads) RACE and
 * produce wrong events: issue them on one stream, or order them with events.
 * Asynchronous on cuda_stream like mdsm_detect; runs the statistics + thresholding kernels as two launches (the
 * "detect_two_pass" form), so any series length is accepted.  Errors: MDSM_EINVAL (null pointers, dtype other than
 * MDSM_F32 / MDSM_U8, sizes < 1, nsamps_out > nsamps, NaN threshold, ndms or nbeams > 65535, too many series),
 * MDSM_ECUDA (the address query or a launch failed). */
#define MDSM_DETECT_NOALLOC_MAX_SERIES 32768
int mdsm_detect_noalloc(const void *d_series, int dtype, int nbeams, int ndms, int64_t nsamps, int64_t nsamps_out,
                        double snr_thresh, mdsm_event *d_events, int64_t max_events, unsigned long long *d_count,
                        void *cuda_stream);

/* Post-processing of the dedispersed series between mdsm_dedisperse and mdsm_detect (section
 * 2.2.3: "optional post-processing").  fp32 series only, layout of d_out ([nbeams][ndms][nsamps], the
 * first nsamps_out samples of a row valid); device pointers, asynchronous on cuda_stream, no allocation.
 *
 * mdsm_median_filter: Eq. 2 with operation = median, y[m] = median{x[i], i in w}, w = `window`
 *   (odd, <= 33) samples centred on m, clipped to the valid samples at the two ends; an even number of remaining
 *   points gives the mean of the two middle ones.  d_filtered must be a different buffer of the same layout; only
 *   t < nsamps_out of the rows [beam0, beam0+nb) is written.
 * mdsm_detrend: per series, subtract the least-squares line over t = 0..nsamps_out-1 and divide by the population
 *   standard deviation of the residual, in place; a series with zero residual variance becomes
 *   zeros.  d_params (may be NULL) receives [nbeams][ndms][3] = mean, slope, standard deviation (fp64, device).
 * Errors: MDSM_EINVAL for a bad beam range / window / null or aliased buffers. */
int mdsm_median_filter(mdsm_plan *plan, const float *d_series, float *d_filtered, int beam0, int nb, int window,
                       void *cuda_stream);
int mdsm_detrend(mdsm_plan *plan, float *d_series, int beam0, int nb, double *d_params, void *cuda_stream);

/* Power calculation, the first GPU stage of the paper's pipeline: d_power[i] = re^2 + im^2 of the
 * 16-bit complex channelised voltages d_volt[i] = (re, im), any layout (the call is element-wise, so
 * [beam][chan][time][2] in gives [beam][chan][time] out).  The sum is exact in integers and rounded once to float.
 * Device pointers, 16-byte aligned, caller-owned; asynchronous on cuda_stream; needs no plan.  MDSM_EINVAL for
 * null / misaligned buffers or n < 0. */
int mdsm_power_i16(const int16_t *d_volt, float *d_power, int64_t n, void *cuda_stream);

/* mu-law quantiser of a (non-negative) float power series to 8 bits (Eq. 5):
 *   Xmax = max x;  code = floor(255 * log(1 + mu x / Xmax) / log(1 + mu) + 0.5)   (fp64; x <= 0, NaN or Xmax == 0 -> 0).
 * d_x [n] floats, d_code [n] bytes, both 16-byte aligned device buffers; d_xmax: one device float that receives Xmax
 * (the decoder needs it).  Asynchronous on cuda_stream; needs no plan.  MDSM_EINVAL for null / misaligned buffers,
 * n < 0 or mu <= 0. */
int mdsm_mulaw_u8(const float *d_x, uint8_t *d_code, int64_t n, double mu, float *d_xmax, void *cuda_stream);

/* mu-law quantiser of the 16-bit complex channelised voltages to 2 x 4 bits per sample ("16-bit complex
 * values are quantized to 4-bits with two complex components packed into one byte"; Eq. 5; Fig. 5b; reading G-ii):
 *   Xmax = max |component| of the buffer;  code(v) = sign(v) * floor(7 * log(1 + mu |v| / Xmax) / log(1 + mu) + 0.5) in [-7, 7];
 *   packed[i] = (code(re_i) & 15) | (code(im_i) & 15) << 4   (two's-complement nibbles; Xmax = 0 -> zeros).
 * d_volt [n][2] int16 (re, im), d_packed [n] bytes, both 16-byte aligned device buffers; d_xmax_thr: nine device int32 that
 * receive Xmax and the law as integer thresholds (thr[k] = smallest |v| with code >= k + 1, k < 7; the decoder's table).
 * Asynchronous on cuda_stream; needs no plan.  MDSM_EINVAL for null / misaligned buffers, n < 0 or mu <= 0. */
int mdsm_mulaw_c4(const int16_t *d_volt, uint8_t *d_packed, int64_t n, double mu, int32_t *d_xmax_thr, void *cuda_stream);

/* Host candidate stage (north_star: "clustering and the analytic DM-SNR candidate
 * filter stay on the host").  Both calls take HOST pointers, run on the calling thread and need neither a plan nor a GPU.
 *
 * mdsm_cluster_events: density clustering of detections in (time [samples], DM [pc cm^-3], SNR), beam by beam
 *   (one list per beam).  q is a neighbour of p when |dt| <= eps_t, |dDM| <= eps_dm and |dSNR| <= eps_snr
 *   ("a different value to each dimension (T_t, SNR_t, DM_t)"); a core point has >= min_pts neighbours,
 *   itself included.  exact = 0: FDBSCAN: only the representative border points of a core point's
 *   neighbourhood (per dimension and direction the farthest neighbour of this cluster) are expanded; exact = 1: DBSCAN.
 *   h_labels[i] receives the cluster id of event i (0 .. *h_nclusters - 1, numbered beam by beam in order of discovery)
 *   or -1 (noise); *h_nqueries (may be NULL) the number of neighbourhood queries made.  DM of an event =
 *   dm_low + dm_idx * dm_step.
 * mdsm_classify_clusters: the eight steps of PAPER.md:144-156 per cluster: DM-SNR signature (strongest detection per DM),
 *   k_smooth-element moving average (odd), the DM with the most detections (DM < 1.0 => broadband RFI), the pulse width
 *   at that DM, normalisation, the model curve of Eq. 3 with zeta of Eq. 4 (bw_mhz = bandwidth, nu_ghz = centre
 *   frequency), the RMSE between the two, RMSE > rmse_max => RFI.
 *   h_results [nclusters][5] = class (0 candidate, 1 RFI: DM < 1, 2 RFI: curve mismatch, -1 empty cluster id),
 *   dm_idx of the peak, its SNR, width in ms, RMSE.
 * MDSM_EINVAL for null pointers / non-positive eps / even k_smooth / labels out of range. */
int mdsm_cluster_events(const mdsm_event *h_events, int64_t n, double dm_low, double dm_step, double eps_t,
                        double eps_dm, double eps_snr, int min_pts, int exact, int32_t *h_labels,
                        int64_t *h_nclusters, int64_t *h_nqueries);
int mdsm_classify_clusters(const mdsm_event *h_events, const int32_t *h_labels, int64_t n, int64_t nclusters,
                           double dm_low, double dm_step, double tsamp, double bw_mhz, double nu_ghz, int k_smooth,
                           double rmse_max, double *h_results);

/* The whole chain from HOST buffers (per-beam threads copy their input to the GPU;
 * north_star item 4: beam groups on separate CUDA streams with overlapped host-to-device copies).
 * h_in [nbeams][nchans][nsamps] (pinned memory overlaps best); the clipped data is NOT copied back.
 * clip is skipped when window == 0.  Events are copied to h_events (up to max_events) and
 * *h_count receives the total found.  Device buffers are plan-owned and allocated on first use.
 * Synchronises before returning.  Returns MDSM_EOVERFLOW if *h_count > max_events. */
int mdsm_pipeline_host(mdsm_plan *plan, const void *h_in, int dtype,
                       int window, double k_chan, double k_spec, double snr_thresh,
                       mdsm_event *h_events, int64_t max_events, uint64_t *h_count,
                       int nstreams);

/* Register-only add-issue microbenchmark on all SMs of the current device (the measured
 * denominator of the dedispersion roofline).
 * kind 0: FADD, 1: FADD2 (add.f32x2, two results per lane-instruction), 2: integer add.
 * *adds_per_s receives 32-bit add results per second.  Synchronises. */
int mdsm_measure_add_peak(int kind, double *adds_per_s);

#ifdef __cplusplus
}
#endif
#endif /* MDSM_H */
