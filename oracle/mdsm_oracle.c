/*
 * mdsm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU restatement of the three stages of the
 * Medicina BEST-2 transient pipeline hot path (arXiv:1307.5700), written from
 * the paper text and the readings listed in
 * DESIGN.md section 3.  It shares no code, header, table or constant generator
 * with the CUDA library (paper_1307_5700_b200/csrc).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * Everything is the definition written out, in the paper's order:
 *   orc_delay_table     Eq. 1           -> integer delays
 *   orc_dedisperse_*    brute force        -> out[b][d][t]
 *   orc_rfi_clip_*      channel + spectrum thresholding
 *   orc_detect_*        n-sigma thresholding
 *
 * fp64 everywhere a floating-point decision is taken; every fp64 operation is
 * one IEEE op in the order written (build with -ffp-contract=off, no
 * -ffast-math).  No blocking, no fusion, no reordering beyond the two loop
 * orders (naive: b,d,t,c; rows: b,d,c,t) that SURVEY.md section 8(c) asks for,
 * both of which add the channels of one output in ascending c.
 *
 * Parity pins: see tests/test_oracle_*.py (closed-form delay values, DM=0 row,
 * impulse recovery, linearity, brute force vs numpy, clip invariants,
 * detection vs brute-force filter).  The CHOICE of per-buffer mean/rms clip
 * thresholds (reading B-i) has no worked numbers in the paper: "parity
 * unpinned" against the paper for orc_rfi_clip_* thresholds; pinned only by
 * invariants.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ A ---- */
/* Eq. 1: dt = 4.15e6 ms * (f1^-2 - f2^-2) * DM, f in MHz.
 * north_star fixes the constant to 4.148808e3 s MHz^2 pc^-1 cm^3, reference
 * frequency f_top (channel 0, the highest), f_c = f_top + c*foff (channel
 * centre), and round() = floor(x + 0.5) in fp64 (readings A1, A2). */
void orc_delay_table(int nchans, double f_top, double foff, double tsamp,
                     double dm_low, double dm_step, int ndms, int32_t *delay)
{
    for (int d = 0; d < ndms; ++d) {
        double dm = dm_low + (double)d * dm_step;
        for (int c = 0; c < nchans; ++c) {
            double f = f_top + (double)c * foff;
            double x = 4.148808e3 * dm * (1.0 / (f * f) - 1.0 / (f_top * f_top)) / tsamp;
            delay[(size_t)d * nchans + c] = (int32_t)floor(x + 0.5);
        }
    }
}

/* ------------------------------------------------------------------ C ---- */
/* Brute-force incoherent dedispersion (north_star):
 *   out[b][d][t] = sum_c in[b][c][t + delay(d,c)],  t in [0, nsamps_out)
 * in  : [nbeams][nchans][nsamps], time fastest
 * out : [nbeams][ndms][nsamps_out] fp64 sums (ascending c)
 * absum (may be NULL): same loop over |in|  (for the fp32 tolerance). */
void orc_dedisperse_f32_naive(const float *in, int nbeams, int nchans, int64_t nsamps,
                              const int32_t *delay, int ndms, int64_t nsamps_out,
                              double *out, double *absum)
{
    for (int b = 0; b < nbeams; ++b)
        for (int d = 0; d < ndms; ++d)
            for (int64_t t = 0; t < nsamps_out; ++t) {
                double s = 0.0, a = 0.0;
                for (int c = 0; c < nchans; ++c) {
                    double v = (double)in[((size_t)b * nchans + c) * nsamps + t + delay[(size_t)d * nchans + c]];
                    s += v;
                    a += fabs(v);
                }
                size_t o = ((size_t)b * ndms + d) * nsamps_out + t;
                out[o] = s;
                if (absum) absum[o] = a;
            }
}

void orc_dedisperse_f32_rows(const float *in, int nbeams, int nchans, int64_t nsamps,
                             const int32_t *delay, int ndms, int64_t nsamps_out,
                             double *out, double *absum)
{
    int64_t nrows = (int64_t)nbeams * ndms;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int b = (int)(r / ndms), d = (int)(r % ndms);
        double *o = out + (size_t)r * nsamps_out;
        double *a = absum ? absum + (size_t)r * nsamps_out : NULL;
        for (int64_t t = 0; t < nsamps_out; ++t) o[t] = 0.0;
        if (a) for (int64_t t = 0; t < nsamps_out; ++t) a[t] = 0.0;
        for (int c = 0; c < nchans; ++c) {
            const float *x = in + ((size_t)b * nchans + c) * nsamps + delay[(size_t)d * nchans + c];
            for (int64_t t = 0; t < nsamps_out; ++t) o[t] += (double)x[t];
            if (a) for (int64_t t = 0; t < nsamps_out; ++t) a[t] += fabs((double)x[t]);
        }
    }
}

/* Selected rows only: rows[i] = b*ndms + d.  out/absum: [nrows_sel][nsamps_out].
 * Used for sampled parity at sizes where the full output is too slow. */
void orc_dedisperse_f32_sel(const float *in, int nbeams, int nchans, int64_t nsamps,
                            const int32_t *delay, int ndms, int64_t nsamps_out,
                            const int64_t *rows, int64_t nrows_sel, double *out, double *absum)
{
    (void)nbeams;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < nrows_sel; ++i) {
        int b = (int)(rows[i] / ndms), d = (int)(rows[i] % ndms);
        double *o = out + (size_t)i * nsamps_out;
        double *a = absum ? absum + (size_t)i * nsamps_out : NULL;
        for (int64_t t = 0; t < nsamps_out; ++t) o[t] = 0.0;
        if (a) for (int64_t t = 0; t < nsamps_out; ++t) a[t] = 0.0;
        for (int c = 0; c < nchans; ++c) {
            const float *x = in + ((size_t)b * nchans + c) * nsamps + delay[(size_t)d * nchans + c];
            for (int64_t t = 0; t < nsamps_out; ++t) o[t] += (double)x[t];
            if (a) for (int64_t t = 0; t < nsamps_out; ++t) a[t] += fabs((double)x[t]);
        }
    }
}

/* uint8 in, uint32 accumulate: exact, order-free (max 4096*255 << 2^32). */
void orc_dedisperse_u8_naive(const uint8_t *in, int nbeams, int nchans, int64_t nsamps,
                             const int32_t *delay, int ndms, int64_t nsamps_out, uint32_t *out)
{
    for (int b = 0; b < nbeams; ++b)
        for (int d = 0; d < ndms; ++d)
            for (int64_t t = 0; t < nsamps_out; ++t) {
                uint32_t s = 0;
                for (int c = 0; c < nchans; ++c)
                    s += in[((size_t)b * nchans + c) * nsamps + t + delay[(size_t)d * nchans + c]];
                out[((size_t)b * ndms + d) * nsamps_out + t] = s;
            }
}

void orc_dedisperse_u8_rows(const uint8_t *in, int nbeams, int nchans, int64_t nsamps,
                            const int32_t *delay, int ndms, int64_t nsamps_out, uint32_t *out)
{
    int64_t nrows = (int64_t)nbeams * ndms;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < nrows; ++r) {
        int b = (int)(r / ndms), d = (int)(r % ndms);
        uint32_t *o = out + (size_t)r * nsamps_out;
        for (int64_t t = 0; t < nsamps_out; ++t) o[t] = 0;
        for (int c = 0; c < nchans; ++c) {
            const uint8_t *x = in + ((size_t)b * nchans + c) * nsamps + delay[(size_t)d * nchans + c];
            for (int64_t t = 0; t < nsamps_out; ++t) o[t] += x[t];
        }
    }
}

void orc_dedisperse_u8_sel(const uint8_t *in, int nbeams, int nchans, int64_t nsamps,
                           const int32_t *delay, int ndms, int64_t nsamps_out,
                           const int64_t *rows, int64_t nrows_sel, uint32_t *out)
{
    (void)nbeams;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < nrows_sel; ++i) {
        int b = (int)(rows[i] / ndms), d = (int)(rows[i] % ndms);
        uint32_t *o = out + (size_t)i * nsamps_out;
        for (int64_t t = 0; t < nsamps_out; ++t) o[t] = 0;
        for (int c = 0; c < nchans; ++c) {
            const uint8_t *x = in + ((size_t)b * nchans + c) * nsamps + delay[(size_t)d * nchans + c];
            for (int64_t t = 0; t < nsamps_out; ++t) o[t] += x[t];
        }
    }
}

/* ------------------------------------------------------------------ B ---- */
/* RFI clip (PAPER.md:79 channel thresholding, :81 spectrum thresholding), with
 * north_star's "k sigma of their mean/rms" thresholds in place of the paper's
 * polynomial-fit thresholds (readings B-i .. B-viii in DESIGN.md).
 * Per beam, on all nsamps input samples, one-sided, in this order:
 *  B1 per channel: S=sum x, Q=sum x^2; mean=S/N; var=Q/N-mean*mean (clamp 0);
 *     sig=sqrt(var); repl = u8: (S+N/2)/N (integer)  f32: (float)mean
 *  B2 per chunk j of W samples: C=sum; thr = W*mean + (k_chan*sig)*sqrt(W);
 *     raw=(C>thr); mask[j]=raw[j-1]|raw[j]|raw[j+1]; flagged chunks := repl
 *  B3 per time t on the modified data: s_t=sum_c x; M1=sum s, M2=sum s^2;
 *     mean_s=M1/N; var_s=M2/N-mean_s^2 (clamp 0); sig_s=sqrt;
 *     spec_mask[t]=(s_t > mean_s + k_spec*sig_s); flagged spectra := repl_c
 * Optional debug outputs (may be NULL): chan_mean/chan_sig [nb][nchans],
 * chan_thr [nb][nchans] (threshold on the chunk SUM), spec_thr [nb] and
 * spec_sum [nb][nsamps] (sums seen by B3), repl (as double) [nb][nchans].
 * Returns 0, or -1 on bad arguments (N % W != 0 -> reading B-viii). */
#define ORC_CLIP_BODY(T, IS_INT)                                                              \
    if (window < 1 || nsamps % window != 0) return -1;                                        \
    int64_t nchunk = nsamps / window;                                                         \
    int rc = 0;                                                                               \
    _Pragma("omp parallel for schedule(dynamic, 1)")                                          \
    for (int b = 0; b < nbeams; ++b) {                                                        \
        T *xb = in + (size_t)b * nchans * nsamps;                                             \
        T *repl = (T *)malloc(sizeof(T) * (size_t)nchans);                                    \
        uint8_t *raw = (uint8_t *)malloc((size_t)nchunk);                                     \
        double *st = (double *)malloc(sizeof(double) * (size_t)nsamps);                       \
        uint64_t *sti = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)nsamps);                \
        if (!repl || !raw || !st || !sti) { rc = -2; free(repl); free(raw); free(st); free(sti); continue; } \
        double dN = (double)nsamps;                                                           \
        for (int c = 0; c < nchans; ++c) {                                                    \
            T *x = xb + (size_t)c * nsamps;                                                   \
            /* B1 */                                                                          \
            double mean, var;                                                                 \
            if (IS_INT) {                                                                     \
                uint64_t S = 0, Q = 0;                                                        \
                for (int64_t t = 0; t < nsamps; ++t) { uint64_t v = (uint64_t)x[t]; S += v; Q += v * v; } \
                mean = (double)S / dN;                                                        \
                var = (double)Q / dN - mean * mean;                                           \
                repl[c] = (T)((S + (uint64_t)(nsamps / 2)) / (uint64_t)nsamps);               \
            } else {                                                                          \
                double S = 0.0, Q = 0.0;                                                      \
                for (int64_t t = 0; t < nsamps; ++t) { double v = (double)x[t]; S += v; Q += v * v; } \
                mean = S / dN;                                                                \
                var = Q / dN - mean * mean;                                                   \
                repl[c] = (T)mean;                                                            \
            }                                                                                 \
            if (var < 0.0) var = 0.0;                                                         \
            double sig = sqrt(var);                                                           \
            double thr = (double)window * mean + (k_chan * sig) * sqrt((double)window);       \
            if (chan_mean) chan_mean[(size_t)b * nchans + c] = mean;                          \
            if (chan_sig) chan_sig[(size_t)b * nchans + c] = sig;                             \
            if (chan_thr) chan_thr[(size_t)b * nchans + c] = thr;                             \
            if (repl_out) repl_out[(size_t)b * nchans + c] = (double)repl[c];                 \
            /* B2 */                                                                          \
            for (int64_t j = 0; j < nchunk; ++j) {                                            \
                double C;                                                                     \
                if (IS_INT) {                                                                 \
                    uint64_t Ci = 0;                                                          \
                    for (int64_t t = j * window; t < (j + 1) * window; ++t) Ci += (uint64_t)x[t]; \
                    C = (double)Ci;                                                           \
                } else {                                                                      \
                    C = 0.0;                                                                  \
                    for (int64_t t = j * window; t < (j + 1) * window; ++t) C += (double)x[t]; \
                }                                                                             \
                raw[j] = (C > thr) ? 1 : 0;                                                   \
            }                                                                                 \
            for (int64_t j = 0; j < nchunk; ++j) {                                            \
                uint8_t m = raw[j];                                                           \
                if (j > 0) m |= raw[j - 1];                                                   \
                if (j + 1 < nchunk) m |= raw[j + 1];                                          \
                if (chan_mask) chan_mask[((size_t)b * nchans + c) * nchunk + j] = m;          \
                if (m) for (int64_t t = j * window; t < (j + 1) * window; ++t) x[t] = repl[c]; \
            }                                                                                 \
        }                                                                                     \
        /* B3 */                                                                              \
        double mean_s, var_s;                                                                 \
        if (IS_INT) {                                                                         \
            uint64_t M1 = 0, M2 = 0;                                                          \
            for (int64_t t = 0; t < nsamps; ++t) {                                            \
                uint64_t s = 0;                                                               \
                for (int c = 0; c < nchans; ++c) s += (uint64_t)xb[(size_t)c * nsamps + t];   \
                sti[t] = s; st[t] = (double)s; M1 += s; M2 += s * s;                          \
            }                                                                                 \
            mean_s = (double)M1 / dN;                                                         \
            var_s = (double)M2 / dN - mean_s * mean_s;                                        \
        } else {                                                                              \
            double M1 = 0.0, M2 = 0.0;                                                        \
            for (int64_t t = 0; t < nsamps; ++t) {                                            \
                double s = 0.0;                                                               \
                for (int c = 0; c < nchans; ++c) s += (double)xb[(size_t)c * nsamps + t];     \
                st[t] = s; M1 += s; M2 += s * s;                                              \
            }                                                                                 \
            mean_s = M1 / dN;                                                                 \
            var_s = M2 / dN - mean_s * mean_s;                                                \
        }                                                                                     \
        if (var_s < 0.0) var_s = 0.0;                                                         \
        double sig_s = sqrt(var_s);                                                           \
        double thr_s = mean_s + k_spec * sig_s;                                               \
        if (spec_thr) { spec_thr[3 * b] = thr_s; spec_thr[3 * b + 1] = mean_s; spec_thr[3 * b + 2] = sig_s; } \
        for (int64_t t = 0; t < nsamps; ++t) {                                                \
            uint8_t m = (st[t] > thr_s) ? 1 : 0;                                              \
            if (spec_sum) spec_sum[(size_t)b * nsamps + t] = st[t];                           \
            if (spec_mask) spec_mask[(size_t)b * nsamps + t] = m;                             \
            if (m) for (int c = 0; c < nchans; ++c) xb[(size_t)c * nsamps + t] = repl[c];     \
        }                                                                                     \
        free(repl); free(raw); free(st); free(sti);                                           \
    }                                                                                         \
    return rc;

int orc_rfi_clip_f32(float *in, int nbeams, int nchans, int64_t nsamps, int window,
                     double k_chan, double k_spec, uint8_t *chan_mask, uint8_t *spec_mask,
                     double *chan_mean, double *chan_sig, double *chan_thr, double *repl_out,
                     double *spec_thr, double *spec_sum)
{
    ORC_CLIP_BODY(float, 0)
}

int orc_rfi_clip_u8(uint8_t *in, int nbeams, int nchans, int64_t nsamps, int window,
                    double k_chan, double k_spec, uint8_t *chan_mask, uint8_t *spec_mask,
                    double *chan_mean, double *chan_sig, double *chan_thr, double *repl_out,
                    double *spec_thr, double *spec_sum)
{
    ORC_CLIP_BODY(uint8_t, 1)
}

/* ------------------------------------------------------------------ D ---- */
/* n-sigma thresholding of each dedispersed series, with the
 * series normalised by its own mean and population rms (readings
 * D-i .. D-vii).  Per (b,d) over t in [0, n), n = nsamps_out:
 *   S=sum out, Q=sum out^2; mean=S/n; var=Q/n-mean*mean (clamp 0); rms=sqrt
 *   rms == 0 -> no events;  snr=((double)out[t]-mean)/rms;  event iff snr > thr
 * series : [nseries][stride], first n of each row valid.
 * events are written in (series, t) order as 4 parallel arrays; returns the
 * total count (which may exceed max_events; only the first max_events are
 * stored).  series index = b*ndms + d; the caller splits it.
 * stats (may be NULL): [nseries][2] = mean, rms. */
typedef struct { int32_t beam, dm_idx, t; float snr; } orc_event;

#define ORC_DETECT_BODY(T, IS_INT)                                                            \
    int64_t count = 0;                                                                        \
    double dn = (double)n;                                                                    \
    for (int64_t r = 0; r < nseries; ++r) {                                                   \
        const T *x = series + (size_t)r * stride;                                             \
        double mean, var;                                                                     \
        if (IS_INT) {                                                                         \
            uint64_t S = 0, Q = 0;                                                            \
            for (int64_t t = 0; t < n; ++t) { uint64_t v = (uint64_t)x[t]; S += v; Q += v * v; } \
            mean = (double)S / dn;                                                            \
            var = (double)Q / dn - mean * mean;                                               \
        } else {                                                                              \
            double S = 0.0, Q = 0.0;                                                          \
            for (int64_t t = 0; t < n; ++t) { double v = (double)x[t]; S += v; Q += v * v; }  \
            mean = S / dn;                                                                    \
            var = Q / dn - mean * mean;                                                       \
        }                                                                                     \
        if (var < 0.0) var = 0.0;                                                             \
        double rms = sqrt(var);                                                               \
        if (stats) { stats[2 * r] = mean; stats[2 * r + 1] = rms; }                           \
        if (rms == 0.0) continue;                                                             \
        for (int64_t t = 0; t < n; ++t) {                                                     \
            double snr = ((double)x[t] - mean) / rms;                                         \
            if (snr > snr_thresh) {                                                           \
                if (count < max_events) {                                                     \
                    events[count].beam = (int32_t)(r / ndms);                                 \
                    events[count].dm_idx = (int32_t)(r % ndms);                               \
                    events[count].t = (int32_t)t;                                             \
                    events[count].snr = (float)snr;                                           \
                }                                                                             \
                ++count;                                                                      \
            }                                                                                 \
        }                                                                                     \
    }                                                                                         \
    return count;

int64_t orc_detect_f32(const float *series, int64_t nseries, int ndms, int64_t stride, int64_t n,
                       double snr_thresh, orc_event *events, int64_t max_events, double *stats)
{
    ORC_DETECT_BODY(float, 0)
}

int64_t orc_detect_f64(const double *series, int64_t nseries, int ndms, int64_t stride, int64_t n,
                       double snr_thresh, orc_event *events, int64_t max_events, double *stats)
{
    ORC_DETECT_BODY(double, 0)
}

int64_t orc_detect_u32(const uint32_t *series, int64_t nseries, int ndms, int64_t stride, int64_t n,
                       double snr_thresh, orc_event *events, int64_t max_events, double *stats)
{
    ORC_DETECT_BODY(uint32_t, 1)
}

/* ------------------------------------------------------------------------------------------------
 * Post-processing of the dedispersed series (section 2.2.3) -- SURVEY 8(f) NEXT-1.
 *
 * orc_median_filter_f32: Eq. 2 with operation = median: y[m] = median{ x[i], i in w }, w = the
 *   neighbourhood of `window` (odd) points centred on m.  Readings (E-i): the neighbourhood is
 *   clipped to the valid samples [0, n) at the two ends (the paper's kernel loads "overlapping values at the edges"
 *   but does not say what stands in beyond the series); with an even number of points left, the median is the mean
 *   of the two middle ones.  Pinned by brute force against numpy.median and by isolated-outlier / monotone-series
 *   invariants (tests/test_oracle_postprocess.py).
 * orc_detrend_f32: best-fit line by linear regression over t = 0..n-1 (pass 1), subtract it and take the standard
 *   deviation of the residual (pass 2), divide (pass 3) -- PAPER.md:110.  Population standard deviation (1/n);
 *   a series with zero residual variance becomes all zeros (reading E-ii).  fp64 throughout, result cast to float.
 *   Pinned against the closed-form least-squares solution (numpy.polyfit) and exact lines.
 * ------------------------------------------------------------------------------------------------ */
void orc_median_filter_f32(const float *in, int64_t nseries, int64_t stride, int64_t n, int window, float *out)
{
    const int h = window / 2;
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < nseries; ++s) {
        const float *x = in + s * stride;
        float *y = out + s * stride;
        float buf[1024];
        for (int64_t m = 0; m < n; ++m) {
            int64_t lo = m - h, hi = m + h;
            if (lo < 0) lo = 0;
            if (hi > n - 1) hi = n - 1;
            int cnt = 0;
            for (int64_t i = lo; i <= hi; ++i) {          /* insertion sort of the neighbourhood */
                float v = x[i];
                int k = cnt++;
                while (k > 0 && buf[k - 1] > v) { buf[k] = buf[k - 1]; --k; }
                buf[k] = v;
            }
            if (cnt & 1) y[m] = buf[cnt / 2];
            else y[m] = (float)(((double)buf[cnt / 2 - 1] + (double)buf[cnt / 2]) / 2.0);
        }
    }
}

/* params[s] = (mean, slope, std of the residual) */
void orc_detrend_f32(const float *in, int64_t nseries, int64_t stride, int64_t n, float *out, double *params)
{
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < nseries; ++s) {
        const float *x = in + s * stride;
        float *y = out + s * stride;
        const double tbar = ((double)n - 1.0) / 2.0;
        double sy = 0.0, sty = 0.0, stt = 0.0;
        for (int64_t t = 0; t < n; ++t) {                /* pass 1: regression parameters */
            const double dt = (double)t - tbar;
            sy += (double)x[t];
            sty += dt * (double)x[t];
            stt += dt * dt;
        }
        const double mean = sy / (double)n;
        const double slope = stt > 0.0 ? sty / stt : 0.0;
        double sr = 0.0;
        for (int64_t t = 0; t < n; ++t) {                /* pass 2: residual variance */
            const double r = (double)x[t] - (mean + slope * ((double)t - tbar));
            sr += r * r;
        }
        const double sd = sqrt(sr / (double)n);
        for (int64_t t = 0; t < n; ++t) {                /* pass 3: normalise */
            const double r = (double)x[t] - (mean + slope * ((double)t - tbar));
            y[t] = sd > 0.0 ? (float)(r / sd) : 0.0f;
        }
        if (params) { params[3 * s] = mean; params[3 * s + 1] = slope; params[3 * s + 2] = sd; }
    }
}

/* ------------------------------------------------------------------------------------------------
 * Power calculation (the first GPU stage, "power calculation", on the 16-bit complex channelised
 * voltages of the beamformer) -- SURVEY 8(f) NEXT-4.
 *   power[i] = re[i]^2 + im[i]^2, voltages interleaved (re, im) int16; the sum is an exact integer < 2^31 + 1, the
 *   result is that integer rounded to nearest float.  Pinned by hand-computed values (tests/test_oracle_power.py).
 * ------------------------------------------------------------------------------------------------ */
void orc_power_i16(const int16_t *volt, int64_t n, float *power)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const int64_t re = volt[2 * i], im = volt[2 * i + 1];
        power[i] = (float)(double)(re * re + im * im);      /* int64 -> double exact, double -> float round to nearest */
    }
}

/* ------------------------------------------------------------------------------------------------
 * mu-law quantiser of a channelised power series, 32-bit float -> 8 bits (Eq. 5) -- SURVEY 8(f)
 * NEXT-4.   y = Xmax * log(1 + mu |x| / Xmax) / log(1 + mu) * sign(x),  Xmax = the maximum of the series.
 * Readings (G-i): the paper does not say how y becomes 8 bits; power is non-negative, so the
 * code is unsigned, code = floor(255 * y / Xmax + 0.5); negative or NaN input and an all-zero series give code 0.
 * fp64 with log1p.  Pinned by closed-form values (x = 0, x = Xmax, the mu -> 0 linear limit, monotonicity, the
 * textbook mid-point x/Xmax = (sqrt(1+mu) - 1)/mu -> y/Xmax = 1/2).  xmax_out (may be NULL) receives Xmax.
 * ------------------------------------------------------------------------------------------------ */
void orc_mulaw_u8(const float *x, int64_t n, double mu, uint8_t *code, float *xmax_out)
{
    float xmax = 0.0f;
    for (int64_t i = 0; i < n; ++i)
        if (x[i] > xmax) xmax = x[i];
    if (xmax_out) *xmax_out = xmax;
    const double den = log1p(mu);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double v = 0.0;
        if (xmax > 0.0f && x[i] > 0.0f) v = 255.0 * (log1p(mu * ((double)x[i] / (double)xmax)) / den);
        code[i] = (uint8_t)floor(v + 0.5);
    }
}
