/*
 * mdsm_oracle_next.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (second file of the oracle, same rules as mdsm_oracle.c).
 *
 * Plain CPU restatements of the SURVEY.md section 8(f) "NEXT" rows, written from /root/reference/PAPER.md and the
 * readings of DESIGN.md section 3 (ids H-*, K-*, G-ii, C-ii):
 *   orc_bandpass_clip_f32   the paper's own RFI stage: averaged bandpass, masking + interpolation of RFI channels,
 *                           p-th order least-squares fit, RMSE channel thresholds, mean/std spectrum threshold,
 *                           fitted-value replacement, bandpass subtraction          (Fig. 3)
 *   orc_dbscan / orc_fdbscan   density clustering of (time, DM, SNR) detections
 *   orc_classify_cluster    the 8-step DM-SNR-curve classifier with Eqs. 3 and 4
 *   orc_mulaw_c4            mu-law quantiser 2 x 16 bit -> 2 x 4 bit in one byte      (Fig. 5b)
 *   orc_dedisperse_u16_rows brute-force dedispersion of 16-bit (and, unpacked by the caller, 4-bit) input
 * Shares no code with the CUDA library.  fp64 wherever a decision is taken, one IEEE operation per written operation
 * (-ffp-contract=off).  Pins: tests/test_oracle_next.py.
 * "Parity unpinned against the paper" for the bandpass stage's thresholds (the paper prints no worked numbers: the
 * way RFI channels are recognised before the fit and the meaning of "mean and standard deviation" are readings H-ii,
 * H-vi); its arithmetic is pinned by exact recovery of a polynomial bandpass, numpy.polyfit and invariants.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ================================================================== bandpass stage (NEXT-2) ==== */
static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

static double median_of(const double *v, int n, double *tmp)
{
    memcpy(tmp, v, sizeof(double) * (size_t)n);
    qsort(tmp, (size_t)n, sizeof(double), cmp_double);
    return (n & 1) ? tmp[n / 2] : 0.5 * (tmp[n / 2 - 1] + tmp[n / 2]);
}

/* Least-squares polynomial of order p through (u_c, y_c), u_c = 2c/(n-1) - 1 (u = 0 when n = 1): normal equations
 * in the monomial basis, Gaussian elimination with partial pivoting, all fp64.  coef[k] multiplies u^k.
 * Returns 0, or -1 when the system is singular (p >= n). */
int orc_polyfit_u(const double *y, int n, int p, double *coef)
{
    enum { PMAX = 16 };
    if (p < 0 || p >= PMAX || n < 1) return -1;
    double A[PMAX][PMAX + 1];
    for (int i = 0; i <= p; ++i)
        for (int j = 0; j <= p + 1; ++j) A[i][j] = 0.0;
    for (int c = 0; c < n; ++c) {
        const double u = n > 1 ? 2.0 * (double)c / (double)(n - 1) - 1.0 : 0.0;
        double pw[2 * PMAX];
        pw[0] = 1.0;
        for (int k = 1; k <= 2 * p; ++k) pw[k] = pw[k - 1] * u;
        for (int i = 0; i <= p; ++i) {
            for (int j = 0; j <= p; ++j) A[i][j] += pw[i + j];
            A[i][p + 1] += pw[i] * y[c];
        }
    }
    for (int i = 0; i <= p; ++i) {
        int piv = i;
        for (int r = i + 1; r <= p; ++r)
            if (fabs(A[r][i]) > fabs(A[piv][i])) piv = r;
        if (A[piv][i] == 0.0) return -1;
        if (piv != i)
            for (int j = 0; j <= p + 1; ++j) { double t = A[i][j]; A[i][j] = A[piv][j]; A[piv][j] = t; }
        for (int r = i + 1; r <= p; ++r) {
            const double f = A[r][i] / A[i][i];
            for (int j = i; j <= p + 1; ++j) A[r][j] -= f * A[i][j];
        }
    }
    for (int i = p; i >= 0; --i) {
        double s = A[i][p + 1];
        for (int j = i + 1; j <= p; ++j) s -= A[i][j] * coef[j];
        coef[i] = s / A[i][i];
    }
    return 0;
}

/* The paper's RFI stage for one buffer of float power data in[b][c][t], in place, per beam:
 *  H1  bp[c]   = (sum_t x[c][t]) / N                                   "averaged bandpass"
 *  H2  med = median_c bp, mad = median_c |bp - med|;  rfi[c] = (bp[c] - med) > k_mask * 1.4826 * mad  (reading H-ii:
 *      the paper does not say how "channels containing high power RFI" are recognised);  bpi[c] = bp[c] unless
 *      rfi[c], then the mean of the nearest un-masked channel on either side (the one that exists at a band edge)
 *      "replacing their values with the mean of the neighboring channels, thus interpolating the bandpass"
 *  H3  fit[c]  = order-p least-squares polynomial through bpi          (Fig. 3)
 *  H4  rmse    = sqrt(mean_c (fit - bpi)^2);  mean_bp, std_bp = mean and population std of bpi over channels
 *      "RMSE ... used as a thresholding factor for the channel thresholding stage, whilst the mean and standard
 *      deviation are used for the spectrum thresholding stage" (reading H-vi: of the bandpass)
 *  H5  channel thresholding: chunks of W samples; raw = (chunk mean > fit[c] + k_chan * rmse); a
 *      flagged chunk and its two time neighbours are replaced by (float)fit[c] "the channel's fitted bandpass value"
 *  H6  spectrum thresholding on the data as modified by H5: m_t = (sum_c x[c][t]) / nchans;
 *      flag when m_t > mean_bp + k_spec * std_bp; flagged spectra := (float)fit[c] for every c
 *  H7  subtract != 0: x[c][t] -= (float)fit[c] for every sample ("subtracted from all the spectra")
 * Outputs (any may be NULL): chan_mask [nb][nchans][N/W], spec_mask [nb][N], fit/bpi [nb][nchans],
 * stats [nb][4] = rmse, mean_bp, std_bp, number of masked channels.  Returns 0, -1 on bad arguments. */
int orc_bandpass_clip_f32(float *in, int nbeams, int nchans, int64_t nsamps, int window, int order, double k_mask,
                          double k_chan, double k_spec, int subtract, uint8_t *chan_mask, uint8_t *spec_mask,
                          double *fit_out, double *bpi_out, double *stats)
{
    if (window < 1 || nsamps % window != 0 || order < 0 || order > 12 || order >= nchans) return -1;
    const int64_t nchunk = nsamps / window;
    double *bp = (double *)malloc(sizeof(double) * (size_t)nchans * 5);
    uint8_t *raw = (uint8_t *)malloc((size_t)nchunk);
    if (!bp || !raw) { free(bp); free(raw); return -2; }
    double *bpi = bp + nchans, *fit = bp + 2 * nchans, *tmp = bp + 3 * nchans, *dev = bp + 4 * nchans;
    for (int b = 0; b < nbeams; ++b) {
        float *xb = in + (size_t)b * nchans * nsamps;
        /* H1 */
        for (int c = 0; c < nchans; ++c) {
            double S = 0.0;
            const float *x = xb + (size_t)c * nsamps;
            for (int64_t t = 0; t < nsamps; ++t) S += (double)x[t];
            bp[c] = S / (double)nsamps;
        }
        /* H2 */
        const double med = median_of(bp, nchans, tmp);
        for (int c = 0; c < nchans; ++c) dev[c] = fabs(bp[c] - med);
        const double mad = median_of(dev, nchans, tmp);
        const double lim = (k_mask * 1.4826) * mad;
        int nmask = 0;
        for (int c = 0; c < nchans; ++c) nmask += (bp[c] - med) > lim;
        for (int c = 0; c < nchans; ++c) {
            bpi[c] = bp[c];
            if (!((bp[c] - med) > lim)) continue;
            int l = c - 1, r = c + 1;
            while (l >= 0 && (bp[l] - med) > lim) --l;
            while (r < nchans && (bp[r] - med) > lim) ++r;
            if (l >= 0 && r < nchans) bpi[c] = 0.5 * (bp[l] + bp[r]);
            else if (l >= 0) bpi[c] = bp[l];
            else if (r < nchans) bpi[c] = bp[r];
        }
        /* H3 */
        double coef[16];
        if (orc_polyfit_u(bpi, nchans, order, coef) != 0) { free(bp); free(raw); return -1; }
        for (int c = 0; c < nchans; ++c) {
            const double u = nchans > 1 ? 2.0 * (double)c / (double)(nchans - 1) - 1.0 : 0.0;
            double v = coef[order];
            for (int k = order - 1; k >= 0; --k) v = v * u + coef[k];        /* Horner */
            fit[c] = v;
        }
        /* H4 */
        double se = 0.0, s1 = 0.0, s2 = 0.0;
        for (int c = 0; c < nchans; ++c) {
            const double e = fit[c] - bpi[c];
            se += e * e; s1 += bpi[c]; s2 += bpi[c] * bpi[c];
        }
        const double rmse = sqrt(se / (double)nchans);
        const double mean_bp = s1 / (double)nchans;
        double var_bp = s2 / (double)nchans - mean_bp * mean_bp;
        if (var_bp < 0.0) var_bp = 0.0;
        const double std_bp = sqrt(var_bp);
        if (stats) { stats[4 * b] = rmse; stats[4 * b + 1] = mean_bp; stats[4 * b + 2] = std_bp; stats[4 * b + 3] = (double)nmask; }
        for (int c = 0; c < nchans; ++c) {
            if (fit_out) fit_out[(size_t)b * nchans + c] = fit[c];
            if (bpi_out) bpi_out[(size_t)b * nchans + c] = bpi[c];
        }
        /* H5 */
        for (int c = 0; c < nchans; ++c) {
            float *x = xb + (size_t)c * nsamps;
            const double thr = fit[c] + k_chan * rmse;
            for (int64_t j = 0; j < nchunk; ++j) {
                double C = 0.0;
                for (int64_t t = j * window; t < (j + 1) * window; ++t) C += (double)x[t];
                raw[j] = (C / (double)window > thr) ? 1 : 0;
            }
            for (int64_t j = 0; j < nchunk; ++j) {
                uint8_t m = raw[j];
                if (j > 0) m |= raw[j - 1];
                if (j + 1 < nchunk) m |= raw[j + 1];
                if (chan_mask) chan_mask[((size_t)b * nchans + c) * nchunk + j] = m;
                if (m) for (int64_t t = j * window; t < (j + 1) * window; ++t) x[t] = (float)fit[c];
            }
        }
        /* H6 */
        const double thr_s = mean_bp + k_spec * std_bp;
        for (int64_t t = 0; t < nsamps; ++t) {
            double s = 0.0;
            for (int c = 0; c < nchans; ++c) s += (double)xb[(size_t)c * nsamps + t];
            const uint8_t m = (s / (double)nchans > thr_s) ? 1 : 0;
            if (spec_mask) spec_mask[(size_t)b * nsamps + t] = m;
            if (m) for (int c = 0; c < nchans; ++c) xb[(size_t)c * nsamps + t] = (float)fit[c];
        }
        /* H7 */
        if (subtract)
            for (int c = 0; c < nchans; ++c) {
                float *x = xb + (size_t)c * nsamps;
                const float f = (float)fit[c];
                for (int64_t t = 0; t < nsamps; ++t) x[t] = x[t] - f;
            }
    }
    free(bp); free(raw);
    return 0;
}

/* ================================================================== clustering (NEXT-3) ======== */
/* Detections are points x[i] = (time, DM, SNR) ("(time, DM, intensity) triplets").  The distance
 * function "assigns a different value to each dimension (T_t, SNR_t, DM_t)": reading K-i, q is in the
 * neighbourhood of p when |dt| <= eps[0] and |dDM| <= eps[1] and |dSNR| <= eps[2] (p is its own neighbour).
 * A point is a core point when its neighbourhood holds at least min_pts points. */
static int in_box(const double *x, int64_t i, int64_t j, const double *eps)
{
    return fabs(x[3 * i] - x[3 * j]) <= eps[0] && fabs(x[3 * i + 1] - x[3 * j + 1]) <= eps[1] &&
           fabs(x[3 * i + 2] - x[3 * j + 2]) <= eps[2];
}

static int64_t region_query(const double *x, int64_t n, int64_t p, const double *eps, int64_t *out)
{
    int64_t m = 0;
    for (int64_t j = 0; j < n; ++j)
        if (in_box(x, p, j, eps)) out[m++] = j;          /* ascending index order */
    return m;
}

/* Textbook DBSCAN (the definitions quoted at PAPER.md:118-120: a cluster is a maximal set of density-connected
 * points, everything else is noise).  Points are visited in index order; a cluster grows breadth-first through the
 * FULL neighbourhood of every core point; a border point keeps the first cluster that reaches it.
 * label[i] = cluster id (0, 1, ... in order of discovery) or -1 (noise).  Returns the number of clusters. */
int64_t orc_dbscan(const double *x, int64_t n, const double *eps, int min_pts, int32_t *label)
{
    int64_t *nb = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n ? n : 1));
    int64_t *queue = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n ? n : 1));
    uint8_t *queued = (uint8_t *)calloc((size_t)(n ? n : 1), 1);
    for (int64_t i = 0; i < n; ++i) label[i] = -2;        /* -2 = unclassified */
    int32_t cid = 0;
    for (int64_t p = 0; p < n; ++p) {
        if (label[p] != -2) continue;
        int64_t m = region_query(x, n, p, eps, nb);
        if (m < min_pts) { label[p] = -1; continue; }
        int64_t head = 0, tail = 0;
        label[p] = cid;
        queue[tail++] = p; queued[p] = 1;
        while (head < tail) {
            const int64_t q = queue[head++];
            m = region_query(x, n, q, eps, nb);
            if (m < min_pts) continue;                   /* border point: belongs, does not expand */
            for (int64_t k = 0; k < m; ++k) {
                const int64_t r = nb[k];
                if (label[r] == -2 || label[r] == -1) label[r] = cid;
                if (label[r] == cid && !queued[r]) { queue[tail++] = r; queued[r] = 1; }
            }
        }
        ++cid;
    }
    free(nb); free(queue); free(queued);
    return cid;
}

/* FDBSCAN (after Zhou et al. 2000): as DBSCAN, but a core point's neighbourhood contributes only
 * REPRESENTATIVE points as seeds for further expansion: "at the border of a core point's neighborhood, two for each
 * dimension, one for each direction when placing the core point at the origin".  Reading K-ii: for dimension k and
 * direction s the representative is the neighbour of this cluster with the largest s (x_q[k] - x_p[k]) > 0, the lowest
 * index among equals; a point is expanded at most once.  Every neighbour of an expanded core point still joins the
 * cluster; fewer region queries are made, so clusters can split where DBSCAN would chain them. */
int64_t orc_fdbscan(const double *x, int64_t n, const double *eps, int min_pts, int32_t *label, int64_t *n_queries)
{
    int64_t *nb = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n ? n : 1));
    int64_t *queue = (int64_t *)malloc(sizeof(int64_t) * (size_t)(6 * (n ? n : 1)));
    uint8_t *expanded = (uint8_t *)calloc((size_t)(n ? n : 1), 1);
    for (int64_t i = 0; i < n; ++i) label[i] = -2;
    int32_t cid = 0;
    int64_t nq = 0;
    for (int64_t p = 0; p < n; ++p) {
        if (label[p] != -2) continue;
        int64_t m = region_query(x, n, p, eps, nb); ++nq;
        if (m < min_pts) { label[p] = -1; continue; }
        int64_t head = 0, tail = 0;
        queue[tail++] = p;
        int first = 1;
        while (head < tail) {
            const int64_t q = queue[head++];
            if (expanded[q]) continue;
            expanded[q] = 1;
            if (!first) { m = region_query(x, n, q, eps, nb); ++nq; }
            first = 0;
            if (m < min_pts) continue;
            for (int64_t k = 0; k < m; ++k)
                if (label[nb[k]] == -2 || label[nb[k]] == -1) label[nb[k]] = cid;
            for (int dim = 0; dim < 3; ++dim)
                for (int dir = 1; dir >= -1; dir -= 2) {
                    int64_t best = -1;
                    double bestv = 0.0;
                    for (int64_t k = 0; k < m; ++k) {
                        const int64_t r = nb[k];
                        if (label[r] != cid) continue;
                        const double v = (double)dir * (x[3 * r + dim] - x[3 * q + dim]);
                        if (v > bestv) { bestv = v; best = r; }      /* strict: the lowest index among equals */
                    }
                    if (best >= 0 && !expanded[best]) queue[tail++] = best;
                }
        }
        ++cid;
    }
    if (n_queries) *n_queries = nq;
    free(nb); free(queue); free(expanded);
    return cid;
}

/* ================================================================== candidate classifier (NEXT-3) */
/* Eq. 3: S(dDM)/S = sqrt(pi)/2 * erf(zeta)/zeta, = 1 at zeta = 0 (even in zeta). */
double orc_dm_response(double zeta)
{
    const double z = fabs(zeta);
    if (z < 1e-12) return 1.0;
    return 0.5 * sqrt(3.14159265358979323846) * erf(z) / z;
}

/* Eq. 4: zeta = 6.91e-3 * dDM * bandwidth_MHz / (W_ms * nu_GHz^3). */
double orc_zeta(double ddm, double bw_mhz, double w_ms, double nu_ghz)
{
    return 6.91e-3 * ddm * bw_mhz / (w_ms * (nu_ghz * nu_ghz * nu_ghz));
}

/* The eight steps of PAPER.md:144-156 for ONE cluster of m detections (t[i], dm_idx[i], snr[i]):
 *  1 signature over d in [dmin, dmax] of the cluster: sig[d] = max SNR of the detections at d, cnt[d] = their number
 *    (reading K-iii: "collapsing the time dimension" keeps the strongest detection of each DM; 0 where there is none)
 *  2 k-element moving average, centred, clipped to [dmin, dmax] (divided by the number of elements present)
 *  3 d* = the DM with the most detections (lowest d among equals), snr* = its maximum SNR; DM(d*) < 1.0 -> RFI
 *  4 W = (t_last - t_first + 1) * tsamp of the detections at d*          (reading K-iv), in ms
 *  5 normalise the smoothed signature by its maximum
 *  6 model[d] = Eq. 3 at zeta(DM_d - DM_d*) (Eq. 4; bandwidth and centre frequency of the band)
 *  7 rmse = sqrt(mean_d (model - signature)^2) over [dmin, dmax]
 *  8 rmse > rmse_max -> RFI, else candidate
 * res[0] = class (0 candidate, 1 RFI: DM < 1, 2 RFI: curve mismatch), res[1] = d*, res[2] = snr*, res[3] = W_ms,
 * res[4] = rmse (0 for class 1).  Returns 0, -1 on bad arguments. */
int orc_classify_cluster(const int32_t *t, const int32_t *dm_idx, const float *snr, int64_t m, double dm_low,
                         double dm_step, double tsamp, double bw_mhz, double nu_ghz, int k_smooth, double rmse_max,
                         double *res)
{
    if (m < 1 || k_smooth < 1 || !(k_smooth & 1)) return -1;
    int dmin = dm_idx[0], dmax = dm_idx[0];
    for (int64_t i = 1; i < m; ++i) { if (dm_idx[i] < dmin) dmin = dm_idx[i]; if (dm_idx[i] > dmax) dmax = dm_idx[i]; }
    const int nd = dmax - dmin + 1;
    double *sig = (double *)calloc((size_t)nd * 3, sizeof(double));
    int64_t *cnt = (int64_t *)calloc((size_t)nd, sizeof(int64_t));
    double *sm = sig + nd, *model = sig + 2 * nd;
    for (int64_t i = 0; i < m; ++i) {                                     /* 1 */
        const int d = dm_idx[i] - dmin;
        if (cnt[d] == 0 || (double)snr[i] > sig[d]) sig[d] = (double)snr[i];
        cnt[d] += 1;
    }
    const int h = k_smooth / 2;
    for (int d = 0; d < nd; ++d) {                                        /* 2 */
        double s = 0.0; int c = 0;
        for (int e = d - h; e <= d + h; ++e) if (e >= 0 && e < nd) { s += sig[e]; ++c; }
        sm[d] = s / (double)c;
    }
    int dstar = 0;                                                        /* 3 */
    for (int d = 1; d < nd; ++d) if (cnt[d] > cnt[dstar]) dstar = d;
    res[1] = (double)(dstar + dmin);
    res[2] = sig[dstar];
    const double dm_star = dm_low + (double)(dstar + dmin) * dm_step;
    int32_t t0 = 0, t1 = 0; int have = 0;                                 /* 4 */
    for (int64_t i = 0; i < m; ++i)
        if (dm_idx[i] - dmin == dstar) {
            if (!have || t[i] < t0) t0 = t[i];
            if (!have || t[i] > t1) t1 = t[i];
            have = 1;
        }
    const double w_ms = (double)(t1 - t0 + 1) * tsamp * 1e3;
    res[3] = w_ms;
    if (dm_star < 1.0) { res[0] = 1.0; res[4] = 0.0; free(sig); free(cnt); return 0; }
    double mx = 0.0;                                                      /* 5 */
    for (int d = 0; d < nd; ++d) if (sm[d] > mx) mx = sm[d];
    double se = 0.0;
    for (int d = 0; d < nd; ++d) {                                        /* 6, 7 */
        const double ddm = (dm_low + (double)(d + dmin) * dm_step) - dm_star;
        model[d] = orc_dm_response(orc_zeta(ddm, bw_mhz, w_ms, nu_ghz));
        const double e = model[d] - (mx > 0.0 ? sm[d] / mx : 0.0);
        se += e * e;
    }
    const double rmse = sqrt(se / (double)nd);
    res[4] = rmse;
    res[0] = rmse > rmse_max ? 2.0 : 0.0;                                 /* 8 */
    free(sig); free(cnt);
    return 0;
}

/* ================================================================== 4-bit quantiser (NEXT-4) ==== */
/* Eq. 5 for the complex channelised voltages: "16-bit complex values are quantized to 4-bits with two
 * complex components packed into one byte", Fig. 5b: signed 16 bit -> signed 4 bit.  Reading G-ii:
 *   Xmax = max |component| of the buffer;  code(v) = sign(v) * floor(7 * log(1 + mu |v| / Xmax) / log(1 + mu) + 0.5)
 *   in [-7, 7] as a two's-complement nibble;  byte = (code(re) & 15) | (code(im) & 15) << 4;  Xmax = 0 -> zeros. */
void orc_mulaw_c4(const int16_t *volt, int64_t n, double mu, uint8_t *packed, int32_t *xmax_out)
{
    int32_t xmax = 0;
    for (int64_t i = 0; i < 2 * n; ++i) {
        const int32_t a = volt[i] < 0 ? -(int32_t)volt[i] : (int32_t)volt[i];
        if (a > xmax) xmax = a;
    }
    if (xmax_out) *xmax_out = xmax;
    const double den = log1p(mu);
    for (int64_t i = 0; i < n; ++i) {
        int code[2];
        for (int k = 0; k < 2; ++k) {
            const int32_t v = volt[2 * i + k];
            const int32_t a = v < 0 ? -v : v;
            int c = 0;
            if (xmax > 0 && a > 0) c = (int)floor(7.0 * (log1p(mu * ((double)a / (double)xmax)) / den) + 0.5);
            code[k] = v < 0 ? -c : c;
        }
        packed[i] = (uint8_t)((code[0] & 15) | ((code[1] & 15) << 4));
    }
}

/* ================================================================== 16-bit dedispersion input (NEXT-4) */
/* out[b][d][t] = sum_c in[b][c][t + delay(d,c)] for uint16 samples, uint32 accumulation (exact: 4096 x 65535 < 2^32);
 * the 4-bit variant is this routine on the caller's unpacked nibbles.  Loop order b, d, c, t as orc_dedisperse_u8_rows. */
void orc_dedisperse_u16_rows(const uint16_t *in, int nbeams, int nchans, int64_t nsamps, const int32_t *delay, int ndms,
                             int64_t nsamps_out, uint32_t *out)
{
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int b = 0; b < nbeams; ++b)
        for (int d = 0; d < ndms; ++d) {
            uint32_t *o = out + ((size_t)b * ndms + d) * (size_t)nsamps_out;
            for (int64_t t = 0; t < nsamps_out; ++t) o[t] = 0;
            for (int c = 0; c < nchans; ++c) {
                const uint16_t *x = in + ((size_t)b * nchans + c) * (size_t)nsamps + delay[(size_t)d * nchans + c];
                for (int64_t t = 0; t < nsamps_out; ++t) o[t] += (uint32_t)x[t];
            }
        }
}
