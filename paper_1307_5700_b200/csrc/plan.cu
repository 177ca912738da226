// Plan: argument checks, the fp64 host delay table (Eq. 1), device scratch.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <new>

#include "mdsm_internal.h"

static thread_local char g_err[512] = "";

void mdsm_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *mdsm_last_error(void) { return g_err; }

// delay(d,c) = round(4.148808e3 * DM_d * (f_c^-2 - f_top^-2) / tsamp), fp64, round = floor(x+0.5).
// Evaluated on the host only: an fp32 evaluation gets hundreds of entries wrong (reading A2).
static void build_delay_table(mdsm_plan *p)
{
    const double kdm = 4.148808e3;
    const double inv_top2 = 1.0 / (p->f_top * p->f_top);
    p->h_delay.resize((size_t)p->ndms * p->nchans);
    for (int d = 0; d < p->ndms; ++d) {
        const double dm = p->dm_low + (double)d * p->dm_step;
        int32_t *row = p->h_delay.data() + (size_t)d * p->nchans;
        for (int c = 0; c < p->nchans; ++c) {
            const double f = p->f_top + (double)c * p->foff;
            const double x = kdm * dm * (1.0 / (f * f) - inv_top2) / p->tsamp;
            row[c] = (int32_t)floor(x + 0.5);
        }
    }
}

static bool alloc_dev(void **ptr, size_t bytes)
{
    cudaError_t e = cudaMalloc(ptr, bytes ? bytes : 1);
    if (e != cudaSuccess) {
        mdsm_set_error("cudaMalloc(%zu bytes) failed: %s", bytes, cudaGetErrorString(e));
        *ptr = nullptr;
        return false;
    }
    return true;
}

extern "C" mdsm_plan *mdsm_plan_create(int nbeams, int nchans, double f_top, double foff, double tsamp,
                                       int64_t nsamps, double dm_low, double dm_step, int ndms)
{
    if (nbeams < 1 || nchans < 1 || ndms < 1 || nsamps < 1) {
        mdsm_set_error("nbeams, nchans, ndms, nsamps must be >= 1");
        return nullptr;
    }
    if (!(foff < 0.0) || !(tsamp > 0.0) || !(dm_step >= 0.0) || !(dm_low >= 0.0) || !(f_top > 0.0) ||
        !(f_top + (nchans - 1) * foff > 0.0)) {
        mdsm_set_error("need foff < 0, tsamp > 0, dm_step >= 0, dm_low >= 0 and all channel frequencies > 0");
        return nullptr;
    }
    if (nsamps >= ((int64_t)1 << 31)) {
        mdsm_set_error("nsamps must be < 2^31");
        return nullptr;
    }
    mdsm_plan *p = new (std::nothrow) mdsm_plan();
    if (!p) {
        mdsm_set_error("out of host memory");
        return nullptr;
    }
    p->nbeams = nbeams; p->nchans = nchans; p->ndms = ndms;
    p->f_top = f_top; p->foff = foff; p->tsamp = tsamp; p->dm_low = dm_low; p->dm_step = dm_step;
    p->nsamps = nsamps;
    {
        // guard against int32 overflow of the largest delay before building the table
        const double f_lo = f_top + (double)(nchans - 1) * foff;
        const double xmax = 4.148808e3 * (dm_low + (ndms - 1) * dm_step) * (1.0 / (f_lo * f_lo) - 1.0 / (f_top * f_top)) / tsamp;
        if (!(xmax < (double)nsamps)) {
            mdsm_set_error("nsamps (%lld) must exceed the maximum delay (%.0f samples)", (long long)nsamps, xmax);
            delete p;
            return nullptr;
        }
    }
    build_delay_table(p);
    p->max_delay = p->h_delay.back();
    p->nsamps_out = nsamps - p->max_delay;
    if (p->nsamps_out < 1) {
        mdsm_set_error("nsamps (%lld) must exceed the maximum delay (%lld)", (long long)nsamps, (long long)p->max_delay);
        delete p;
        return nullptr;
    }
    cudaError_t e = cudaGetDevice(&p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    if (e != cudaSuccess) {
        mdsm_set_error("no usable CUDA device: %s", cudaGetErrorString(e));
        delete p;
        return nullptr;
    }
    p->spec_parts = 256;
    bool ok = alloc_dev((void **)&p->d_delay, p->h_delay.size() * sizeof(int32_t)) &&
              alloc_dev((void **)&p->d_chan_stats, (size_t)nbeams * nchans * 4 * sizeof(double)) &&
              alloc_dev((void **)&p->d_bandpass, (size_t)nbeams * nchans * sizeof(double)) &&
              alloc_dev((void **)&p->d_spec_sum, (size_t)nbeams * nsamps * sizeof(double)) &&
              alloc_dev((void **)&p->d_spec_part, (size_t)nbeams * p->spec_parts * 2 * sizeof(double)) &&
              alloc_dev((void **)&p->d_spec_part_u, (size_t)nbeams * p->spec_parts * 2 * sizeof(unsigned long long)) &&
              alloc_dev((void **)&p->d_series_stats, (size_t)nbeams * ndms * 2 * sizeof(double));
    if (ok) {
        e = cudaMemcpy(p->d_delay, p->h_delay.data(), p->h_delay.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            mdsm_set_error("delay table upload failed: %s", cudaGetErrorString(e));
            ok = false;
        }
    }
    if (ok && mdsm_rows_build_tables(p) != MDSM_OK) ok = false;
    if (!ok) {
        mdsm_plan_destroy(p);
        return nullptr;
    }
    return p;
}

extern "C" void mdsm_plan_destroy(mdsm_plan *p)
{
    if (!p) return;
    cudaFree(p->d_delay);
    cudaFree(p->d_chan_stats);
    cudaFree(p->d_bandpass);
    cudaFree(p->d_spec_sum);
    cudaFree(p->d_spec_part);
    cudaFree(p->d_spec_part_u);
    cudaFree(p->d_series_stats);
    cudaFree(p->ws_filt);
    mdsm_rows_free_tables(p);
    for (int k = 0; k < 4; ++k) cudaFree(p->d_scratch[k]);
    cudaFree(p->ws_in);
    cudaFree(p->ws_out);
    cudaFree(p->ws_events);
    cudaFree(p->ws_count);
    for (auto s : p->ws_streams) cudaStreamDestroy(s);
    for (auto ev : p->ws_done) cudaEventDestroy(ev);
    delete p;
}

extern "C" int64_t mdsm_plan_max_delay(const mdsm_plan *p) { return p ? p->max_delay : -1; }
extern "C" int64_t mdsm_plan_nsamps_out(const mdsm_plan *p) { return p ? p->nsamps_out : -1; }
extern "C" int64_t mdsm_plan_launch_count(const mdsm_plan *p) { return p ? p->launches : -1; }

extern "C" int mdsm_plan_get_delays(const mdsm_plan *p, int32_t *h_delays)
{
    MDSM_REQUIRE(p && h_delays, "null argument");
    memcpy(h_delays, p->h_delay.data(), p->h_delay.size() * sizeof(int32_t));
    return MDSM_OK;
}

static void drop_scratch(mdsm_plan *p)
{
    for (int k = 0; k < 4; ++k) {
        cudaFree(p->d_scratch[k]);
        p->d_scratch[k] = nullptr;
        p->scratch_slots[k] = 0;
        p->scratch_bytes[k] = 0;
    }
}

extern "C" int mdsm_plan_set_option(mdsm_plan *p, const char *key, int64_t value)
{
    MDSM_REQUIRE(p && key, "null argument");
    if (strcmp(key, "dedisp_kernel") == 0) {
        MDSM_REQUIRE(value >= 0 && value <= 3, "dedisp_kernel must be 0 (auto), 1 (direct), 2 (pre-summed rows, shared-memory operands) or 3 (pre-summed rows, TMEM operands)");
        p->dedisp_kernel = (int)value;
        return MDSM_OK;
    }
    if (strcmp(key, "group_size") == 0) {
        MDSM_REQUIRE(value >= 0 && value <= 8, "group_size must be 0 (chosen by the plan) or 1..8 channels");
        // the tables and the scratch layout change: wait for whatever still uses them, then drop the reservation
        MDSM_CUDA_TRY(cudaDeviceSynchronize());
        drop_scratch(p);
        p->group_size = (int)value;
        return mdsm_rows_build_tables(p);
    }
    if (strcmp(key, "post_median_window") == 0) {
        MDSM_REQUIRE(value == 0 || (value >= 1 && value <= 33 && (value & 1)), "post_median_window must be 0 (off) or odd and <= 33");
        p->post_median_window = (int)value;
        return MDSM_OK;
    }
    if (strcmp(key, "detect_two_pass") == 0) {
        MDSM_REQUIRE(value == 0 || value == 1, "detect_two_pass must be 0 or 1");
        p->detect_two_pass = (int)value;
        return MDSM_OK;
    }
    if (strcmp(key, "post_detrend") == 0) {
        MDSM_REQUIRE(value == 0 || value == 1, "post_detrend must be 0 or 1");
        p->post_detrend = (int)value;
        return MDSM_OK;
    }
    mdsm_set_error("unknown option '%s'", key);
    return MDSM_EINVAL;
}

static int check_common(const mdsm_plan *p, const void *ptr, int dtype, int beam0, int nb, bool dedisp_input = false)
{
    MDSM_REQUIRE(p, "null plan");
    MDSM_REQUIRE(ptr, "null data pointer");
    MDSM_REQUIRE(dtype == MDSM_F32 || dtype == MDSM_U8 || (dedisp_input && mdsm_dtype_ok(dtype)),
                 dedisp_input ? "dtype must be MDSM_F32, MDSM_U8, MDSM_U16 or MDSM_U4" : "dtype must be MDSM_F32 or MDSM_U8");
    MDSM_REQUIRE(beam0 >= 0 && nb >= 1 && beam0 + nb <= p->nbeams, "beam range [%d, %d) outside [0, %d)", beam0,
                 beam0 + nb, p->nbeams);
    int dev = -1;
    MDSM_CUDA_TRY(cudaGetDevice(&dev));
    MDSM_REQUIRE(dev == p->device, "the plan belongs to device %d, the current device is %d", p->device, dev);
    return MDSM_OK;
}

extern "C" int mdsm_rfi_clip(mdsm_plan *p, void *d_in, int dtype, int beam0, int nb, int window, double k_chan,
                             double k_spec, uint8_t *d_chan_mask, uint8_t *d_spec_mask, void *cuda_stream)
{
    int rc = check_common(p, d_in, dtype, beam0, nb);
    if (rc) return rc;
    MDSM_REQUIRE(window >= 1 && p->nsamps % window == 0, "window must be >= 1 and divide nsamps");
    MDSM_REQUIRE(k_chan == k_chan && k_spec == k_spec, "thresholds must not be NaN");
    return mdsm_launch_clip(p, d_in, dtype, beam0, nb, window, k_chan, k_spec, d_chan_mask, d_spec_mask,
                            (cudaStream_t)cuda_stream);
}

extern "C" int mdsm_bandpass_clip(mdsm_plan *p, float *d_in, int beam0, int nb, int window, int order, double k_mask,
                                  double k_chan, double k_spec, int subtract, uint8_t *d_chan_mask, uint8_t *d_spec_mask,
                                  double *d_fit, double *d_stats, void *cuda_stream)
{
    int rc = check_common(p, d_in, MDSM_F32, beam0, nb);
    if (rc) return rc;
    MDSM_REQUIRE(window >= 1 && p->nsamps % window == 0, "window must be >= 1 and divide nsamps");
    MDSM_REQUIRE(order >= 0 && order <= 12 && order < p->nchans, "order must be in [0, 12] and below nchans");
    MDSM_REQUIRE(k_mask == k_mask && k_chan == k_chan && k_spec == k_spec, "thresholds must not be NaN");
    return mdsm_launch_bandpass_clip(p, d_in, beam0, nb, window, order, k_mask, k_chan, k_spec, subtract, d_chan_mask, d_spec_mask,
                                     d_fit, d_stats, (cudaStream_t)cuda_stream);
}

extern "C" int mdsm_dedisperse(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                               void *cuda_stream)
{
    int rc = check_common(p, d_in, dtype, beam0, nb, true);
    if (rc) return rc;
    MDSM_REQUIRE(d_out, "null output pointer");
    MDSM_REQUIRE(dtype != MDSM_U4 || p->nsamps % 2 == 0, "MDSM_U4 needs an even nsamps (two samples per byte)");
    MDSM_REQUIRE(dtype != MDSM_U16 || (double)p->nchans * 65535.0 < 4294967296.0, "MDSM_U16: nchans * 65535 must fit 32 bits");
    const RowsTables &rt = mdsm_rows_of(p, dtype);
    if (p->dedisp_kernel == 1 || (p->dedisp_kernel == 0 && !rt.ok))
        return mdsm_launch_dedisperse_direct(p, d_in, dtype, beam0, nb, d_out, (cudaStream_t)cuda_stream);
    MDSM_REQUIRE(rt.ok, "the pre-summed-rows kernel has no tables for this plan (see mdsm_plan_kernel_info)");
    MDSM_REQUIRE(p->dedisp_kernel != 3 || (dtype == MDSM_F32 && p->tmem_f32.ok), "the TMEM variant has no tables for this plan / dtype");
    MDSM_REQUIRE(p->d_scratch[dtype] != nullptr,
                 "dedispersion scratch not reserved: call mdsm_plan_reserve(plan, dtype, 0) once before mdsm_dedisperse");
    return mdsm_launch_dedisperse_rows(p, d_in, dtype, beam0, nb, d_out, (cudaStream_t)cuda_stream);
}

extern "C" int mdsm_plan_reserve(mdsm_plan *p, int dtype, int64_t max_bytes)
{
    MDSM_REQUIRE(p, "null plan");
    MDSM_REQUIRE(mdsm_dtype_ok(dtype), "dtype must be MDSM_F32, MDSM_U8, MDSM_U16 or MDSM_U4");
    MDSM_REQUIRE(max_bytes >= 0, "max_bytes must be >= 0 (0 = default)");
    const size_t per_beam = mdsm_rows_scratch_bytes_per_beam(p, dtype);
    if (per_beam == 0) return MDSM_OK;                       // this plan runs the direct kernel: nothing to reserve
    void *&scratch = p->d_scratch[dtype];
    int &slots = p->scratch_slots[dtype];
    size_t &bytes = p->scratch_bytes[dtype];
    // max_bytes = 0 asks for "a reservation", not for a new size: an existing one (the caller's explicit cap included)
    // stays as it is.  Without this, mdsm_pipeline_host's own reserve call replaced a caller's cap, and on a device where
    // not every beam fits the size derived from the free memory changed from call to call (free / realloc every buffer).
    if (scratch && max_bytes == 0) return MDSM_OK;
    size_t limit = (size_t)max_bytes;
    if (limit == 0) {
        size_t free_b = 0, total_b = 0;
        MDSM_CUDA_TRY(cudaMemGetInfo(&free_b, &total_b));
        limit = free_b / 4;                                   // default: at most a quarter of what is free now
    }
    int want = (int)std::min<size_t>((size_t)p->nbeams, limit / per_beam);
    if (want < 1) want = 1;
    if (scratch && slots == want) return MDSM_OK;
    if (scratch) {
        MDSM_CUDA_TRY(cudaDeviceSynchronize());
        cudaFree(scratch);
        scratch = nullptr; slots = 0; bytes = 0;
    }
    const cudaError_t e = cudaMalloc(&scratch, per_beam * (size_t)want);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        scratch = nullptr;
        mdsm_set_error("mdsm_plan_reserve: cudaMalloc(%zu bytes for %d beams of pre-summed rows) failed: %s", per_beam * (size_t)want,
                       want, cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? MDSM_ENOMEM : MDSM_ECUDA;
    }
    slots = want;
    bytes = per_beam * (size_t)want;
    return MDSM_OK;
}

extern "C" int mdsm_plan_kernel_info(const mdsm_plan *p, int dtype, char *buf, int64_t buflen)
{
    MDSM_REQUIRE(p && buf && buflen > 0, "null argument");
    MDSM_REQUIRE(mdsm_dtype_ok(dtype), "dtype must be MDSM_F32, MDSM_U8, MDSM_U16 or MDSM_U4");
    const bool f32 = dtype == MDSM_F32;
    const RowsTables &rt = mdsm_rows_of(p, dtype);
    const bool rows = p->dedisp_kernel != 1 && rt.ok;
    if (!rows) {
        snprintf(buf, (size_t)buflen, "kernel=direct reason=%s", p->dedisp_kernel == 1 ? "option" : "no_tables");
        return 0;
    }
    if (p->dedisp_kernel == 3 && !(f32 && p->tmem_f32.ok)) {
        // the same verdict mdsm_dedisperse gives: the TMEM variant exists for fp32 plans with TMEM tables only
        snprintf(buf, (size_t)buflen, "kernel=none reason=%s", f32 ? "no_tmem_tables" : "tmem_f32_only");
        mdsm_set_error("dedisp_kernel = 3 (TMEM variant) has no tables for this plan / dtype: mdsm_dedisperse will return MDSM_EINVAL");
        return MDSM_EINVAL;
    }
    const bool tmem = f32 && p->tmem_f32.ok && p->dedisp_kernel == 3;
    const TmemTables &tt = p->tmem_f32;
    if (tmem)
        snprintf(buf, (size_t)buflen,
                 "kernel=rows operands=tmem group_size=%d dms_per_block=%d tile_samples=%d groups_per_slab=%.2f tmem_cols_per_group=%.1f "
                 "row_slots=%d row_pitch=%d stages=%d smem_bytes=%zu nyrows=%d scratch_slots=%d scratch_bytes=%zu",
                 rt.G, tt.DB, tt.span, tt.groups_per_slab, tt.cols_per_group, tt.CS, tt.pitch, tt.stages, tt.smem_bytes, rt.nyrows,
                 p->scratch_slots[dtype], p->scratch_bytes[dtype]);
    else
    snprintf(buf, (size_t)buflen,
             "kernel=rows operands=smem group_size=%d dms_per_block=%d tile_samples=%d groups_per_slab=%d row_slots=%d row_pitch=%d stages=%d "
             "smem_bytes=%zu nyrows=%d rows_per_block=%.0f scratch_slots=%d scratch_bytes=%zu",
             rt.G, rt.DB, rt.stride, rt.Q, rt.CS, rt.pitch, rt.stages, rt.smem_bytes, rt.nyrows, rt.rows_per_block,
             p->scratch_slots[dtype], p->scratch_bytes[dtype]);
    return 1;
}

extern "C" int mdsm_detect(mdsm_plan *p, const void *d_out, int dtype, int beam0, int nb, double snr_thresh,
                           mdsm_event *d_events, int64_t max_events, unsigned long long *d_count,
                           void *cuda_stream)
{
    int rc = check_common(p, d_out, dtype, beam0, nb);
    if (rc) return rc;
    MDSM_REQUIRE(d_count, "null count pointer");
    MDSM_REQUIRE(max_events >= 0 && (d_events || max_events == 0), "bad event buffer");
    MDSM_REQUIRE(snr_thresh == snr_thresh, "snr_thresh must not be NaN");
    return mdsm_launch_detect(p, d_out, dtype, beam0, nb, snr_thresh, d_events, max_events, d_count,
                              (cudaStream_t)cuda_stream);
}
