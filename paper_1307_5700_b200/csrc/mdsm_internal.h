// Internal declarations shared by the libmdsm translation units (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "mdsm.h"

void mdsm_set_error(const char *fmt, ...);

#define MDSM_CUDA_TRY(expr)                                                                   \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess) {                                                             \
            mdsm_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, \
                           __LINE__);                                                         \
            return MDSM_ECUDA;                                                                \
        }                                                                                     \
    } while (0)

#define MDSM_REQUIRE(cond, ...)          \
    do {                                 \
        if (!(cond)) {                   \
            mdsm_set_error(__VA_ARGS__); \
            return MDSM_EINVAL;          \
        }                                \
    } while (0)

// Plan-time tables of the dedispersion kernels (see dedisperse_rows.cu and DESIGN.md section 6.1).
struct RowsTables {
    bool ok = false;
    int G = 0;                                    // channels per pre-summed group
    int D = 0, T = 0, NW = 0, DB = 0;             // DMs per warp, words per thread and DM, consumer warps, DMs per block
    int span = 0, stride = 0;                     // samples a tile's accumulators cover per DM / outputs it owns (its time step)
    int Q = 0, CS = 0, pitch = 0;                 // groups per slab, row slots per stage, elements per row slot
    int nslab = 0, nblk = 0, ngroups = 0, nyrows = 0, dmax = 0, maxpat = 0, slabs_per_part = 0;
    long long ystride = 0;                        // elements per y row (nsamps rounded up to 16 bytes)
    int sigma_max = 0, stages = 0;
    size_t smem_bytes = 0;
    double rows_per_block = 0.0;                  // y rows a DM block stages per tile (statistics for kernel_info)
    void *d_rowdesc = nullptr;                    // int4 [nblk][nslab][CS]
    uint32_t *d_ent = nullptr;                    // [nblk][nslab][DB*Q]
    int32_t *d_sigma = nullptr;                   // [DB]
    int32_t *d_group_row0 = nullptr;              // [ngroups + 1]
    int16_t *d_ydelta = nullptr;                  // [nyrows][8]
};

// Tables of the TMEM-window variant of the main kernel (fp32; dedisperse_rows.cu): the same
// pre-summed rows, staged TMA -> shared memory -> tensor memory, consumed with tcgen05.ld at run-time column offsets.
struct TmemTables {
    bool ok = false;
    int D = 0, P = 0, DB = 0, span = 0;           // DMs per warp, outputs per lane and DM, DMs per block, outputs per tile and DM
    int CS = 0, pitch = 0, stages = 0;            // row slots per shared-memory stage, words per slot, stages
    int nslab_max = 0, nblk = 0, tabw = 0;        // slabs per block (padded), DM blocks, 32-bit words of a slab's table slice
    int sigma_max = 0;
    size_t smem_bytes = 0;
    double groups_per_slab = 0.0, cols_per_group = 0.0;   // statistics for kernel_info
    void *d_rowdesc = nullptr;                    // int4 [nblk][nslab_max][CS]
    uint32_t *d_tab = nullptr;                    // [nblk][nslab_max][tabw]
    int32_t *d_nslab = nullptr;                   // [nblk]
    int32_t *d_sigma = nullptr;                   // [DB]
};

struct mdsm_plan {
    int nbeams, nchans, ndms;
    double f_top, foff, tsamp, dm_low, dm_step;
    int64_t nsamps, max_delay, nsamps_out;
    int device;
    int sm_count;
    std::vector<int32_t> h_delay;  // [ndms][nchans]
    int32_t *d_delay = nullptr;

    // clip scratch
    double *d_chan_stats = nullptr;   // [nbeams][nchans][4] = mean, sig, thr(unused), repl
    double *d_bandpass = nullptr;     // [nbeams][nchans] averaged bandpass (mdsm_bandpass_clip)
    double *d_spec_sum = nullptr;     // [nbeams][nsamps]    spectrum sums (fp64; exact for u8)
    double *d_spec_part = nullptr;    // [nbeams][spec_parts][2] partial M1, M2 (f32 path)
    unsigned long long *d_spec_part_u = nullptr;  // same, integer path
    int spec_parts = 0;
    // detect scratch
    double *d_series_stats = nullptr; // [nbeams][ndms][2] = mean, rms

    int detect_two_pass = 0;          // option "detect_two_pass": 1 = statistics and thresholding as two launches (comparison)
    int dedisp_kernel = 0;            // option "dedisp_kernel": 0 auto, 1 direct, 2 rows
    int group_size = 0;               // option "group_size": channels per pre-summed group, 0 = chosen by the cost model
    // rows_f32: 32-bit rows (MDSM_F32 and, with integer adds, MDSM_U16); rows_u8 / rows_u4: packed 16-bit rows, flushed to the
    // uint32 output every 256 / 4096 channels (what a 16-bit lane holds of 255s / 15s)
    RowsTables rows_f32, rows_u8, rows_u4;
    TmemTables tmem_f32;
    void *d_scratch[4] = {nullptr, nullptr, nullptr, nullptr};  // per dtype: pre-summed rows [slots][nyrows][ystride] (mdsm_plan_reserve)
    int scratch_slots[4] = {0, 0, 0, 0};                        // beams the scratch holds at a time
    size_t scratch_bytes[4] = {0, 0, 0, 0};

    // host pipeline workspace (allocated on first mdsm_pipeline_host)
    void *ws_in = nullptr; size_t ws_in_bytes = 0;
    void *ws_out = nullptr; size_t ws_out_bytes = 0;
    void *ws_filt = nullptr; size_t ws_filt_bytes = 0;    // median-filtered series (options post_median_window)
    int post_median_window = 0, post_detrend = 0;         // optional post-processing inside mdsm_pipeline_host (fp32)
    mdsm_event *ws_events = nullptr; int64_t ws_max_events = 0;
    unsigned long long *ws_count = nullptr;
    std::vector<cudaStream_t> ws_streams;
    std::vector<cudaEvent_t> ws_done;

    int64_t launches = 0;
};

inline const RowsTables &mdsm_rows_of(const mdsm_plan *p, int dtype)
{
    return dtype == MDSM_U8 ? p->rows_u8 : (dtype == MDSM_U4 ? p->rows_u4 : p->rows_f32);
}
inline bool mdsm_dtype_ok(int dtype) { return dtype >= MDSM_F32 && dtype <= MDSM_U4; }

// stage launchers (each returns an MDSM_* status)
int mdsm_launch_clip(mdsm_plan *p, void *d_in, int dtype, int beam0, int nb, int window, double k_chan,
                     double k_spec, uint8_t *d_chan_mask, uint8_t *d_spec_mask, cudaStream_t st);
int mdsm_launch_bandpass_clip(mdsm_plan *p, float *in, int beam0, int nb, int window, int order, double k_mask, double k_chan,
                              double k_spec, int subtract, uint8_t *chan_mask, uint8_t *spec_mask, double *d_fit, double *d_stats,
                              cudaStream_t st);
int mdsm_launch_dedisperse_direct(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                  cudaStream_t st);
int mdsm_launch_dedisperse_rows(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                cudaStream_t st);
int mdsm_rows_build_tables(mdsm_plan *p);
void mdsm_rows_free_tables(mdsm_plan *p);
size_t mdsm_rows_scratch_bytes_per_beam(const mdsm_plan *p, int dtype);
int mdsm_launch_detect(mdsm_plan *p, const void *d_out, int dtype, int beam0, int nb, double snr_thresh,
                       mdsm_event *d_events, int64_t max_events, unsigned long long *d_count, cudaStream_t st);
