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

// Geometry of the tiled dedispersion kernel (see dedisperse_tiled.cu and DESIGN.md section 6).
struct TiledTables {
    int dms_per_warp = 0, warps = 0, tpt = 0, cs = 0;   // D, NW, T (samples per thread), channels per slab
    int dm_block = 0, n_dm_blocks = 0;            // DB = D*NW
    int tile_t = 0;                               // 32*T output samples per CTA
    int row_words = 0;                            // staged elements (f32 / u16) per channel row
    int max_off = 0;                              // largest per-DM register offset
    int32_t *d_row_start = nullptr;               // [n_dm_blocks][nchans]   first staged sample - tile_t0
    void *d_warp_tab = nullptr;                   // [n_dm_blocks][nslab][warps][CS] packed window base + per-DM offsets
    int32_t *d_sigma = nullptr;                   // [n_dm_blocks*dm_block]  output time shear per DM
    int sigma_max = 0;
    // pair pre-sum mode (fp32): rows are (channel pair, delay difference) sums, see dedisperse_tiled.cu
    bool pairs = false;
    int nslab_max = 0, nyrows = 0, nparts = 1;                // slabs per block (padded), rows of the pre-summed copy per beam
    int32_t *d_src_row = nullptr;                 // [n_dm_blocks][nslab_max*CS]  row of the pre-summed copy staged as row r (-1: none)
    int32_t *d_nslab_blk = nullptr;               // [n_dm_blocks]  slabs of this block
    int32_t *d_yrow_chan = nullptr, *d_yrow_delta = nullptr;   // [npairs + 1] first pre-summed row of every pair; [nyrows] delay difference of a row
    int geom = 0;                                 // index of the compiled geometry the tables were built for
    bool ok = false;
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
    double *d_spec_sum = nullptr;     // [nbeams][nsamps]    spectrum sums (fp64; exact for u8)
    double *d_spec_part = nullptr;    // [nbeams][spec_parts][2] partial M1, M2 (f32 path)
    unsigned long long *d_spec_part_u = nullptr;  // same, integer path
    int spec_parts = 0;
    // detect scratch
    double *d_series_stats = nullptr; // [nbeams][ndms][2] = mean, rms

    int dedisp_kernel = 0;            // 0 auto, 1 direct, 2 tiled
    int tiled_geom_f32 = -1, tiled_geom_u8 = -1;   // compiled tile geometry per dtype (option "tiled_geom_*"), -1 = automatic
    TiledTables tiled_f32, tiled_u8;
    void *d_pairs = nullptr; size_t pairs_bytes = 0;   // pre-summed channel pairs of an fp32 input (allocated on first use)
    int pair_presum_u8 = 1;                            // option "pair_presum_u8" (integer kernel)
    int pair_presum = 1;                               // option "pair_presum" (fp32 only; falls back when the tables do not fit)
    void *d_widen = nullptr; size_t widen_bytes = 0;   // uint16 copy of a uint8 input (allocated on first use)

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

// stage launchers (each returns an MDSM_* status)
int mdsm_launch_clip(mdsm_plan *p, void *d_in, int dtype, int beam0, int nb, int window, double k_chan,
                     double k_spec, uint8_t *d_chan_mask, uint8_t *d_spec_mask, cudaStream_t st);
int mdsm_launch_dedisperse_direct(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                  cudaStream_t st);
int mdsm_launch_dedisperse_tiled(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                 cudaStream_t st);
int mdsm_tiled_build_tables(mdsm_plan *p);
int mdsm_tiled_num_geoms(int dtype);
void mdsm_tiled_free_tables(mdsm_plan *p);
int mdsm_launch_detect(mdsm_plan *p, const void *d_out, int dtype, int beam0, int nb, double snr_thresh,
                       mdsm_event *d_events, int64_t max_events, unsigned long long *d_count, cudaStream_t st);
