// Host-buffer chain: multibeam batching across CUDA streams with overlapped host-to-device
// copies (BASELINE.json north_star item 4; the paper's per-beam threads each copy their own
// beam to the GPU).  The beams are split into nstreams contiguous groups, group g on stream g:
//   H2D(group g) -> clip -> dedisperse -> detect, so group g+1's copy overlaps group g's compute.
#include "mdsm_internal.h"

static int ensure(void **ptr, size_t *have, size_t need)
{
    if (*ptr && *have >= need) return MDSM_OK;
    if (*ptr) cudaFree(*ptr);
    *ptr = nullptr;
    *have = 0;
    cudaError_t e = cudaMalloc(ptr, need ? need : 1);
    if (e != cudaSuccess) {
        mdsm_set_error("workspace cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
        *ptr = nullptr;
        return e == cudaErrorMemoryAllocation ? MDSM_ENOMEM : MDSM_ECUDA;
    }
    *have = need;
    return MDSM_OK;
}

extern "C" int mdsm_pipeline_host(mdsm_plan *p, const void *h_in, int dtype, int window, double k_chan,
                                  double k_spec, double snr_thresh, mdsm_event *h_events, int64_t max_events,
                                  uint64_t *h_count, int nstreams)
{
    MDSM_REQUIRE(p && h_in && h_count, "null argument");
    MDSM_REQUIRE(dtype == MDSM_F32 || dtype == MDSM_U8, "dtype must be MDSM_F32 or MDSM_U8");
    MDSM_REQUIRE(max_events >= 0 && (h_events || max_events == 0), "bad event buffer");
    MDSM_REQUIRE(window >= 0 && (window == 0 || p->nsamps % window == 0), "window must be 0 (no clip) or divide nsamps");
    if (nstreams < 1) nstreams = 1;
    if (nstreams > p->nbeams) nstreams = p->nbeams;
    int rc;
    if (p->dedisp_kernel != 1) {
        // scratch of the dedispersion kernel (no-op once reserved).  Beam groups on different streams may only run
        // side by side when every beam has its own scratch slot; otherwise the whole chain goes through one stream.
        if ((rc = mdsm_plan_reserve(p, dtype, 0))) return rc;
        const int slots = p->scratch_slots[dtype];
        if (slots > 0 && slots < p->nbeams) nstreams = 1;
    }
    const size_t esize = dtype == MDSM_F32 ? 4 : 1;
    const size_t beam_in = (size_t)p->nchans * p->nsamps * esize;
    if ((rc = ensure(&p->ws_in, &p->ws_in_bytes, beam_in * p->nbeams))) return rc;
    if ((rc = ensure(&p->ws_out, &p->ws_out_bytes, (size_t)p->nbeams * p->ndms * p->nsamps * 4))) return rc;
    const bool post = dtype == MDSM_F32 && (p->post_median_window > 1 || p->post_detrend);
    if (post && p->post_median_window > 1 &&
        (rc = ensure(&p->ws_filt, &p->ws_filt_bytes, (size_t)p->nbeams * p->ndms * p->nsamps * 4))) return rc;
    if (!p->ws_events || p->ws_max_events < max_events) {
        cudaFree(p->ws_events);
        p->ws_events = nullptr;
        MDSM_CUDA_TRY(cudaMalloc((void **)&p->ws_events, sizeof(mdsm_event) * (size_t)(max_events ? max_events : 1)));
        p->ws_max_events = max_events;
    }
    if (!p->ws_count) MDSM_CUDA_TRY(cudaMalloc((void **)&p->ws_count, sizeof(unsigned long long)));
    while ((int)p->ws_streams.size() < nstreams) {
        cudaStream_t s;
        MDSM_CUDA_TRY(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
        p->ws_streams.push_back(s);
        cudaEvent_t ev;
        MDSM_CUDA_TRY(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        p->ws_done.push_back(ev);
    }
    // everything that enqueues work runs inside this lambda: on an error the copies from the caller's h_in and the kernels
    // already in flight are waited for before returning, so that the caller may free or reuse its buffers
    auto enqueue = [&]() -> int {
    // the counter is zeroed on stream 0; the other streams wait for that before their first detect
        MDSM_CUDA_TRY(cudaMemsetAsync(p->ws_count, 0, sizeof(unsigned long long), p->ws_streams[0]));
        MDSM_CUDA_TRY(cudaEventRecord(p->ws_done[0], p->ws_streams[0]));
        for (int s = 1; s < nstreams; ++s) MDSM_CUDA_TRY(cudaStreamWaitEvent(p->ws_streams[s], p->ws_done[0], 0));

        // contiguous beam groups, one per stream: whole groups per launch keep the persistent dedispersion grid full
        // (one beam is only ~7 waves of tiles), while group g+1's copy still overlaps group g's kernels
        const int per = (p->nbeams + nstreams - 1) / nstreams;
        for (int b = 0, g = 0; b < p->nbeams; b += per, ++g) {
            cudaStream_t st = p->ws_streams[g % nstreams];
            const int nb = b + per <= p->nbeams ? per : p->nbeams - b;
            MDSM_CUDA_TRY(cudaMemcpyAsync((char *)p->ws_in + beam_in * b, (const char *)h_in + beam_in * b, beam_in * nb,
                                          cudaMemcpyHostToDevice, st));
            if (window > 0 && (rc = mdsm_rfi_clip(p, p->ws_in, dtype, b, nb, window, k_chan, k_spec, nullptr, nullptr, st))) return rc;
            if ((rc = mdsm_dedisperse(p, p->ws_in, dtype, b, nb, p->ws_out, st))) return rc;
            const void *series = p->ws_out;
            if (post) {                      // the paper's optional post-processing stage, fp32 series only
                if (p->post_median_window > 1) {
                    if ((rc = mdsm_median_filter(p, (const float *)p->ws_out, (float *)p->ws_filt, b, nb, p->post_median_window, st))) return rc;
                    series = p->ws_filt;
                }
                if (p->post_detrend && (rc = mdsm_detrend(p, (float *)series, b, nb, nullptr, st))) return rc;
            }
            if ((rc = mdsm_detect(p, series, dtype, b, nb, snr_thresh, p->ws_events, max_events, p->ws_count, st))) return rc;
        }
        // join every stream into stream 0, then read back the count and the events
        for (int s = 1; s < nstreams; ++s) {
            MDSM_CUDA_TRY(cudaEventRecord(p->ws_done[s], p->ws_streams[s]));
            MDSM_CUDA_TRY(cudaStreamWaitEvent(p->ws_streams[0], p->ws_done[s], 0));
        }
        return MDSM_OK;
    };
    if ((rc = enqueue()) != MDSM_OK) {
        for (cudaStream_t s : p->ws_streams) cudaStreamSynchronize(s);
        return rc;
    }
    unsigned long long cnt = 0;
    MDSM_CUDA_TRY(cudaMemcpyAsync(&cnt, p->ws_count, sizeof(cnt), cudaMemcpyDeviceToHost, p->ws_streams[0]));
    MDSM_CUDA_TRY(cudaStreamSynchronize(p->ws_streams[0]));
    *h_count = cnt;
    const size_t ncopy = (size_t)(cnt < (unsigned long long)max_events ? cnt : (unsigned long long)max_events);
    if (ncopy) {
        MDSM_CUDA_TRY(cudaMemcpyAsync(h_events, p->ws_events, ncopy * sizeof(mdsm_event), cudaMemcpyDeviceToHost, p->ws_streams[0]));
        MDSM_CUDA_TRY(cudaStreamSynchronize(p->ws_streams[0]));
    }
    if (cnt > (unsigned long long)max_events) {
        mdsm_set_error("event buffer overflow: %llu events found, %lld stored", cnt, (long long)max_events);
        return MDSM_EOVERFLOW;
    }
    return MDSM_OK;
}
