// Direct (global-load) brute-force dedispersion: the simple reference kernel of the CUDA path.
//   out[b][d][t] = sum_c in[b][c][t + delay(d,c)]
// One thread owns kPer outputs of one DM spaced blockDim apart (coalesced along t); the DM's
// delay row is staged in shared memory.  Used for shapes / alignments the tiled kernel does not
// take, and as a second CUDA implementation to cross-check the tiled kernel.
#include "mdsm_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kPer = 4;

// U4: TIn = uint8_t holds two 4-bit samples per byte along time (low nibble first); a row is nsamps / 2 bytes
template <typename TIn, typename TOut, bool U4 = false>
__global__ void __launch_bounds__(kThreads)
dedisperse_direct_kernel(const TIn *__restrict__ in, TOut *__restrict__ out, const int32_t *__restrict__ delay,
                         int beam0, int nchans, int ndms, long long nsamps, long long nsamps_out)
{
    extern __shared__ int32_t sdelay[];
    const int d = blockIdx.y;
    const int b = beam0 + blockIdx.z;
    for (int c = threadIdx.x; c < nchans; c += kThreads) sdelay[c] = delay[(size_t)d * nchans + c];
    __syncthreads();
    const long long t0 = (long long)blockIdx.x * (kThreads * kPer) + threadIdx.x;
    const size_t row_elems = U4 ? (size_t)nsamps / 2 : (size_t)nsamps;
    const TIn *base = in + (size_t)b * nchans * row_elems;
    TOut acc[kPer];
    bool ok[kPer];
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
        acc[k] = 0;
        ok[k] = t0 + k * kThreads < nsamps_out;
    }
    for (int c = 0; c < nchans; ++c) {
        if constexpr (U4) {
            const TIn *row = base + (size_t)c * row_elems;
            const long long s0 = sdelay[c] + t0;
#pragma unroll
            for (int k = 0; k < kPer; ++k)
                if (ok[k]) {
                    const long long sidx = s0 + k * kThreads;
                    acc[k] += (TOut)((row[sidx >> 1] >> (4 * (int)(sidx & 1))) & 15);
                }
        } else {
            const TIn *row = base + (size_t)c * nsamps + sdelay[c] + t0;
#pragma unroll
            for (int k = 0; k < kPer; ++k)
                if (ok[k]) acc[k] += (TOut)row[k * kThreads];
        }
    }
    TOut *orow = out + ((size_t)b * ndms + d) * (size_t)nsamps + t0;
#pragma unroll
    for (int k = 0; k < kPer; ++k)
        if (ok[k]) orow[k * kThreads] = acc[k];
}

}  // namespace

int mdsm_launch_dedisperse_direct(mdsm_plan *p, const void *d_in, int dtype, int beam0, int nb, void *d_out,
                                  cudaStream_t st)
{
    dim3 grid((unsigned)((p->nsamps_out + kThreads * kPer - 1) / (kThreads * kPer)), p->ndms, nb);
    MDSM_REQUIRE(p->ndms <= 65535 && nb <= 65535, "ndms and nb must be <= 65535 for the direct kernel");
    const size_t smem = (size_t)p->nchans * sizeof(int32_t);
    MDSM_REQUIRE(smem <= 48 * 1024, "direct kernel supports nchans <= 12288");
    if (dtype == MDSM_F32)
        dedisperse_direct_kernel<float, float><<<grid, kThreads, smem, st>>>(
            (const float *)d_in, (float *)d_out, p->d_delay, beam0, p->nchans, p->ndms, p->nsamps, p->nsamps_out);
    else if (dtype == MDSM_U8)
        dedisperse_direct_kernel<uint8_t, uint32_t><<<grid, kThreads, smem, st>>>(
            (const uint8_t *)d_in, (uint32_t *)d_out, p->d_delay, beam0, p->nchans, p->ndms, p->nsamps, p->nsamps_out);
    else if (dtype == MDSM_U16)
        dedisperse_direct_kernel<uint16_t, uint32_t><<<grid, kThreads, smem, st>>>(
            (const uint16_t *)d_in, (uint32_t *)d_out, p->d_delay, beam0, p->nchans, p->ndms, p->nsamps, p->nsamps_out);
    else
        dedisperse_direct_kernel<uint8_t, uint32_t, true><<<grid, kThreads, smem, st>>>(
            (const uint8_t *)d_in, (uint32_t *)d_out, p->d_delay, beam0, p->nchans, p->ndms, p->nsamps, p->nsamps_out);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    return MDSM_OK;
}
