// Post-processing of the dedispersed series (section 2.2.3).
//
//   median_filter_kernel  Eq. 2 with operation = median: the paper's layout -- a 2-D grid, one row of
//                         CTAs per series, every CTA stages its slice plus a halo in shared memory and every thread
//                         takes the median of its points' neighbourhoods.  The neighbourhood is clipped to [0, n) at
//                         the ends (reading E-i); selection is by rank counting (stable ranks, so ties are harmless),
//                         which needs no sorting network per window size.  Bit-identical to the oracle.
//   detrend_kernel        one CTA per series: pass 1 regression sums (the residual variance follows
//                         algebraically from the sum of squares), pass 2 subtract + normalise from L2; fp64 sums.
// Both are HBM-bound: one read + one write of the series.
#include "mdsm_internal.h"

namespace {

constexpr int kThreads = 256;
constexpr int kPer = 8;                         // outputs per thread (that many independent loads in flight while staging)
constexpr int kTile = kThreads * kPer;          // outputs per CTA
constexpr int kMaxHalf = 16;                    // window <= 33

// median of the 2H+1 values w[0..2H] by H+1 passes of a bubble sort (min/max pairs: exact selection, no NaNs here)
template <int H> __device__ __forceinline__ float median_full(float (&w)[2 * H + 1])
{
    constexpr int W = 2 * H + 1;
#pragma unroll
    for (int p = 0; p <= H; ++p)
#pragma unroll
        for (int i = 0; i + 1 < W - p; ++i) {
            const float lo = fminf(w[i], w[i + 1]), hi = fmaxf(w[i], w[i + 1]);
            w[i] = lo;
            w[i + 1] = hi;
        }
    return w[H];
}

// HFAST > 0: compiled window (registers, unrolled) for the points whose neighbourhood is whole; the clipped
// neighbourhoods at the two ends of a series, and windows without a compiled variant, go through rank counting.
template <int HFAST>
__global__ void __launch_bounds__(kThreads)
median_filter_kernel(const float *__restrict__ in, float *__restrict__ out, int beam0, int ndms, long long nsamps, long long n,
                     int half)
{
    __shared__ float sx[kTile + 2 * kMaxHalf];
    const size_t row = ((size_t)(beam0 + blockIdx.z) * ndms + blockIdx.y) * (size_t)nsamps;
    const float *x = in + row;
    float *y = out + row;
    const long long t0 = (long long)blockIdx.x * kTile;
    for (int i = threadIdx.x; i < kTile + 2 * half; i += kThreads) {
        const long long t = t0 - half + i;
        sx[i] = (t >= 0 && t < n) ? x[t] : 0.0f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
        const int u = threadIdx.x + k * kThreads;          // coalesced outputs
        const long long m = t0 + u;
        if (m >= n) continue;
        if (HFAST > 0 && m - half >= 0 && m + half <= n - 1) {
            float w[2 * (HFAST > 0 ? HFAST : 1) + 1];
#pragma unroll
            for (int i = 0; i < 2 * HFAST + 1; ++i) w[i] = sx[u + i];
            y[m] = median_full<(HFAST > 0 ? HFAST : 1)>(w);
            continue;
        }
        int lo = u, hi = u + 2 * half;                     // window in sx coordinates (centre = u + half)
        if (m - half < 0) lo += (int)(half - m);
        if (m + half > n - 1) hi -= (int)(m + half - (n - 1));
        const int cnt = hi - lo + 1;
        const int r1 = cnt / 2, r0 = (cnt & 1) ? r1 : r1 - 1;
        float v0 = 0.0f, v1 = 0.0f;
        for (int i = lo; i <= hi; ++i) {
            const float a = sx[i];
            int rank = 0;
            for (int j = lo; j <= hi; ++j) {
                const float b = sx[j];
                rank += (b < a) || (b == a && j < i);
            }
            if (rank == r0) v0 = a;
            if (rank == r1) v1 = a;
        }
        y[m] = (cnt & 1) ? v1 : (float)(((double)v0 + (double)v1) / 2.0);
    }
}

__device__ __forceinline__ double block_sum(double v, double *red)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    __syncthreads();                                        // red[] free again
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kThreads / 32; ++i) s += red[i];
    return s;
}

__global__ void __launch_bounds__(kThreads)
detrend_kernel(float *__restrict__ series, int beam0, int ndms, long long nsamps, long long n, double *__restrict__ params)
{
    __shared__ double red[kThreads / 32];
    const size_t sidx = (size_t)(beam0 + blockIdx.y) * ndms + blockIdx.x;
    float *x = series + sidx * (size_t)nsamps;
    const double tbar = __ddiv_rn(__dsub_rn((double)n, 1.0), 2.0);
    const bool vec = ((uintptr_t)x % 16 == 0);
    const long long n4 = vec ? n / 4 : 0;
    // pass 1 (HBM): regression sums and the sum of squares; the residual variance follows algebraically,
    //   sum r^2 = sum (y - mean)^2 - slope^2 * sum (t - tbar)^2   (fp64: cancellation ~1e-14 relative)
    double sy = 0.0, syy = 0.0, sty = 0.0;
    constexpr int U = 4;                                    // independent 128-bit loads in flight per thread
    for (long long base = 0; base < n4; base += (long long)U * kThreads) {
        float4 q[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = base + (long long)u * kThreads + threadIdx.x;
            q[u] = i < n4 ? reinterpret_cast<const float4 *>(x)[i] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = base + (long long)u * kThreads + threadIdx.x;
            if (i >= n4) continue;
            const double v[4] = {(double)q[u].x, (double)q[u].y, (double)q[u].z, (double)q[u].w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                sy += v[k];
                syy += v[k] * v[k];
                sty += ((double)(4 * i + k) - tbar) * v[k];
            }
        }
    }
    for (long long t = n4 * 4 + threadIdx.x; t < n; t += kThreads) {
        const double v = (double)x[t];
        sy += v;
        syy += v * v;
        sty += ((double)t - tbar) * v;
    }
    sy = block_sum(sy, red);
    syy = block_sum(syy, red);
    sty = block_sum(sty, red);
    const double dn = (double)n;
    const double stt = dn * (dn * dn - 1.0) / 12.0;         // sum (t - tbar)^2, closed form
    const double mean = sy / dn;
    const double slope = stt > 0.0 ? sty / stt : 0.0;
    double sr = (syy - dn * mean * mean) - slope * slope * stt;
    if (sr < 0.0) sr = 0.0;
    // a constant series has sr == rounding noise of syy - n mean^2: compare with the scale of the data
    const double sd = (sr <= 1e-24 * (syy > 1.0 ? syy : 1.0)) ? 0.0 : sqrt(sr / dn);
    const double inv = sd > 0.0 ? 1.0 / sd : 0.0;
    // pass 2 (L2): subtract the line, normalise
    for (long long base = 0; base < n4; base += (long long)U * kThreads) {
        float4 qq[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = base + (long long)u * kThreads + threadIdx.x;
            qq[u] = i < n4 ? reinterpret_cast<const float4 *>(x)[i] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = base + (long long)u * kThreads + threadIdx.x;
            if (i >= n4) continue;
            float4 q = qq[u];
            const double t = (double)(4 * i) - tbar;
            q.x = (float)(((double)q.x - (mean + slope * t)) * inv);
            q.y = (float)(((double)q.y - (mean + slope * (t + 1.0))) * inv);
            q.z = (float)(((double)q.z - (mean + slope * (t + 2.0))) * inv);
            q.w = (float)(((double)q.w - (mean + slope * (t + 3.0))) * inv);
            reinterpret_cast<float4 *>(x)[i] = q;
        }
    }
    for (long long t = n4 * 4 + threadIdx.x; t < n; t += kThreads)
        x[t] = (float)(((double)x[t] - (mean + slope * ((double)t - tbar))) * inv);
    if (threadIdx.x == 0 && params) { params[3 * sidx] = mean; params[3 * sidx + 1] = slope; params[3 * sidx + 2] = sd; }
}

static int check_range(const mdsm_plan *p, const void *ptr, int beam0, int nb)
{
    MDSM_REQUIRE(p && ptr, "null argument");
    MDSM_REQUIRE(beam0 >= 0 && nb >= 1 && beam0 + nb <= p->nbeams, "beam range [%d, %d) outside the plan's %d beams", beam0, beam0 + nb, p->nbeams);
    MDSM_REQUIRE(p->ndms <= 65535 && nb <= 65535, "ndms and nb must be <= 65535");
    return MDSM_OK;
}

}  // namespace

extern "C" int mdsm_median_filter(mdsm_plan *p, const float *d_series, float *d_filtered, int beam0, int nb, int window,
                                  void *cuda_stream)
{
    int rc = check_range(p, d_series, beam0, nb);
    if (rc) return rc;
    MDSM_REQUIRE(d_filtered && d_filtered != d_series, "the filtered series need their own buffer");
    MDSM_REQUIRE(window >= 1 && (window & 1) && window <= 2 * kMaxHalf + 1, "window must be odd and <= %d", 2 * kMaxHalf + 1);
    dim3 grid((unsigned)((p->nsamps_out + kTile - 1) / kTile), p->ndms, nb);
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    const int h = window / 2;
#define MDSM_MEDIAN(H) median_filter_kernel<H><<<grid, kThreads, 0, st>>>(d_series, d_filtered, beam0, p->ndms, p->nsamps, p->nsamps_out, h)
    switch (h) {
        case 1: MDSM_MEDIAN(1); break;
        case 2: MDSM_MEDIAN(2); break;
        case 3: MDSM_MEDIAN(3); break;
        case 4: MDSM_MEDIAN(4); break;
        default: MDSM_MEDIAN(0); break;
    }
#undef MDSM_MEDIAN
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    return MDSM_OK;
}

extern "C" int mdsm_detrend(mdsm_plan *p, float *d_series, int beam0, int nb, double *d_params, void *cuda_stream)
{
    int rc = check_range(p, d_series, beam0, nb);
    if (rc) return rc;
    dim3 grid(p->ndms, nb);
    detrend_kernel<<<grid, kThreads, 0, (cudaStream_t)cuda_stream>>>(d_series, beam0, p->ndms, p->nsamps, p->nsamps_out, d_params);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    return MDSM_OK;
}
