// Detection kernels (PAPER.md:116 n-sigma thresholding; normalisation by the series' own
// mean / standard deviation; readings D-i..D-vii in DESIGN.md section 3).
//
//   series_stats_kernel  one CTA per (beam, dm) series: S, Q over t < nsamps_out by warp-shuffle
//                        reduction (uint64 exact for uint32 series, fp64 for float series),
//                        then mean / rms with single IEEE fp64 ops in the oracle's order.
//   threshold_emit_kernel  every sample: snr = ((double)x - mean)/rms > thr ?  Candidates are
//                        pre-filtered in the element type (one compare per sample against a bound
//                        rounded down; a warp without candidates leaves), then with one fp64
//                        subtract-compare; events are appended with warp-aggregated atomics (one
//                        atomicAdd per warp per vote).
#include "mdsm_internal.h"

namespace {

constexpr int kThreads = 256;

template <typename A> __device__ __forceinline__ A wsum(A v)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    return v;
}

template <typename T> __device__ __forceinline__ T as_elem(unsigned w);
template <> __device__ __forceinline__ float as_elem<float>(unsigned w) { return __uint_as_float(w); }
template <> __device__ __forceinline__ uint32_t as_elem<uint32_t>(unsigned w) { return w; }

template <typename T> constexpr bool kIsFloat = false;
template <> constexpr bool kIsFloat<float> = true;

template <typename T> struct SAcc;
template <> struct SAcc<float> { using type = double; };
template <> struct SAcc<uint32_t> { using type = unsigned long long; };

template <typename T>
__global__ void __launch_bounds__(kThreads)
series_stats_kernel(const T *__restrict__ out, int beam0, int ndms, long long nsamps, long long n,
                    double *__restrict__ stats)
{
    using A = typename SAcc<T>::type;
    const int d = blockIdx.x, b = beam0 + blockIdx.y;
    const T *x = out + ((size_t)b * ndms + d) * (size_t)nsamps;
    A S = 0, Q = 0;
    const bool vec = ((uintptr_t)x % 16 == 0);
    if (vec) {
        const long long n4 = n / 4;
        const uint4 *xv = reinterpret_cast<const uint4 *>(x);
        for (long long i = threadIdx.x; i < n4; i += kThreads) {
            const uint4 v = xv[i];
            const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const A e = (A)as_elem<T>(w[k]);
                S += e;
                Q += e * e;
            }
        }
        for (long long i = n4 * 4 + threadIdx.x; i < n; i += kThreads) {
            A e = (A)x[i];
            S += e;
            Q += e * e;
        }
    } else {
        for (long long i = threadIdx.x; i < n; i += kThreads) {
            A e = (A)x[i];
            S += e;
            Q += e * e;
        }
    }
    __shared__ A red[2][kThreads / 32];
    S = wsum(S);
    Q = wsum(Q);
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = S; red[1][threadIdx.x >> 5] = Q; }
    __syncthreads();
    if (threadIdx.x == 0) {
        A s = 0, q = 0;
        for (int i = 0; i < kThreads / 32; ++i) { s += red[0][i]; q += red[1][i]; }
        const double dn = (double)n;
        const double mean = __ddiv_rn((double)s, dn);
        double var = __dsub_rn(__ddiv_rn((double)q, dn), __dmul_rn(mean, mean));
        if (var < 0.0) var = 0.0;
        double *o = stats + ((size_t)b * ndms + d) * 2;
        o[0] = mean;
        o[1] = __dsqrt_rn(var);
    }
}

// Thresholds the four samples t0 .. t0+3 of one series x (n valid samples) and appends the events; called by whole warps.
template <typename T>
__device__ __forceinline__ void threshold_emit4(const T *__restrict__ x, long long n, long long t0, int b, int d, double mean,
                                                double rms, double thr, double cut, mdsm_event *__restrict__ events,
                                                long long max_events, unsigned long long *__restrict__ count)
{
    T v[4];
    if (t0 + 3 < n && ((uintptr_t)x % 16 == 0)) {
        const uint4 u = *reinterpret_cast<const uint4 *>(x + t0);
        const unsigned w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = as_elem<T>(w[k]);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = (t0 + k < n) ? x[t0 + k] : (T)0;
    }
    const int lane = threadIdx.x & 31;
    // Cheap conservative pre-filter in the element type: a sample can only be an event if x > mean + cut, so one
    // compare per sample against a bound rounded DOWN (with a 1e-12 relative margin for the fp64 subtraction below)
    // rules almost everything out, and a warp none of whose 128 samples passes skips the fp64 path altogether.
    bool cand = false;
    {
        const double bound = mean + cut;
        const double slack = bound - (fabs(bound) * 1e-12 + 1e-300);
        if (kIsFloat<T>) {                                         // float series
            const float cf = __double2float_rd(slack);
#pragma unroll
            for (int k = 0; k < 4; ++k) cand |= (t0 + k < n) && ((float)v[k] > cf);
        } else {                                                    // uint32 series
            const double fl = floor(slack);
            const bool all = fl < 0.0;
            const uint32_t cu = all ? 0u : (fl >= 4294967295.0 ? 0xffffffffu : (uint32_t)fl);
#pragma unroll
            for (int k = 0; k < 4; ++k) cand |= (t0 + k < n) && (all || (uint32_t)v[k] > cu);
        }
    }
    if (!__any_sync(0xffffffffu, cand)) return;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        bool hit = false;
        double snr = 0.0;
        if (t0 + k < n) {
            const double dv = __dsub_rn((double)v[k], mean);
            if (dv > cut) {
                snr = __ddiv_rn(dv, rms);
                hit = snr > thr;
            }
        }
        const unsigned ballot = __ballot_sync(0xffffffffu, hit);
        if (ballot) {
            unsigned long long base = 0;
            const int leader = __ffs(ballot) - 1;
            if (lane == leader) base = atomicAdd(count, (unsigned long long)__popc(ballot));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (hit) {
                const unsigned long long slot = base + __popc(ballot & ((1u << lane) - 1));
                if (slot < (unsigned long long)max_events) {
                    mdsm_event e;
                    e.beam = b; e.dm_idx = d; e.t = (int32_t)(t0 + k); e.snr = (float)snr;
                    events[slot] = e;
                }
            }
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(kThreads)
threshold_emit_kernel(const T *__restrict__ out, int beam0, int ndms, long long nsamps, long long n,
                      const double *__restrict__ stats, double thr, mdsm_event *__restrict__ events,
                      long long max_events, unsigned long long *__restrict__ count)
{
    const int d = blockIdx.y, b = beam0 + blockIdx.z;
    const double mean = stats[((size_t)b * ndms + d) * 2];
    const double rms = stats[((size_t)b * ndms + d) * 2 + 1];
    if (rms == 0.0) return;                          // whole CTA: uniform
    // snr > thr  =>  x - mean > thr*rms*(1 - 2^-40): cheap conservative pre-filter (thr*rms >= 0);
    // for negative thresholds every sample is a candidate.
    const double cut = thr > 0.0 ? thr * rms * (1.0 - 9.094947017729282e-13) : -1.7976931348623157e308;
    const T *x = out + ((size_t)b * ndms + d) * (size_t)nsamps;
    const long long t0 = ((long long)blockIdx.x * kThreads + threadIdx.x) * 4;
    threshold_emit4<T>(x, n, t0, b, d, mean, rms, thr, cut, events, max_events, count);
}

// a5 + a6 in ONE launch and ONE read of `out`: a CTA of 256 threads owns a series (several CTAs per SM overlap their passes).  Pass 1 (from HBM) reduces S and Q and
// records the maximum of every 128-sample chunk (what one warp loads per step) in shared memory; once mean and rms are
// known, pass 2 looks at the chunk maxima only and re-reads (from L2) just the chunks that can hold an event:
// snr > thr  =>  x > mean + thr*rms*(1 - 2^-40), a bound rounded down in the element type.
constexpr int kFusedThreads = 256;
template <typename T>
__global__ void __launch_bounds__(kFusedThreads)
detect_fused_kernel(const T *__restrict__ out, int beam0, int ndms, long long nsamps, long long n, double *__restrict__ stats,
                    double thr, mdsm_event *__restrict__ events, long long max_events, unsigned long long *__restrict__ count)
{
    using A = typename SAcc<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *cmax = reinterpret_cast<T *>(smem_raw);                    // [ceil(n4 / 32)] chunk maxima
    const int d = blockIdx.x, b = beam0 + blockIdx.y;
    const T *x = out + ((size_t)b * ndms + d) * (size_t)nsamps;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    A S = 0, Q = 0;
    const bool vec = ((uintptr_t)x % 16 == 0);
    const long long n4 = vec ? n / 4 : 0;
    const uint4 *xv = reinterpret_cast<const uint4 *>(x);
    constexpr int U = 4;                                                  // independent 128-bit loads in flight per thread
    const T lowest = kIsFloat<T> ? (T)(-3.402823466e38f) : (T)0;
    for (long long base = 0; base < n4; base += (long long)U * kFusedThreads) {
        uint4 v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = base + (long long)u * kFusedThreads + threadIdx.x;
            v[u] = i < n4 ? xv[i] : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = base + (long long)u * kFusedThreads + threadIdx.x;
            T m = lowest;
            if (i < n4) {
                const unsigned w[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const T t = as_elem<T>(w[k]);
                    const A e = (A)t;
                    S += e;
                    Q += e * e;
                    m = t > m ? t : m;
                }
            }
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) {
                const T other = __shfl_xor_sync(0xffffffffu, m, o);
                m = other > m ? other : m;
            }
            const long long c = ((base + (long long)u * kFusedThreads) >> 5) + warp;
            if (lane == 0 && c * 32 < n4) cmax[c] = m;
        }
    }
    for (long long i = n4 * 4 + threadIdx.x; i < n; i += kFusedThreads) {
        A e = (A)x[i];
        S += e;
        Q += e * e;
    }
    __shared__ A red[2][kFusedThreads / 32];
    __shared__ double s_stats[2];
    S = wsum(S);
    Q = wsum(Q);
    if (lane == 0) { red[0][warp] = S; red[1][warp] = Q; }
    __syncthreads();
    if (threadIdx.x == 0) {
        A s = 0, q = 0;
        for (int i = 0; i < kFusedThreads / 32; ++i) { s += red[0][i]; q += red[1][i]; }
        const double dn = (double)n;
        const double mean = __ddiv_rn((double)s, dn);
        double var = __dsub_rn(__ddiv_rn((double)q, dn), __dmul_rn(mean, mean));
        if (var < 0.0) var = 0.0;
        double *o = stats + ((size_t)b * ndms + d) * 2;
        o[0] = s_stats[0] = mean;
        o[1] = s_stats[1] = __dsqrt_rn(var);
    }
    __syncthreads();
    const double mean = s_stats[0], rms = s_stats[1];
    if (rms == 0.0) return;
    const double cut = thr > 0.0 ? thr * rms * (1.0 - 9.094947017729282e-13) : -1.7976931348623157e308;
    // the same conservative bound threshold_emit4 applies per sample, here per chunk maximum
    const double bound = mean + cut;
    const double slack = bound - (fabs(bound) * 1e-12 + 1e-300);
    bool all = false;
    T cb;
    if (kIsFloat<T>) {
        cb = (T)__double2float_rd(slack);
        all = !(slack > -3.0e38);
    } else {
        const double fl = floor(slack);
        all = fl < 0.0;
        cb = (T)(all ? 0u : (fl >= 4294967295.0 ? 0xffffffffu : (uint32_t)fl));
    }
    const long long nchunks = (n4 + 31) / 32;
    for (long long c = warp; c < nchunks; c += kFusedThreads / 32)
        if (all || cmax[c] > cb)                                  // the vector part only (n4 * 4 samples): the rest follows below
            threshold_emit4<T>(x, n4 * 4, (c * 32 + lane) * 4, b, d, mean, rms, thr, cut, events, max_events, count);
    // what the vector loop did not cover (an unaligned row: everything; else the last n % 4 samples)
    for (long long t0 = n4 * 4 + (long long)threadIdx.x * 4; t0 - (long long)lane * 4 < n; t0 += (long long)kFusedThreads * 4)
        threshold_emit4<T>(x, n, t0, b, d, mean, rms, thr, cut, events, max_events, count);
}

template <typename T>
int launch_detect_t(mdsm_plan *p, const T *out, int beam0, int nb, double thr, mdsm_event *ev, long long max_events,
                    unsigned long long *count, cudaStream_t st)
{
    MDSM_REQUIRE(p->ndms <= 65535 && nb <= 65535, "ndms and nb must be <= 65535");
    dim3 g1(p->ndms, nb);
    const size_t fsmem = (size_t)((p->nsamps_out / 4 + 31) / 32 + 1) * sizeof(T);
    if (p->detect_two_pass || fsmem > 160 * 1024) {
        // the two-launch form (statistics, then a grid over (time, series)): option "detect_two_pass" for comparison, and
        // by itself for series whose chunk maxima do not fit the fused kernel's shared memory (nsamps_out above ~5.2 M)
        series_stats_kernel<T><<<g1, kThreads, 0, st>>>(out, beam0, p->ndms, p->nsamps, p->nsamps_out, p->d_series_stats);
        MDSM_CUDA_TRY(cudaGetLastError());
        dim3 g2((unsigned)((p->nsamps_out + kThreads * 4 - 1) / (kThreads * 4)), p->ndms, nb);
        threshold_emit_kernel<T><<<g2, kThreads, 0, st>>>(out, beam0, p->ndms, p->nsamps, p->nsamps_out, p->d_series_stats,
                                                          thr, ev, max_events, count);
        MDSM_CUDA_TRY(cudaGetLastError());
        p->launches += 2;
        return MDSM_OK;
    }
    if (fsmem > 48 * 1024) MDSM_CUDA_TRY(cudaFuncSetAttribute(detect_fused_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fsmem));
    detect_fused_kernel<T><<<g1, kFusedThreads, fsmem, st>>>(out, beam0, p->ndms, p->nsamps, p->nsamps_out, p->d_series_stats, thr, ev,
                                                        max_events, count);
    MDSM_CUDA_TRY(cudaGetLastError());
    p->launches += 1;
    return MDSM_OK;
}

}  // namespace

int mdsm_launch_detect(mdsm_plan *p, const void *d_out, int dtype, int beam0, int nb, double snr_thresh,
                       mdsm_event *d_events, int64_t max_events, unsigned long long *d_count, cudaStream_t st)
{
    if (dtype == MDSM_F32)
        return launch_detect_t<float>(p, (const float *)d_out, beam0, nb, snr_thresh, d_events, max_events, d_count, st);
    return launch_detect_t<uint32_t>(p, (const uint32_t *)d_out, beam0, nb, snr_thresh, d_events, max_events, d_count, st);
}

// ---------------------------------------------------------------------------------------------------------------------
// mdsm_detect_noalloc (include/mdsm.h): detection for callers that must not allocate device memory -- plug-ins that
// live inside a host application which owns the GPU's memory, and real-time loops in which cudaMalloc's device-wide
// synchronisation would stall the other beams.  It is the two-launch form above (series_stats_kernel, then
// threshold_emit_kernel) with the (mean, rms) pairs the first kernel hands to the second kept in a fixed array of the
// library's device image instead of plan-owned cudaMalloc memory.  No plan, no cudaMalloc / cudaFree.
//
// g_noalloc_series_stats is resident on every GPU that loads this module, until the process exits (512 KB each).
// In HOST code the name below is only a handle for the runtime, not a device address: handing it to a kernel as a
// pointer would fault, or quietly touch host memory on systems where the GPU can reach it.  noalloc_scratch() turns it
// into the real device address once per device with cudaGetSymbolAddress and the launches use that address.
#include <mutex>

namespace {

static __device__ __align__(256) double g_noalloc_series_stats[2 * (size_t)MDSM_DETECT_NOALLOC_MAX_SERIES];

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mutex;
double *g_noalloc_addr[kNoallocMaxDevices] = {};           // device address of the array, per device ordinal; 0 = not asked yet

// Device address of the array on the CURRENT device.  The first call per device asks the runtime (which loads this
// library's module on that device if no kernel of it ran there before); later calls read the table.
int noalloc_scratch(double **addr)
{
    int dev = -1;
    MDSM_CUDA_TRY(cudaGetDevice(&dev));
    MDSM_REQUIRE(dev >= 0 && dev < kNoallocMaxDevices, "mdsm_detect_noalloc: device ordinal %d outside 0..%d", dev,
                 kNoallocMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[dev]) {
        void *a = nullptr;
        MDSM_CUDA_TRY(cudaGetSymbolAddress(&a, g_noalloc_series_stats));
        MDSM_REQUIRE(a != nullptr, "mdsm_detect_noalloc: the runtime returned a null address for the scratch array");
        g_noalloc_addr[dev] = static_cast<double *>(a);
    }
    *addr = g_noalloc_addr[dev];
    return MDSM_OK;
}

template <typename T>
int launch_detect_noalloc_t(const T *series, int nbeams, int ndms, long long nsamps, long long n, double thr, mdsm_event *ev,
                            long long max_events, unsigned long long *count, double *stats, cudaStream_t st)
{
    // Nothing in `stats` needs clearing: series_stats_kernel writes the pair of every (beam, dm) of this call before
    // threshold_emit_kernel (same stream, so ordered after it) reads exactly those pairs.
    series_stats_kernel<T><<<dim3(ndms, nbeams), kThreads, 0, st>>>(series, 0, ndms, nsamps, n, stats);
    MDSM_CUDA_TRY(cudaGetLastError());
    dim3 g2((unsigned)((n + kThreads * 4 - 1) / (kThreads * 4)), ndms, nbeams);
    threshold_emit_kernel<T><<<g2, kThreads, 0, st>>>(series, 0, ndms, nsamps, n, stats, thr, ev, max_events, count);
    MDSM_CUDA_TRY(cudaGetLastError());
    return MDSM_OK;
}

}  // namespace

extern "C" int mdsm_detect_noalloc(const void *d_series, int dtype, int nbeams, int ndms, int64_t nsamps, int64_t nsamps_out,
                                   double snr_thresh, mdsm_event *d_events, int64_t max_events, unsigned long long *d_count,
                                   void *cuda_stream)
{
    MDSM_REQUIRE(d_series && d_count, "mdsm_detect_noalloc: null series or count pointer");
    MDSM_REQUIRE(dtype == MDSM_F32 || dtype == MDSM_U8, "mdsm_detect_noalloc: dtype must be MDSM_F32 (float series) or MDSM_U8 (uint32 series)");
    MDSM_REQUIRE(nbeams >= 1 && ndms >= 1 && nbeams <= 65535 && ndms <= 65535, "mdsm_detect_noalloc: nbeams and ndms must be in 1..65535");
    MDSM_REQUIRE(nsamps_out >= 1 && nsamps_out <= nsamps, "mdsm_detect_noalloc: need 1 <= nsamps_out <= nsamps");
    MDSM_REQUIRE((nsamps_out + kThreads * 4 - 1) / (kThreads * 4) <= 2147483647LL, "mdsm_detect_noalloc: series too long");
    MDSM_REQUIRE(max_events >= 0 && (d_events || max_events == 0), "mdsm_detect_noalloc: bad event buffer");
    MDSM_REQUIRE(snr_thresh == snr_thresh, "mdsm_detect_noalloc: snr_thresh must not be NaN");
    MDSM_REQUIRE((long long)nbeams * ndms <= (long long)MDSM_DETECT_NOALLOC_MAX_SERIES,
                 "mdsm_detect_noalloc: %lld series (nbeams * ndms) exceed the fixed scratch of MDSM_DETECT_NOALLOC_MAX_SERIES = %d series; "
                 "this entry point never allocates, so split the series over several calls on one stream",
                 (long long)nbeams * ndms, (int)MDSM_DETECT_NOALLOC_MAX_SERIES);
    double *stats = nullptr;
    const int rc = noalloc_scratch(&stats);
    if (rc) return rc;
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    if (dtype == MDSM_F32)
        return launch_detect_noalloc_t<float>((const float *)d_series, nbeams, ndms, nsamps, nsamps_out, snr_thresh, d_events,
                                              max_events, d_count, stats, st);
    return launch_detect_noalloc_t<uint32_t>((const uint32_t *)d_series, nbeams, ndms, nsamps, nsamps_out, snr_thresh, d_events,
                                             max_events, d_count, stats, st);
}
