// mu-law quantiser, 32-bit float power series -> 8 bits (Eq. 5).  The paper runs
// it on the CPU with a log lookup table next to the disk writer; here it is two HBM-bound kernels:
//   mulaw_max_kernel   Xmax = max x (non-negative floats order like their bit patterns: one atomicMax per CTA)
//   mulaw_code_kernel  code = floor(255 * log1p(mu x / Xmax) / log1p(mu) + 0.5), fp64 like the oracle (reading G-i);
//                      16 samples per thread and step: four 128-bit loads, one 128-bit store.
// 5 bytes per sample (4 + 4 read over the two passes minus what L2 keeps, 1 written).
#include "mdsm_internal.h"

namespace {

__global__ void __launch_bounds__(256) mulaw_max_kernel(const float *__restrict__ x, long long n, unsigned *__restrict__ xmax_bits)
{
    float m = 0.0f;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long n4 = n / 4;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += stride) {
        const float4 v = reinterpret_cast<const float4 *>(x)[i];
        m = fmaxf(m, fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)));          // fmaxf drops NaNs
    }
    for (long long i = n4 * 4 + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += stride) m = fmaxf(m, x[i]);
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, s));
    __shared__ float red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < 8; ++i) m = fmaxf(m, red[i]);
        atomicMax(xmax_bits, __float_as_uint(m));                        // m >= +0: bit patterns are ordered
    }
}

// The decision is the oracle's fp64 one; fp32 settles it whenever the value is not within 1e-3 of a rounding boundary,
// which spares 99.8 % of the samples the fp64 logarithm.
__device__ __forceinline__ unsigned code_of(float x, double xmax, double mu, double inv_den, float xmax_f, float mu_f, float inv_den_f)
{
    if (!(xmax > 0.0) || !(x > 0.0f)) return 0u;
    // 255 log2(1 + a) / log2(1 + mu) with the hardware log2 (MUFU.LG2): the absolute error of vf stays below 1e-4 (rounding of
    // 1 + a to fp32 costs 2^-24 relative to the argument, the unit itself ~2^-22), far inside the 1e-3 guard band
    // (mu >= 1 only: for a small mu the rounding of 1 + a is amplified by 1 / log2(1 + mu), and log1pf takes over)
    const float vf = mu_f >= 1.0f ? 255.0f * (__log2f(1.0f + mu_f * __fdividef(x, xmax_f)) * inv_den_f)
                                  : 255.0f * (log1pf(mu_f * (x / xmax_f)) * inv_den_f);
    const float fr = vf - floorf(vf);
    // guard band: 1e-3 for log1pf; 5e-4 for the hardware log2 with mu >= 1.  Worst-case error of vf on that path, at mu = 1
    // (where the scale 255 / log2(1 + mu) is largest): MUFU.LG2's 2^-22 absolute error x 255 = 6e-5, __fdividef's 2 ulp and
    // the fp32 rounding of 1 + a another ~5e-5 after the same scaling, the two product roundings near vf = 255 3e-5:
    // about 1.5e-4 in all, so 5e-4 leaves a factor three (a band of 2.5e-4 left less than two).
    if (fabsf(fr - 0.5f) >= (mu_f >= 1.0f ? 5e-4f : 1e-3f)) return (unsigned)floorf(vf + 0.5f);
    const double v = 255.0 * (log1p(mu * ((double)x / xmax)) * inv_den);
    return (unsigned)floor(v + 0.5);
}

__global__ void __launch_bounds__(256) mulaw_code_kernel(const float *__restrict__ x, long long n, double mu,
                                                         const unsigned *__restrict__ xmax_bits, uint8_t *__restrict__ code)
{
    const double xmax = (double)__uint_as_float(*xmax_bits);
    const double inv_den = 1.0 / log1p(mu);
    const float xmax_f = (float)xmax, mu_f = (float)mu, inv_den_f = (float)(mu >= 1.0 ? 1.0 / log2(1.0 + mu) : inv_den);
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long n16 = n / 16;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n16; i += stride) {
        unsigned w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float4 v = reinterpret_cast<const float4 *>(x)[4 * i + q];
            w[q] = code_of(v.x, xmax, mu, inv_den, xmax_f, mu_f, inv_den_f) | (code_of(v.y, xmax, mu, inv_den, xmax_f, mu_f, inv_den_f) << 8) |
                   (code_of(v.z, xmax, mu, inv_den, xmax_f, mu_f, inv_den_f) << 16) | (code_of(v.w, xmax, mu, inv_den, xmax_f, mu_f, inv_den_f) << 24);
        }
        reinterpret_cast<uint4 *>(code)[i] = make_uint4(w[0], w[1], w[2], w[3]);
    }
    for (long long i = n16 * 16 + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += stride)
        code[i] = (uint8_t)code_of(x[i], xmax, mu, inv_den, xmax_f, mu_f, inv_den_f);
}

}  // namespace

extern "C" int mdsm_mulaw_u8(const float *d_x, uint8_t *d_code, int64_t n, double mu, float *d_xmax, void *cuda_stream)
{
    MDSM_REQUIRE(n >= 0 && d_xmax && (n == 0 || (d_x && d_code)), "null argument");
    MDSM_REQUIRE(mu > 0.0, "mu must be > 0");
    MDSM_REQUIRE((uintptr_t)d_x % 16 == 0 && (uintptr_t)d_code % 16 == 0, "buffers must be 16-byte aligned");
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    MDSM_CUDA_TRY(cudaMemsetAsync(d_xmax, 0, sizeof(float), st));
    if (n == 0) return MDSM_OK;
    int dev = 0, nsm = 0;
    MDSM_CUDA_TRY(cudaGetDevice(&dev));
    MDSM_CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const long long want = (n / 4 + 255) / 256 + 1;
    const int grid = (int)(want < (long long)nsm * 16 ? want : (long long)nsm * 16);
    mulaw_max_kernel<<<grid, 256, 0, st>>>(d_x, n, (unsigned *)d_xmax);
    MDSM_CUDA_TRY(cudaGetLastError());
    mulaw_code_kernel<<<grid, 256, 0, st>>>(d_x, n, mu, (const unsigned *)d_xmax, d_code);
    MDSM_CUDA_TRY(cudaGetLastError());
    return MDSM_OK;
}

// ------------------------------------------------------------------ 2 x 16 bit -> 2 x 4 bit (Fig. 5b; reading G-ii)
// code(v) = sign(v) * floor(7 * log1p(mu |v| / Xmax) / log1p(mu) + 0.5) is monotone in |v| and |v| is an integer <= 32768, so
// the whole law is SEVEN integer thresholds: thr[k] = the smallest |v| whose code is >= k.  The paper uses a lookup table of
// logarithms for the same reason.  Three kernels: max |v| (one atomicMax per CTA), the thresholds (seven
// threads, binary search with the oracle's fp64 expression), the coding pass (eight complex samples per thread and step:
// two 128-bit loads, one 64-bit store; code = number of thresholds <= |v|).  9 bytes per complex sample over the two passes.
namespace {

__global__ void __launch_bounds__(256) c4_max_kernel(const int4 *__restrict__ v, long long n4, const int16_t *__restrict__ tail, int ntail,
                                                     int *__restrict__ xmax)
{
    int m = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += stride) {
        const int4 w = v[i];
        const int ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            m = max(m, abs((int)(short)(ww[k] & 0xffff)));
            m = max(m, abs(ww[k] >> 16));
        }
    }
    if (blockIdx.x == 0 && (int)threadIdx.x < ntail) m = max(m, abs((int)tail[threadIdx.x]));
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, s));
    __shared__ int red[8];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < 8; ++i) m = max(m, red[i]);
        atomicMax(xmax, m);
    }
}

__device__ int c4_code_fp64(int a, int xmax, double mu, double den)
{
    if (xmax <= 0 || a <= 0) return 0;
    return (int)floor(7.0 * (log1p(mu * ((double)a / (double)xmax)) / den) + 0.5);
}

__global__ void c4_threshold_kernel(const int *__restrict__ xmax_p, double mu, int *__restrict__ thr /*[8]*/)
{
    const int k = threadIdx.x + 1;                  // 1..7
    const int xmax = *xmax_p;
    const double den = log1p(mu);
    int lo = 1, hi = xmax + 1;                      // smallest a in [1, xmax] with code(a) >= k, xmax + 1 if none
    while (lo < hi) {
        const int mid = lo + (hi - lo) / 2;
        if (c4_code_fp64(mid, xmax, mu, den) >= k) hi = mid;
        else lo = mid + 1;
    }
    thr[k - 1] = lo;
    if (k == 1) thr[7] = 0x7fffffff;
}

__device__ __forceinline__ unsigned c4_nibble(int v, const int (&t)[7])
{
    const int a = abs(v);
    int c = (a >= t[0]) + (a >= t[1]) + (a >= t[2]) + (a >= t[3]) + (a >= t[4]) + (a >= t[5]) + (a >= t[6]);
    c = v < 0 ? -c : c;
    return (unsigned)c & 15u;
}

__global__ void __launch_bounds__(256) c4_code_kernel(const int16_t *__restrict__ volt, long long n, const int *__restrict__ thr,
                                                      uint8_t *__restrict__ packed)
{
    int t[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) t[k] = thr[k];
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long n8 = n / 8;
    const int4 *v4 = reinterpret_cast<const int4 *>(volt);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n8; i += stride) {
        const int4 a = v4[2 * i], b = v4[2 * i + 1];
        const int w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};        // one complex sample per 32-bit word: re low, im high
        unsigned lo = 0, hi = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            lo |= (c4_nibble((int)(short)(w[k] & 0xffff), t) | (c4_nibble(w[k] >> 16, t) << 4)) << (8 * k);
            hi |= (c4_nibble((int)(short)(w[4 + k] & 0xffff), t) | (c4_nibble(w[4 + k] >> 16, t) << 4)) << (8 * k);
        }
        reinterpret_cast<uint2 *>(packed)[i] = make_uint2(lo, hi);
    }
    for (long long i = n8 * 8 + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += stride)
        packed[i] = (uint8_t)(c4_nibble((int)volt[2 * i], t) | (c4_nibble((int)volt[2 * i + 1], t) << 4));
}

}  // namespace

extern "C" int mdsm_mulaw_c4(const int16_t *d_volt, uint8_t *d_packed, int64_t n, double mu, int32_t *d_xmax_thr, void *cuda_stream)
{
    MDSM_REQUIRE(n >= 0 && d_xmax_thr && (n == 0 || (d_volt && d_packed)), "null argument");
    MDSM_REQUIRE(mu > 0.0, "mu must be > 0");
    MDSM_REQUIRE((uintptr_t)d_volt % 16 == 0 && (uintptr_t)d_packed % 16 == 0 && (uintptr_t)d_xmax_thr % 4 == 0, "buffers must be 16-byte aligned");
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    MDSM_CUDA_TRY(cudaMemsetAsync(d_xmax_thr, 0, 9 * sizeof(int32_t), st));
    if (n == 0) return MDSM_OK;
    int dev = 0, nsm = 0;
    MDSM_CUDA_TRY(cudaGetDevice(&dev));
    MDSM_CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const long long n4 = (2 * n) / 8;                                   // int4 = 8 int16 components
    const long long want = (n4 + 255) / 256 + 1;
    const int grid = (int)(want < (long long)nsm * 16 ? want : (long long)nsm * 16);
    c4_max_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const int4 *>(d_volt), n4, d_volt + n4 * 8, (int)(2 * n - n4 * 8), d_xmax_thr);
    MDSM_CUDA_TRY(cudaGetLastError());
    c4_threshold_kernel<<<1, 7, 0, st>>>(d_xmax_thr, mu, d_xmax_thr + 1);
    MDSM_CUDA_TRY(cudaGetLastError());
    c4_code_kernel<<<grid, 256, 0, st>>>(d_volt, n, d_xmax_thr + 1, d_packed);
    MDSM_CUDA_TRY(cudaGetLastError());
    return MDSM_OK;
}
