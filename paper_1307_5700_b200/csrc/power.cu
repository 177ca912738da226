// Power calculation (the first GPU stage of the paper's pipeline):
//   power[i] = re[i]^2 + im[i]^2 from interleaved 16-bit complex voltages, as float.
// HBM-bound: 4 bytes in + 4 bytes out per sample; 128-bit loads (4 samples) and stores.  The sum is formed exactly in
// 64-bit integers (it can reach 2^31) and rounded once to float, like the oracle.
#include "mdsm_internal.h"

namespace {

__device__ __forceinline__ float power_of(uint32_t w)
{
    const long long re = (short)(w & 0xffffu), im = (short)(w >> 16);
    return __ll2float_rn(re * re + im * im);
}

__global__ void __launch_bounds__(256) power_i16_kernel(const uint32_t *__restrict__ volt, float *__restrict__ power, long long n)
{
    const long long n4 = n / 4;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n4; i += stride) {
        const uint4 v = reinterpret_cast<const uint4 *>(volt)[i];
        float4 o;
        o.x = power_of(v.x); o.y = power_of(v.y); o.z = power_of(v.z); o.w = power_of(v.w);
        reinterpret_cast<float4 *>(power)[i] = o;
    }
    for (long long i = n4 * 4 + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += stride) power[i] = power_of(volt[i]);
}

}  // namespace

extern "C" int mdsm_power_i16(const int16_t *d_volt, float *d_power, int64_t n, void *cuda_stream)
{
    MDSM_REQUIRE(n >= 0 && (n == 0 || (d_volt && d_power)), "null argument");
    MDSM_REQUIRE((uintptr_t)d_volt % 16 == 0 && (uintptr_t)d_power % 16 == 0, "buffers must be 16-byte aligned");
    if (n == 0) return MDSM_OK;
    int dev = 0, nsm = 0;
    MDSM_CUDA_TRY(cudaGetDevice(&dev));
    MDSM_CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const long long want = (n / 4 + 255) / 256 + 1;
    const int grid = (int)(want < (long long)nsm * 16 ? want : (long long)nsm * 16);
    power_i16_kernel<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>((const uint32_t *)d_volt, d_power, n);
    MDSM_CUDA_TRY(cudaGetLastError());
    return MDSM_OK;
}
