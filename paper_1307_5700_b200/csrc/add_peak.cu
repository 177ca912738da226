// Register-only add-issue microbenchmark: the measured denominator of the dedispersion
// roofline ("a register-only FADD (and IADD) microbenchmark on all SMs,
// run in the same session").  16 independent accumulators per thread, 8 CTAs of 256 threads per SM.
#include "mdsm_internal.h"

namespace {

constexpr int kAcc = 16;

template <int KIND>
__global__ void __launch_bounds__(256) add_peak_kernel(float *out, const float *in, int iters)
{
    if (KIND == 0) {
        float acc[kAcc], x[4];
        for (int i = 0; i < kAcc; ++i) acc[i] = in[threadIdx.x + i];
        for (int i = 0; i < 4; ++i) x[i] = in[i + 64 + threadIdx.x];
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < kAcc; ++i) asm volatile("add.f32 %0, %0, %1;" : "+f"(acc[i]) : "f"(x[(i + r) & 3]));
        }
        float s = 0;
        for (int i = 0; i < kAcc; ++i) s += acc[i];
        out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    } else if (KIND == 1) {
        unsigned long long acc[kAcc / 2], x[4];
        const unsigned long long *in2 = reinterpret_cast<const unsigned long long *>(in);
        for (int i = 0; i < kAcc / 2; ++i) acc[i] = in2[threadIdx.x + i];
        for (int i = 0; i < 4; ++i) x[i] = in2[i + 64 + threadIdx.x];
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < kAcc / 2; ++i)
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(acc[i]) : "l"(x[(i + r) & 3]));
        }
        unsigned long long s = 0;
        for (int i = 0; i < kAcc / 2; ++i) s ^= acc[i];
        reinterpret_cast<unsigned long long *>(out)[blockIdx.x * blockDim.x + threadIdx.x] = s;
    } else {
        int acc[kAcc], x[4];
        const int *ini = reinterpret_cast<const int *>(in);
        for (int i = 0; i < kAcc; ++i) acc[i] = ini[threadIdx.x + i];
        for (int i = 0; i < 4; ++i) x[i] = ini[i + 64 + threadIdx.x];
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < kAcc; ++i) asm volatile("add.s32 %0, %0, %1;" : "+r"(acc[i]) : "r"(x[(i + r) & 3]));
        }
        int s = 0;
        for (int i = 0; i < kAcc; ++i) s ^= acc[i];
        reinterpret_cast<int *>(out)[blockIdx.x * blockDim.x + threadIdx.x] = s;
    }
}

}  // namespace

extern "C" int mdsm_measure_add_peak(int kind, double *adds_per_s)
{
    MDSM_REQUIRE(adds_per_s && kind >= 0 && kind <= 2, "kind must be 0 (FADD), 1 (FADD2) or 2 (IADD)");
    int dev = 0, nsm = 0;
    MDSM_CUDA_TRY(cudaGetDevice(&dev));
    MDSM_CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const int grid = nsm * 8, iters = 4096;
    float *in = nullptr, *out = nullptr;
    MDSM_CUDA_TRY(cudaMalloc((void **)&in, 1 << 16));
    MDSM_CUDA_TRY(cudaMemset(in, 0, 1 << 16));
    MDSM_CUDA_TRY(cudaMalloc((void **)&out, (size_t)grid * 256 * 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) add_peak_kernel<0><<<grid, 256>>>(out, in, iters);
        else if (kind == 1) add_peak_kernel<1><<<grid, 256>>>(out, in, iters);
        else add_peak_kernel<2><<<grid, 256>>>(out, in, iters);
        cudaEventRecord(e1);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) {
            mdsm_set_error("add peak kernel failed: %s", cudaGetErrorString(e));
            cudaFree(in); cudaFree(out);
            return MDSM_ECUDA;
        }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(in);
    cudaFree(out);
    *adds_per_s = (double)grid * 256.0 * iters * 4.0 * kAcc / (best * 1e-3);
    return MDSM_OK;
}
