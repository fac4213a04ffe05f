// nep_peak.cu -- measurement aid: the FP32 FMA rate this GPU reaches on a register-resident loop, so that bench.py can print the
// "alu" roofline's denominator as MEASURED in the same run, next to the derived SMs x 128 lanes x 2 x clock figure.
// Not part of the step: nothing in the NEP path calls it.
#include <cuda_runtime.h>

#include <string>

#include "nep_internal.h"

namespace nep {

// sink for the result of the FMA chains (never read; keeps the compiler from removing the loop)
static __device__ float g_peak_sink;

// 32 independent accumulators per thread (nvcc 12.9 emits 256 scalar FFMA per trip of the loop: cuobjdump -sass), far more
// independent chains than the 4-cycle FMA latency needs at 16 warps per scheduler: the loop is bound by the FMA pipe alone.
__global__ void __launch_bounds__(256) k_fp32_peak(int iters, float a, float b)
{
    float2 x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = make_float2(threadIdx.x * 1e-3f + i, blockIdx.x * 1e-3f - i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int i = 0; i < 16; ++i) { x[i].x = fmaf(x[i].x, a, b); x[i].y = fmaf(x[i].y, a, b); }
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i].x + x[i].y;
    if (s == 123.456f) g_peak_sink = s;
}

}  // namespace nep

extern "C" int nep_measure_fp32_peak(void* cuda_stream, double* tflops)
{
    using namespace nep;
    if (!tflops) return fail(nullptr, NEP_EINVAL, "nep_measure_fp32_peak: tflops is NULL");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t a = nullptr, b = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    const int iters = 4096, blocks = sms * 8;              // 2048 threads per SM
    double best_ms = 1e30;
    for (int rep = 0; rep < 6 && e == cudaSuccess; ++rep) {   // the first launches warm the clocks up; the best of the rest counts
        cudaEventRecord(a, st);
        k_fp32_peak<<<blocks, 256, 0, st>>>(iters, 0.999f, 1e-3f);
        cudaEventRecord(b, st);
        e = cudaEventSynchronize(b);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
        if (e == cudaSuccess && rep >= 2 && ms < best_ms) best_ms = ms;
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    if (e != cudaSuccess) return fail(nullptr, NEP_ECUDA, std::string("nep_measure_fp32_peak: ") + cudaGetErrorString(e));
    const double flops = 2.0 * 32.0 * 8.0 * iters * 256.0 * blocks;   // 2 flops x 32 FMAs x 8 rounds x iterations x threads
    *tflops = flops / (best_ms * 1e-3) / 1e12;
    return NEP_OK;
}
