// probe.cu -- register-only peak probes for the roofline denominators bench.py reports.
// Not part of the method: they measure what the FP32 FMA pipe and the SFU of this GPU
// sustain at the clocks the force kernel actually sees.
#include "ctx.h"

namespace haccsr {

constexpr int kChains = 8;
constexpr int kInner = 64;

// kind 0: scalar FFMA, kChains independent chains per thread
__global__ void __launch_bounds__(256) k_probe_ffma(int iters, float a, float b, float *sink)
{
    float v[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) v[k] = (float)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kInner; ++r)
#pragma unroll
            for (int k = 0; k < kChains; ++k) v[k] = __fmaf_rn(v[k], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += v[k];
    if (s == 123.456f) sink[0] = s;
}

// kind 1: packed fma.rn.f32x2
__global__ void __launch_bounds__(256) k_probe_ffma2(int iters, float a, float b, float *sink)
{
    float2 v[kChains];
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll
    for (int k = 0; k < kChains; ++k) v[k] = make_float2((float)(threadIdx.x + k), (float)k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kInner; ++r)
#pragma unroll
            for (int k = 0; k < kChains; ++k) v[k] = __ffma2_rn(v[k], a2, b2);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += v[k].x + v[k].y;
    if (s == 123.456f) sink[0] = s;
}

// kind 2: MUFU.RSQ
__global__ void __launch_bounds__(256) k_probe_rsqrt(int iters, float a, float b, float *sink)
{
    float v[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) v[k] = 1.f + (float)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kInner; ++r)
#pragma unroll
            for (int k = 0; k < kChains; ++k)
                asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(v[k]));
    }
    float s = a + b;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += v[k];
    if (s == 123.456f) sink[0] = s;
}

__device__ float g_probe_sink;  // never written in practice (the kernels' results are unused)

}  // namespace haccsr

using namespace haccsr;

// See include/haccsr.h.  No allocation: the kernels are register-only and their sink is a
// __device__ variable of the library.
extern "C" int haccsr_probe_peak(int kind, int reps, void *cuda_stream, double *ms, double *ops)
{
    if (!ms || !ops || reps < 1 || kind < 0 || kind > 2) return HACCSR_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HACCSR_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HACCSR_ECUDA;
    float *sink = nullptr;
    if (cudaGetSymbolAddress(reinterpret_cast<void **>(&sink), g_probe_sink) != cudaSuccess)
        return HACCSR_ECUDA;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess) return HACCSR_ECUDA;
    if (cudaEventCreate(&e1) != cudaSuccess) {
        cudaEventDestroy(e0);
        return HACCSR_ECUDA;
    }
    const int grid = sms * 8, block = 256;
    const int iters = (kind == 2) ? 256 : 1024;
    double best = 1e300;
    int status = HACCSR_OK;
    for (int r = 0; r < reps + 1; ++r) {  // first repetition is the warm-up
        cudaEventRecord(e0, st);
        switch (kind) {
        case 0: k_probe_ffma<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        case 1: k_probe_ffma2<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        default: k_probe_rsqrt<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) {
            status = HACCSR_ECUDA;
            break;
        }
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        if (r > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (status != HACCSR_OK) return status;
    const double threads = (double)grid * block;
    // kind 0: FMAs, kind 1: FMAs (two per packed instruction), kind 2: rsqrts
    *ops = threads * iters * kInner * kChains * (kind == 1 ? 2.0 : 1.0);
    *ms = best;
    return HACCSR_OK;
}
