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

// kind 3: the force kernel's instruction mix per source pair without memory:
// 8.5 packed FP32 ops + 2 rsqrt + 2 compare/select + 2 integer band tests.
__global__ void __launch_bounds__(256) k_probe_mix(int iters, float a, float b, float *sink)
{
    float2 acc[4], x[4];
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    bool near = false;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        acc[k] = make_float2(0.f, 0.f);
        x[k] = make_float2((float)(threadIdx.x + k) * 1e-3f, (float)k * 1e-3f);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 16; ++r)
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                float2 dx = __fadd2_rn(x[k], a2), dy = __fadd2_rn(x[k], b2),
                       dz = __fadd2_rn(x[(k + 1) & 3], b2);
                float2 u = __ffma2_rn(dx, dx, b2);
                u = __ffma2_rn(dy, dy, u);
                u = __ffma2_rn(dz, dz, u);
                float2 q;
                asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(q.x) : "f"(u.x));
                asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(q.y) : "f"(u.y));
                float2 h = __ffma2_rn(a2, u, b2);
                h = __ffma2_rn(h, u, a2);
                h = __ffma2_rn(h, u, b2);
                h = __ffma2_rn(h, u, a2);
                h = __ffma2_rn(h, u, b2);
                float2 f = __ffma2_rn(__fmul2_rn(q, q), q, h);
                f.x = (u.x < a) ? f.x : 0.f;
                f.y = (u.y < a) ? f.y : 0.f;
                near |= (__float_as_uint(u.x) - 0x41100000u) < 16u;
                near |= (__float_as_uint(u.y) - 0x41100000u) < 16u;
                acc[k] = __ffma2_rn(f, dx, acc[k]);
                x[k] = __ffma2_rn(f, dy, x[k]);
                acc[(k + 2) & 3] = __ffma2_rn(f, dz, acc[(k + 2) & 3]);
            }
    }
    float s = near ? 1.f : 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) s += acc[k].x + acc[k].y + x[k].x + x[k].y;
    if (s == 123.456f) sink[0] = s;
}

}  // namespace haccsr

using namespace haccsr;

extern "C" int haccsr_probe_peak(int kind, int reps, void *cuda_stream, double *ms, double *ops)
{
    if (!ms || !ops || reps < 1 || kind < 0 || kind > 3) return HACCSR_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HACCSR_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HACCSR_ECUDA;
    float *sink = nullptr;
    if (cudaMalloc(&sink, 4) != cudaSuccess) return HACCSR_ECUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 8, block = 256;
    const int iters = (kind == 2) ? 256 : 1024;
    double best = 1e300;
    for (int r = 0; r < reps + 1; ++r) {  // first repetition is the warm-up
        cudaEventRecord(e0, st);
        switch (kind) {
        case 0: k_probe_ffma<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        case 1: k_probe_ffma2<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        case 2: k_probe_rsqrt<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        default: k_probe_mix<<<grid, block, 0, st>>>(iters / 4, 9.1f, 0.1f, sink); break;
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) {
            cudaFree(sink);
            return HACCSR_ECUDA;
        }
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        if (r > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    const double threads = (double)grid * block;
    double per_thread;
    if (kind == 0) per_thread = (double)iters * kInner * kChains;            // FMAs
    else if (kind == 1) per_thread = (double)iters * kInner * kChains * 2;  // FMAs
    else if (kind == 2) per_thread = (double)iters * kInner * kChains;      // rsqrts
    else per_thread = (double)(iters / 4) * 16 * 4 * 2;                     // source pairs
    *ms = best;
    *ops = threads * per_thread;
    return HACCSR_OK;
}
