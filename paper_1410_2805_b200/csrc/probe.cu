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

// kinds 3-5: a register/shared-memory-only copy of the force kernel's pair loop (T = 2:
// sources as LDS.128 broadcasts, two targets per lane, packed arithmetic, SFU rsqrt), with
// (SEL) the cutoff select FSETP + FSEL and (BAND) the guard-band test VIADDMNMX switched on or
// off.  What the loop's instruction mix can reach with no global memory, no staging, no tails.
template <bool SEL, bool BAND>
__global__ void __launch_bounds__(256) k_probe_mix(int iters, float a, float b, float cut,
                                                   uint32_t lo, float *sink)
{
    __shared__ float4 sh[3][64];
    if (threadIdx.x < 64)
        for (int k = 0; k < 3; ++k)
            sh[k][threadIdx.x] = make_float4(threadIdx.x * 1e-3f + k, 0.5f + k, 0.25f * k, 1.f);
    __syncthreads();
    float2 ax[2], ay[2], az[2];
    float xi[2], yi[2], zi[2];
    for (int t = 0; t < 2; ++t) {
        ax[t] = ay[t] = az[t] = make_float2(0.f, 0.f);
        xi[t] = threadIdx.x * 1e-3f + t;
        yi[t] = a + t;
        zi[t] = b + t;
    }
    const float2 eps2 = make_float2(b, b);
    const float2 n5 = make_float2(a * 1e-7f, a * 1e-7f), n4 = make_float2(a * 1e-5f, a * 1e-5f),
                 n3 = make_float2(a * 1e-4f, a * 1e-4f), n2 = make_float2(a * 1e-3f, a * 1e-3f),
                 n1 = make_float2(a * 1e-2f, a * 1e-2f), n0 = make_float2(a, a);
    uint32_t band = 0xffffffffu;
    for (int it = 0; it < iters; ++it) {
#pragma unroll 2
        for (int g = 0; g < 16; ++g) {
            const float4 X = sh[0][g], Y = sh[1][g], Z = sh[2][g];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const float2 sx2 = h ? make_float2(X.z, X.w) : make_float2(X.x, X.y);
                const float2 sy2 = h ? make_float2(Y.z, Y.w) : make_float2(Y.x, Y.y);
                const float2 sz2 = h ? make_float2(Z.z, Z.w) : make_float2(Z.x, Z.y);
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const float2 dx = __fadd2_rn(sx2, make_float2(-xi[t], -xi[t]));
                    const float2 dy = __fadd2_rn(sy2, make_float2(-yi[t], -yi[t]));
                    const float2 dz = __fadd2_rn(sz2, make_float2(-zi[t], -zi[t]));
                    float2 u = __ffma2_rn(dx, dx, eps2);
                    u = __ffma2_rn(dy, dy, u);
                    u = __ffma2_rn(dz, dz, u);
                    float2 q;
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(q.x) : "f"(u.x));
                    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(q.y) : "f"(u.y));
                    float2 hh = __ffma2_rn(n5, u, n4);
                    hh = __ffma2_rn(hh, u, n3);
                    hh = __ffma2_rn(hh, u, n2);
                    hh = __ffma2_rn(hh, u, n1);
                    hh = __ffma2_rn(hh, u, n0);
                    float2 f = __ffma2_rn(__fmul2_rn(q, q), q, hh);
                    if (SEL) {
                        f.x = (u.x < cut) ? f.x : 0.f;
                        f.y = (u.y < cut) ? f.y : 0.f;
                    }
                    if (BAND) {
                        band = min(band, __float_as_uint(u.x) - lo);
                        band = min(band, __float_as_uint(u.y) - lo);
                    }
                    ax[t] = __ffma2_rn(f, dx, ax[t]);
                    ay[t] = __ffma2_rn(f, dy, ay[t]);
                    az[t] = __ffma2_rn(f, dz, az[t]);
                }
            }
        }
    }
    float s = (band < 16u) ? 1.f : 0.f;
    for (int t = 0; t < 2; ++t) s += ax[t].x + ax[t].y + ay[t].x + ay[t].y + az[t].x + az[t].y;
    if (s == 123.456f) sink[0] = s;
}

__device__ __forceinline__ uint32_t probe_hash(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

// kinds 6-7: 16-byte stores of a coalesced read stream into `dst`: kind 6 sends every element
// to a pseudo-random slot of its own 65 536-element (1 MB) window -- the pattern of a direct
// counting-sort scatter, L2-resident -- kind 7 sends every group of RUN consecutive elements to
// a pseudo-randomly placed run of RUN consecutive slots -- what the staged sort writes.
template <int RUN>
__global__ void __launch_bounds__(256) k_probe_store(int64_t n, const float4 *__restrict__ src,
                                                     float4 *__restrict__ dst)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint32_t win = (uint32_t)(i >> 16), in = (uint32_t)i & 0xffffu;
        // a bijection of the window's run indices (odd multiplier, xor), runs kept whole
        const uint32_t run = in / RUN, lane = in % RUN, nrun = 65536u / RUN;
        const uint32_t prun = ((run * 40503u) ^ (probe_hash(win) & (nrun - 1))) & (nrun - 1);
        dst[((int64_t)win << 16) + prun * RUN + lane] = __ldg(src + i);
    }
}

// kind 8: shared-memory atomics with return on pseudo-random counters (9596 of them);
// kind 9: the same on global memory, one counter per 128-byte line.
template <bool GLOBAL>
__global__ void __launch_bounds__(256) k_probe_atomic(int iters, uint32_t K, uint32_t *ctr,
                                                      uint32_t *sink)
{
    extern __shared__ uint32_t sh[];
    if (!GLOBAL) {
        for (uint32_t i = threadIdx.x; i < K; i += blockDim.x) sh[i] = 0;
        __syncthreads();
    }
    uint32_t acc = 0, h = probe_hash(blockIdx.x * blockDim.x + threadIdx.x + 77u);
    for (int it = 0; it < iters; ++it) {
        h = probe_hash(h + it);
        const uint32_t a = h % K;
        acc += GLOBAL ? atomicAdd(ctr + (size_t)a * 32, 1u) : atomicAdd(&sh[a], 1u);
    }
    if (acc == 0x12345u) sink[0] = acc;
}

}  // namespace haccsr

using namespace haccsr;

extern "C" int haccsr_probe_peak(int kind, int reps, void *cuda_stream, double *ms, double *ops)
{
    if (!ms || !ops || reps < 1 || kind < 0 || kind > 9) return HACCSR_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HACCSR_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HACCSR_ECUDA;
    const int64_t n_store = (int64_t)1 << 25;  // 32 Mi float4 = 512 MiB per buffer
    const uint32_t k_ctr = 9596;
    size_t bytes = 16;
    if (kind == 6 || kind == 7) bytes = 2 * sizeof(float4) * (size_t)n_store;
    if (kind == 9) bytes = sizeof(uint32_t) * 32 * (size_t)k_ctr + 16;
    char *buf = nullptr;
    if (cudaMalloc(&buf, bytes) != cudaSuccess) return HACCSR_ECUDA;
    cudaMemsetAsync(buf, 0, bytes, st);
    float *sink = reinterpret_cast<float *>(buf);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 8, block = 256;
    const int iters = (kind == 2) ? 256 : 1024;
    if (kind == 8)
        cudaFuncSetAttribute(k_probe_atomic<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(k_ctr * 4));
    double best = 1e300;
    for (int r = 0; r < reps + 1; ++r) {  // first repetition is the warm-up
        cudaEventRecord(e0, st);
        switch (kind) {
        case 0: k_probe_ffma<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        case 1: k_probe_ffma2<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        case 2: k_probe_rsqrt<<<grid, block, 0, st>>>(iters, 0.999f, 0.001f, sink); break;
        case 3: k_probe_mix<true, true><<<sms * 2, block, 0, st>>>(iters / 4, 0.37f, 0.1f, 9.1f,
                                                                   0x41119990u, sink); break;
        case 4: k_probe_mix<true, false><<<sms * 2, block, 0, st>>>(iters / 4, 0.37f, 0.1f, 9.1f,
                                                                    0x41119990u, sink); break;
        case 5: k_probe_mix<false, false><<<sms * 2, block, 0, st>>>(iters / 4, 0.37f, 0.1f,
                                                                     9.1f, 0x41119990u, sink);
            break;
        case 6: k_probe_store<1><<<grid, block, 0, st>>>(
                n_store, reinterpret_cast<const float4 *>(buf),
                reinterpret_cast<float4 *>(buf) + n_store); break;
        case 7: k_probe_store<32><<<grid, block, 0, st>>>(
                n_store, reinterpret_cast<const float4 *>(buf),
                reinterpret_cast<float4 *>(buf) + n_store); break;
        case 8: k_probe_atomic<false><<<sms * 4, block, k_ctr * 4, st>>>(
                iters, k_ctr, nullptr, reinterpret_cast<uint32_t *>(buf)); break;
        default: k_probe_atomic<true><<<grid, block, 0, st>>>(
                iters / 8, k_ctr, reinterpret_cast<uint32_t *>(buf) + 4,
                reinterpret_cast<uint32_t *>(buf)); break;
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) {
            cudaFree(buf);
            return HACCSR_ECUDA;
        }
        float t = 0.f;
        cudaEventElapsedTime(&t, e0, e1);
        if (r > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    double total;
    const double threads = (double)grid * block;
    if (kind == 0) total = threads * iters * kInner * kChains;            // FMAs
    else if (kind == 1) total = threads * iters * kInner * kChains * 2;  // FMAs
    else if (kind == 2) total = threads * iters * kInner * kChains;      // rsqrts
    else if (kind <= 5) total = (double)sms * 2 * block * (iters / 4) * 16 * 2 * 2 * 2;  // pairs
    else if (kind <= 7) total = (double)n_store;                          // 16-byte stores
    else if (kind == 8) total = (double)sms * 4 * block * iters;          // atomics
    else total = threads * (iters / 8);                                   // atomics
    *ms = best;
    *ops = total;
    return HACCSR_OK;
}
