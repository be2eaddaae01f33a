// shard.cu -- particle overloading (section 2.2): "particles close to the
// boundaries of their domain are replicated" in the neighbouring domains as passive
// particles, after which the short-range step needs no communication.  With slabs of whole
// chaining-mesh layers the overloaded skin of a domain is one cell layer (>= r_max wide) on
// each side: this file selects a layer's particles into a contiguous float4 buffer (the
// message to the neighbouring rank) and appends received records to the SoA arrays.
#include "ctx.h"
#include "mesh.cuh"

namespace haccsr {

// Append {x, y, z, m} of every particle whose (wrapped) position lies in global cell layer
// `layer` to out[0 .. capacity); *count receives the number found even beyond capacity.
// One atomic per warp (ballot + popc), so the records of a warp stay together.
__global__ void __launch_bounds__(256) k_pack_layer(int64_t n, const float *__restrict__ x,
                                                    const float *__restrict__ y,
                                                    const float *__restrict__ z,
                                                    const float *__restrict__ mass, MeshGeom g,
                                                    int layer, float4 *__restrict__ out,
                                                    uint32_t capacity, uint32_t *count,
                                                    DeviceStats *stats)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    bool bad = false;
    const int64_t n_round = (n + 31) & ~(int64_t)31;  // whole warps iterate together
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += stride) {
        bool take = false;
        float pz = 0.f;
        if (i < n) {
            pz = wrap_pos(__ldg(z + i), g.box_l, bad);
            take = cell_coord(pz, g) == layer;
        }
        const unsigned m = __ballot_sync(0xffffffffu, take);
        if (m == 0) continue;
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(count, (uint32_t)__popc(m));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (take) {
            const uint32_t slot = base + (uint32_t)__popc(m & ((1u << lane) - 1u));
            if (slot < capacity)
                out[slot] = make_float4(wrap_pos(__ldg(x + i), g.box_l, bad),
                                        wrap_pos(__ldg(y + i), g.box_l, bad), pz,
                                        mass ? __ldg(mass + i) : 1.f);
        }
    }
    if (bad) stats->error_flag = HACCSR_EDATA;
}

__global__ void __launch_bounds__(256) k_unpack(int64_t n, const float4 *__restrict__ in,
                                                float *__restrict__ x, float *__restrict__ y,
                                                float *__restrict__ z, float *__restrict__ mass)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float4 r = __ldg(in + i);
        x[i] = r.x;
        y[i] = r.y;
        z[i] = r.z;
        if (mass) mass[i] = r.w;
    }
}

static inline int stream_grid(const haccsr_ctx *c, int64_t n)
{
    const int64_t want = (n + 255) / 256, cap = (int64_t)c->n_sms * 16;
    return (int)(want < cap ? (want > 0 ? want : 1) : cap);
}

cudaError_t launch_pack_layer(haccsr_ctx *c, int64_t n, const float *x, const float *y,
                              const float *z, const float *mass, int layer, float4 *out,
                              uint32_t capacity, uint32_t *count)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(count, 0, sizeof(uint32_t), c->stream))) return e;
    if (n > 0)
        k_pack_layer<<<stream_grid(c, n), 256, 0, c->stream>>>(n, x, y, z, mass, geom_of(c),
                                                               layer, out, capacity, count,
                                                               c->stats);
    return cudaGetLastError();
}

cudaError_t launch_unpack(haccsr_ctx *c, int64_t n, const float4 *in, float *x, float *y,
                          float *z, float *mass)
{
    if (n > 0) k_unpack<<<stream_grid(c, n), 256, 0, c->stream>>>(n, in, x, y, z, mass);
    return cudaGetLastError();
}

}  // namespace haccsr
