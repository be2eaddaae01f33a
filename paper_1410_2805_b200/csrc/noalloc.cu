// noalloc.cu -- hacc_sr_cell_start_noalloc (include/haccsr.h): the chaining mesh's occupancy
// table in one call that allocates nothing.  The per-cell counters live in a
// file-scope __device__ array instead of a caller-provided workspace; everything else (wrap
// rule, cell rule, cell numbering) is what hacc_sr_bin uses (mesh.cuh).
//
// g_na_scratch is a HOST-side stand-in in host code, not a device address: its address on
// each device is looked up once, with that device current, by cudaGetSymbolAddress and that
// pointer is what the kernels get.
#include <cmath>
#include <mutex>

#include "mesh.cuh"

namespace haccsr {

constexpr int kNaMaxNc = HACCSR_NOALLOC_MAX_NC;
constexpr int64_t kNaMaxCells = HACCSR_NOALLOC_MAX_CELLS;
constexpr int kNaMaxDevices = 64;
constexpr int kNaScanThreads = 1024, kNaScanItems = 4;
constexpr int kNaScanTile = kNaScanThreads * kNaScanItems;

static_assert(kNaMaxCells == (int64_t)kNaMaxNc * kNaMaxNc * kNaMaxNc, "limits disagree");

// Particles per cell, 1 MiB.  Shared by every call on the device; holds the last call's
// counts between calls, so a call clears the counters of its own cells first.
static __device__ __align__(256) uint32_t g_na_scratch[kNaMaxCells];

static std::mutex g_na_mutex;
static uint32_t *g_na_ptr[kNaMaxDevices] = {};

// Device address of the scratch array on the CURRENT device (looked up once per device).
static cudaError_t na_scratch(uint32_t **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNaMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_na_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_na_ptr[dev] = static_cast<uint32_t *>(p);
    }
    *out = g_na_ptr[dev];
    return cudaSuccess;
}

// The counters of this call's cells start from zero.
__global__ void __launch_bounds__(256) k_na_clear(uint32_t *__restrict__ scratch, int64_t n_cells)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_cells; i += stride)
        scratch[i] = 0u;
}

// One atomic per particle, after merging the lanes of a warp that hit the same cell (halo
// cores put thousands of consecutive particles in one cell).
__global__ void __launch_bounds__(256) k_na_count(int64_t n, const float *__restrict__ x,
                                                  const float *__restrict__ y,
                                                  const float *__restrict__ z, MeshGeom g,
                                                  uint32_t *__restrict__ count)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    // whole warps stay in the loop together (match_any needs the named lanes present)
    for (int64_t base = i0 - lane; base < n; base += stride) {
        const int64_t i = base + lane;
        const bool live = i < n;
        uint32_t cell = 0xffffffffu;
        if (live) {
            bool bad = false;
            const int cx = cell_coord(wrap_pos(x[i], g.box_l, bad), g);
            const int cy = cell_coord(wrap_pos(y[i], g.box_l, bad), g);
            const int cz = cell_coord(wrap_pos(z[i], g.box_l, bad), g);
            cell = (uint32_t)(cx + g.nc * (cy + g.nc * cz));
        }
        const unsigned peers = __match_any_sync(0xffffffffu, cell);
        if (live && lane == __ffs(peers) - 1) atomicAdd(count + cell, (uint32_t)__popc(peers));
    }
}

// Exclusive scan of at most kNaMaxCells counters by ONE block: 64 tiles of 4096 at most, each
// a warp-shuffle block scan, the running total carried from tile to tile.
__global__ void __launch_bounds__(kNaScanThreads) k_na_scan(const uint32_t *__restrict__ count,
                                                            int64_t n_cells,
                                                            uint32_t *__restrict__ cell_start)
{
    __shared__ uint32_t warp_sum[32];
    __shared__ uint32_t carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0u;
    __syncthreads();
    for (int64_t t0 = 0; t0 < n_cells; t0 += kNaScanTile) {
        uint32_t v[kNaScanItems], sum = 0;
#pragma unroll
        for (int k = 0; k < kNaScanItems; ++k) {
            const int64_t i = t0 + (int64_t)threadIdx.x * kNaScanItems + k;
            v[k] = i < n_cells ? count[i] : 0u;
            sum += v[k];
        }
        uint32_t inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        if (lane == 31) warp_sum[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = warp_sum[lane], winc = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, winc, d);
                if (lane >= d) winc += t;
            }
            warp_sum[lane] = winc - w;   // exclusive over warps
        }
        __syncthreads();
        const uint32_t carry = carry_s;
        uint32_t ex = carry + warp_sum[warp] + (inc - sum);
#pragma unroll
        for (int k = 0; k < kNaScanItems; ++k) {
            const int64_t i = t0 + (int64_t)threadIdx.x * kNaScanItems + k;
            if (i < n_cells) cell_start[i] = ex;
            ex += v[k];
        }
        __syncthreads();                 // everyone has read carry_s and warp_sum
        if (threadIdx.x == kNaScanThreads - 1) carry_s = ex;   // total through this tile
        __syncthreads();
    }
    if (threadIdx.x == 0) cell_start[n_cells] = carry_s;
}

}  // namespace haccsr

using namespace haccsr;

extern "C" int hacc_sr_cell_start_noalloc(int64_t n, const float *x, const float *y,
                                          const float *z, float box_L, int nc,
                                          uint32_t *cell_start, void *cuda_stream)
{
    if (n < 0 || n >= (int64_t(1) << 31) || nc < 4 || !cell_start) return HACCSR_EINVAL;
    if (!(box_L > 0.f) || !std::isfinite(box_L)) return HACCSR_EINVAL;
    if (n > 0 && (!x || !y || !z)) return HACCSR_EINVAL;
    if (nc > kNaMaxNc) return HACCSR_ENOMEM;   // beyond the static scratch array
    const int64_t n_cells = (int64_t)nc * nc * nc;

    uint32_t *scratch = nullptr;
    if (na_scratch(&scratch) != cudaSuccess) return HACCSR_ECUDA;
    int sms = 0, dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HACCSR_ECUDA;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);

    MeshGeom g;
    const double scale = (double)nc / (double)box_L;
    g.box_l = box_L;
    g.scale = (float)scale;
    g.dscale_nc = (double)nc;
    g.dbox_l = (double)box_L;
    g.nc = nc;
    g.exact = ((double)(float)scale == scale) ? 1 : 0;
    g.nz = nc;
    g.cz0 = 0;

    const int cap = sms * 8;
    const int64_t want_clear = (n_cells + 255) / 256;
    k_na_clear<<<(int)(want_clear < cap ? want_clear : cap), 256, 0, st>>>(scratch, n_cells);
    if (n > 0) {
        const int64_t want = (n + 255) / 256;
        k_na_count<<<(int)(want < cap ? want : cap), 256, 0, st>>>(n, x, y, z, g, scratch);
    }
    k_na_scan<<<1, kNaScanThreads, 0, st>>>(scratch, n_cells, cell_start);
    return cudaGetLastError() == cudaSuccess ? HACCSR_OK : HACCSR_ECUDA;
}
