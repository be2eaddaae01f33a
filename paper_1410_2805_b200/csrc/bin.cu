// bin.cu -- hacc_sr_bin: the chaining-mesh build = the counting sort
// of sort.cu followed by the force kernel's work list built here ("work queue"
// idea); the exclusive scan both use; the elementwise kick / drift maps.
//
// See DESIGN.md section 6 for bytes per particle and measurements.
#include <math_constants.h>

#include <algorithm>
#include <cstddef>

#include "ctx.h"
#include "mesh.cuh"

namespace haccsr {

// ---------------------------------------------------------------------------------------
// exclusive scan of uint32 (three passes; n <= kScanTile^2)
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t &total)
{
    __shared__ uint32_t warp_sums[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t w = (lane < (blockDim.x >> 5)) ? warp_sums[lane] : 0u;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, w, d);
            if (lane >= d) w += t;
        }
        warp_sums[lane] = w;
    }
    __syncthreads();
    uint32_t base = wid ? warp_sums[wid - 1] : 0u;
    total = warp_sums[(blockDim.x >> 5) - 1];
    __syncthreads();
    return base + inc - v;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_reduce(const uint32_t *__restrict__ in,
                                                            int64_t n,
                                                            uint32_t *__restrict__ block_sums)
{
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < n) s += in[base + k];
    uint32_t total;
    block_exclusive_scan(s, total);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_blocks(uint32_t *block_sums, int n_blocks)
{
    // one block walks the block sums in chunks of kScanTile with a running carry
    // (2 nc^3 work-list counters at nc = 256 make 16 384 block sums)
    uint32_t carry = 0;
    for (int chunk = 0; chunk < n_blocks; chunk += kScanTile) {
        const int base = chunk + threadIdx.x * kScanItems;
        uint32_t v[kScanItems], s = 0;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            v[k] = (base + k < n_blocks) ? block_sums[base + k] : 0u;
            s += v[k];
        }
        uint32_t total;
        uint32_t ex = block_exclusive_scan(s, total) + carry;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            if (base + k < n_blocks) block_sums[base + k] = ex;
            ex += v[k];
        }
        carry += total;
    }
    if (threadIdx.x == 0) block_sums[n_blocks] = carry;
}

// out[i] = exclusive prefix; out[n] = grand total; optional copy (a set of write cursors).
// `copy` may alias `in` (each thread reads its elements before it writes them).
__global__ void __launch_bounds__(kScanBlock) k_scan_apply(const uint32_t *in, int64_t n,
                                                           const uint32_t *__restrict__ block_sums,
                                                           uint32_t *__restrict__ out,
                                                           uint32_t *copy, int n_blocks)
{
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0u;
        s += v[k];
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(s, total) + block_sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) {
            out[base + k] = ex;
            if (copy) copy[base + k] = ex;
        }
        ex += v[k];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = block_sums[n_blocks];
}

// n <= kScanTile: the whole scan in one block, one launch instead of three (small meshes are
// bound by the number of launches).
__global__ void __launch_bounds__(kScanBlock) k_scan_small(const uint32_t *in, int64_t n,
                                                           uint32_t *__restrict__ out,
                                                           uint32_t *copy)
{
    const int64_t base = (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0u;
        s += v[k];
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(s, total);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) {
            out[base + k] = ex;
            if (copy) copy[base + k] = ex;
        }
        ex += v[k];
    }
    if (threadIdx.x == 0) out[n] = total;
}

cudaError_t scan_u32(haccsr_ctx *c, const uint32_t *in, int64_t n, uint32_t *out,
                            uint32_t *copy)
{
    if (n <= kScanTile) {
        k_scan_small<<<1, kScanBlock, 0, c->stream>>>(in, n, out, copy);
        return cudaGetLastError();
    }
    int n_blocks = (int)((n + kScanTile - 1) / kScanTile);
    k_scan_reduce<<<n_blocks, kScanBlock, 0, c->stream>>>(in, n, c->scan_blocks);
    k_scan_blocks<<<1, kScanBlock, 0, c->stream>>>(c->scan_blocks, n_blocks);
    k_scan_apply<<<n_blocks, kScanBlock, 0, c->stream>>>(in, n, c->scan_blocks, out, copy,
                                                         n_blocks);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// work list
// ---------------------------------------------------------------------------------------
// S_c = particles of the 27 neighbour cells of cell c.  In an overloaded slab (nz < nc) the
// first and last layer of the window hold passive particles: sources only, S_c = 0, no items
// ("passive particles near the outer edge get no short-range force").
// `mid` (may be NULL): multi-level time stepping -- the targets of cell c are its first
// mid[c] - cs[c] particles, those of the level being kicked.
// One block = kCsRows consecutive y rows of one layer, one thread per cx (looped for nc > 256).
// The counts of the (kCsRows + 2) x 3 neighbouring rows are loaded into shared memory once
// per z offset and every thread sums its column: 3.75 row loads per output row instead of the
// 18 loads per cell of the cell-by-cell formulation, which was bound by L2 bandwidth.
constexpr int kCsRows = 8;

__global__ void __launch_bounds__(256) k_cell_sources(const uint32_t *__restrict__ cs, int nc,
                                                      int nz, int64_t n_cells,
                                                      const uint32_t *__restrict__ mid,
                                                      uint32_t *__restrict__ cell_sources,
                                                      DeviceStats *stats)
{
    __shared__ uint32_t cnt[kCsRows + 2][kMaxNc + 2];  // [row][1 + cx], x-periodic borders
    const int tiles_y = (nc + kCsRows - 1) / kCsRows;
    const int lz = blockIdx.x / tiles_y, cy0 = (blockIdx.x % tiles_y) * kCsRows;
    const bool slab = nz < nc;
    const bool passive = slab && (lz == 0 || lz == nz - 1);
    unsigned long long work = 0;
    uint32_t nmax = 0;
    for (int cx0 = 0; cx0 < nc; cx0 += blockDim.x) {   // one trip unless nc > 256
        const int cx = cx0 + (int)threadIdx.x;
        uint32_t a[kCsRows + 2];
#pragma unroll
        for (int j = 0; j < kCsRows + 2; ++j) a[j] = 0;
        if (!passive) {
            for (int oz = -1; oz <= 1; ++oz) {
                int qz = lz + oz;            // a slab's active layers have both z neighbours
                if (!slab) {                 // inside the window; the whole box wraps
                    qz += (qz < 0) ? nc : 0;
                    qz -= (qz >= nc) ? nc : 0;
                }
                __syncthreads();
                // all (row, x) pairs in one strided loop: on a small mesh the ten rows' loads
                // are in flight together instead of one dependent round trip per row
                for (int e = threadIdx.x; e < (kCsRows + 2) * nc; e += blockDim.x) {
                    const int j = e / nc, x = e - j * nc;
                    int qy = cy0 - 1 + j;
                    qy += (qy < 0) ? nc : 0;
                    qy -= (qy >= nc) ? nc : 0;
                    qy -= (qy >= nc) ? nc : 0;   // rows past the mesh of the last tile wrap twice
                    const uint32_t *row = cs + (size_t)nc * (size_t)(qy + nc * qz);
                    const uint32_t v = row[x + 1] - row[x];
                    cnt[j][1 + x] = v;
                    if (x == 0) cnt[j][nc + 1] = v;        // periodic borders
                    if (x == nc - 1) cnt[j][0] = v;
                }
                __syncthreads();
                if (cx < nc)
#pragma unroll
                    for (int j = 0; j < kCsRows + 2; ++j)
                        a[j] += cnt[j][cx] + cnt[j][cx + 1] + cnt[j][cx + 2];
            }
        }
        if (cx < nc)
#pragma unroll
            for (int j = 0; j < kCsRows; ++j) {
                const int cy = cy0 + j;
                if (cy >= nc) break;
                const size_t c = (size_t)cx + (size_t)nc * (size_t)(cy + nc * lz);
                uint32_t n_c = passive ? 0u : (mid ? mid[c] : cs[c + 1]) - cs[c];  // targets
                const uint32_t sc = n_c ? a[j] + a[j + 1] + a[j + 2] : 0u;
                cell_sources[c] = sc;
                work += (unsigned long long)n_c * sc;
                nmax = max(nmax, n_c);
            }
    }
    // block reduce
    __shared__ unsigned long long sw[8];
    __shared__ uint32_t sm[8];
#pragma unroll
    for (int d = 16; d; d >>= 1) {
        work += __shfl_xor_sync(0xffffffffu, work, d);
        nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, d));
    }
    if ((threadIdx.x & 31) == 0) {
        sw[threadIdx.x >> 5] = work;
        sm[threadIdx.x >> 5] = nmax;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) {
            work += sw[k];
            nmax = max(nmax, sm[k]);
        }
        if (work) atomicAdd(&stats->n_eval, work);
        if (nmax) atomicMax(&stats->max_cell_count, nmax);
    }
}

__device__ __forceinline__ uint32_t sources_per_split_of(unsigned long long n_eval)
{
    unsigned long long per = (n_eval / kTargetItems + kChunkTargets - 1) / kChunkTargets;
    // small problems (configs[0]: 1600 items for 2368 warps) are cut finer so that every warp
    // of the chip has an item: below 2^31 candidate pairs a source chunk may be 256 long
    // and from 2^34 candidate pairs on a chunk is at least 2048 long: a split item ends in six
    // scattered atomics per target, and with enough work per warp the finer balance no longer
    // pays for them (measured: configs[2]/[4] -1 % at 2048, configs[1] +1 %; 512 costs +15 %)
    const unsigned long long floor_ = (n_eval < (1ull << 31))   ? kSmallSplitSources
                                      : (n_eval < (1ull << 34)) ? kMinSplitSources
                                                                : kLargeSplitSources;
    if (per < floor_) per = floor_;
    if (per > 0x7fffff00ull) per = 0x7fffff00ull;
    return (uint32_t)((per + 63) & ~63ull);  // multiple of the source tile
}

// Target chunks of a cell with n_c particles (force.cu: an item with 32 T targets costs T
// passes over its sources, and a T = 1 item with <= 16 / 8 targets runs 2 / 4 copies of them
// and costs half / a quarter of a pass):
//   full chunks of kChunkTargets, then the rest R = 32 q + r as one 32q-target chunk (T = q,
//   every lane busy) and the tail r: one chunk, or 16 + (r - 16) when 17 <= r <= 24.
// So 40 particles cost 1 + 1/4 passes instead of the 2 of a half-empty T = 2 item.  Measured
// against uniform 128-target chunking: configs[3] +0.4 %, configs[1] +1 %, configs[0] +60 %,
// configs[2]/[4] -0.5 % (more items); keeping tails of more than 16 merged was worse.
__device__ __forceinline__ uint32_t n_target_chunks(uint32_t n_c)
{
    const uint32_t full = n_c / (uint32_t)kChunkTargets, rest = n_c % (uint32_t)kChunkTargets;
    const uint32_t q = rest / 32u, r = rest % 32u;
    return full + (q ? 1u : 0u) + (r ? ((r > 16u && r <= 24u) ? 2u : 1u) : 0u);
}

// How many of those chunks have at most 32 targets (T = 1 items): they are the LAST chunks of
// the cell (the 32-target chunk when q == 1, then the tail).  They are listed in the second
// part of the work list, which k_force_sparse walks.
__device__ __forceinline__ uint32_t n_t1_chunks(uint32_t n_c)
{
    const uint32_t rest = n_c % (uint32_t)kChunkTargets;
    const uint32_t q = rest / 32u, r = rest % 32u;
    return (q == 1u ? 1u : 0u) + (r ? ((r > 16u && r <= 24u) ? 2u : 1u) : 0u);
}

__device__ __forceinline__ void target_chunk(uint32_t n_c, uint32_t ch, uint32_t &t0,
                                             uint32_t &nt)
{
    const uint32_t full = n_c / (uint32_t)kChunkTargets, rest = n_c % (uint32_t)kChunkTargets;
    if (ch < full) {
        t0 = ch * (uint32_t)kChunkTargets;
        nt = (uint32_t)kChunkTargets;
        return;
    }
    const uint32_t q = rest / 32u, r = rest % 32u;
    uint32_t j = ch - full;
    t0 = full * (uint32_t)kChunkTargets;
    if (q) {
        if (j == 0) {
            nt = 32u * q;
            return;
        }
        t0 += 32u * q;
        --j;
    }
    if (r > 16u && r <= 24u) {
        nt = j ? r - 16u : 16u;
        t0 += j ? 16u : 0u;
    } else {
        nt = r;
    }
}

__device__ __forceinline__ void cell_items(uint32_t n_c, uint32_t s_c, uint32_t sps,
                                           uint32_t &chunks, uint32_t &splits)
{
    chunks = n_target_chunks(n_c);
    splits = (s_c + sps - 1) / sps;
}

__global__ void __launch_bounds__(256) k_item_count(const uint32_t *__restrict__ cs,
                                                    const uint32_t *__restrict__ cell_sources,
                                                    const uint32_t *__restrict__ mid,
                                                    int64_t n_cells,
                                                    uint32_t *__restrict__ item_count,
                                                    DeviceStats *stats)
{
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t sps = sources_per_split_of(stats->n_eval);
    if (c == 0) stats->sources_per_split = sps;
    if (c >= n_cells) return;
    uint32_t n_c = (mid ? mid[c] : cs[c + 1]) - cs[c], chunks, splits;
    cell_items(n_c, cell_sources[c], sps, chunks, splits);
    uint32_t items = chunks * splits;
    const uint32_t t1 = n_t1_chunks(n_c) * splits;
    item_count[c] = items - t1;          // items of 33..128 targets come first in the list
    item_count[n_cells + c] = t1;        // then every cell's items of at most 32 targets
    if (splits > 1) atomicAdd(&stats->n_split_items, items);
}

// The items of cell c (one call per thread, whole warps together: small cells are emitted by
// their own lane, big ones by the warp).  item_start may point to shared or global memory.
__device__ __forceinline__ void emit_cell_items(int64_t c, const uint32_t *__restrict__ cs,
                                                const uint32_t *__restrict__ cell_sources,
                                                const uint32_t *item_start,
                                                const uint32_t *__restrict__ mid, int64_t n_cells,
                                                int64_t max_items, WorkItem *__restrict__ items,
                                                DeviceStats *stats)
{
    const int lane = threadIdx.x & 31;
    const uint32_t sps = stats->sources_per_split;
    uint32_t n_c = 0, s_c = 0, chunks = 0, splits = 0, first = 0, first1 = 0;
    if (c < n_cells) {
        n_c = (mid ? mid[c] : cs[c + 1]) - cs[c];
        s_c = cell_sources[c];
        cell_items(n_c, s_c, sps, chunks, splits);
        first = item_start[c];             // the cell's items of more than 32 targets
        first1 = item_start[n_cells + c];  // ... and of at most 32 (its last chunks)
    }
    if (c == 0) {
        uint32_t total = item_start[2 * n_cells];
        stats->n_items = (total > (uint32_t)max_items) ? 0u : total;
        stats->n_dense_items = (total > (uint32_t)max_items) ? 0u : item_start[n_cells];
        if (total > (uint32_t)max_items) stats->error_flag = HACCSR_ENOMEM;
    }
    const uint32_t n_it = chunks * splits;
    auto emit = [&](uint32_t cell, uint32_t nn, uint32_t spl, uint32_t base0, uint32_t base1,
                    uint32_t k) {
        uint32_t ch = k / spl, sp = k - ch * spl;
        uint32_t t0, nt;
        target_chunk(nn, ch, t0, nt);
        const uint32_t n_big = (n_target_chunks(nn) - n_t1_chunks(nn)) * spl;
        const uint32_t base = (k < n_big) ? base0 : base1 - n_big;
        WorkItem w;
        w.cell = cell;
        w.t_begin = t0;
        w.s_begin = sp * sps;
        w.packed = ((nt - 1u) << 24) | (spl > 1 ? (1u << 23) : 0u);
        if ((int64_t)base + k < max_items) items[base + k] = w;
    };
    const bool big = n_it > 32u;
    if (!big)
        for (uint32_t k = 0; k < n_it; ++k) emit((uint32_t)c, n_c, splits, first, first1, k);
    unsigned mask = __ballot_sync(0xffffffffu, big);
    while (mask) {
        int src = __ffs(mask) - 1;
        mask &= mask - 1;
        uint32_t b_cell = (uint32_t)__shfl_sync(0xffffffffu, (uint32_t)c, src);
        uint32_t b_n = __shfl_sync(0xffffffffu, n_c, src);
        uint32_t b_spl = __shfl_sync(0xffffffffu, splits, src);
        uint32_t b_first = __shfl_sync(0xffffffffu, first, src);
        uint32_t b_first1 = __shfl_sync(0xffffffffu, first1, src);
        uint32_t b_nit = __shfl_sync(0xffffffffu, n_it, src);
        for (uint32_t k = lane; k < b_nit; k += 32)
            emit(b_cell, b_n, b_spl, b_first, b_first1, k);
    }
}

__global__ void __launch_bounds__(256) k_emit_items(const uint32_t *__restrict__ cs,
                                                    const uint32_t *__restrict__ cell_sources,
                                                    const uint32_t *__restrict__ item_start,
                                                    const uint32_t *__restrict__ mid,
                                                    int64_t n_cells, int64_t max_items,
                                                    WorkItem *__restrict__ items,
                                                    DeviceStats *stats)
{
    emit_cell_items((int64_t)blockIdx.x * blockDim.x + threadIdx.x, cs, cell_sources, item_start,
                    mid, n_cells, max_items, items, stats);
}

// Meshes of at most kSmallCells cells: item counts, their scan and the emission in ONE block
// (three launches fewer; small problems are bound by the number of launches).
constexpr int kSmallCells = (kScanTile - 1) / 2;

__global__ void __launch_bounds__(kScanBlock) k_items_small(const uint32_t *__restrict__ cs,
                                                            const uint32_t *__restrict__ cell_sources,
                                                            const uint32_t *__restrict__ mid,
                                                            int64_t n_cells, int64_t max_items,
                                                            WorkItem *__restrict__ items,
                                                            DeviceStats *stats)
{
    __shared__ uint32_t count[kScanTile];
    __shared__ uint32_t start[kScanTile + 1];
    __shared__ uint32_t n_split;
    const uint32_t sps = sources_per_split_of(stats->n_eval);
    if (threadIdx.x == 0) n_split = 0;
    for (int i = threadIdx.x; i < kScanTile; i += kScanBlock) count[i] = 0;
    __syncthreads();
    for (int64_t c = threadIdx.x; c < n_cells; c += kScanBlock) {
        uint32_t n_c = (mid ? mid[c] : cs[c + 1]) - cs[c], chunks, splits;
        cell_items(n_c, cell_sources[c], sps, chunks, splits);
        const uint32_t t1 = n_t1_chunks(n_c) * splits;
        count[c] = chunks * splits - t1;
        count[n_cells + c] = t1;
        if (splits > 1) atomicAdd(&n_split, chunks * splits);
    }
    __syncthreads();
    uint32_t v[kScanItems], sum = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = count[threadIdx.x * kScanItems + k];
        sum += v[k];
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan(sum, total);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        start[threadIdx.x * kScanItems + k] = ex;
        ex += v[k];
    }
    if (threadIdx.x == 0) {
        start[kScanTile] = total;
        stats->sources_per_split = sps;
        stats->n_split_items = n_split;
    }
    __syncthreads();
    // entries past 2 n_cells are zero, so start[2 n_cells] is the grand total
    const int64_t rounded = (n_cells + 31) & ~(int64_t)31;
    for (int64_t c = threadIdx.x; c < rounded; c += kScanBlock)
        emit_cell_items(c, cs, cell_sources, start, mid, n_cells, max_items, items, stats);
}

// ---------------------------------------------------------------------------------------
// kick / drift
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_kick(int64_t n, float dt, const float *__restrict__ ax,
                                              const float *__restrict__ ay,
                                              const float *__restrict__ az, float *vx, float *vy,
                                              float *vz)
{
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        vx[i] = fmaf(dt, ax[i], vx[i]);
        vy[i] = fmaf(dt, ay[i], vy[i]);
        vz[i] = fmaf(dt, az[i], vz[i]);
    }
}

__global__ void __launch_bounds__(256) k_drift(int64_t n, float dt, float box_l, float *x,
                                               float *y, float *z, const float *__restrict__ vx,
                                               const float *__restrict__ vy,
                                               const float *__restrict__ vz, DeviceStats *stats)
{
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        x[i] = wrap_pos(fmaf(dt, vx[i], x[i]), box_l, bad);
        y[i] = wrap_pos(fmaf(dt, vy[i], y[i]), box_l, bad);
        z[i] = wrap_pos(fmaf(dt, vz[i], z[i]), box_l, bad);
    }
    if (bad) stats->error_flag = HACCSR_EDATA;
}

static inline int stream_grid(const haccsr_ctx *c, int64_t n, int per_sm)
{
    int64_t want = (n + 255) / 256;
    int64_t cap = (int64_t)c->n_sms * per_sm;
    return (int)(want < cap ? (want > 0 ? want : 1) : cap);
}

int64_t max_items_for(int64_t n_max, int64_t n_cells)
{
    // target chunks <= n/128 + 3 per non-empty cell (and <= n/8 + n/128: a cell needs 17
    // particles for a second tail chunk, 33 for a third); the source splits of a cell multiply
    // its chunks: split-induced items <= kTargetItems + 4 * 27*n/kMinSplit
    int64_t nonempty = n_max < n_cells ? n_max : n_cells;
    int64_t chunks = 3 * nonempty < n_max / 8 + nonempty ? 3 * nonempty : n_max / 8 + nonempty;
    // small problems (n_eval < 2^31) are cut at kSmallSplitSources: at most n_eval / 256 = 2^23
    // more items, and never more than 4 * 27 n / 256
    const int64_t small = std::min<int64_t>(4 * (27 * n_max) / kSmallSplitSources, int64_t(1) << 23);
    return chunks + n_max / 128 + (int64_t)kTargetItems +
           4 * (27 * n_max) / kMinSplitSources + small + 4096;
}

cudaError_t launch_bin(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                       const float *mass)
{
    cudaError_t e;
    // keep the sticky error flag; clear everything else
    if ((e = cudaMemsetAsync(c->stats, 0, offsetof(DeviceStats, error_flag), c->stream))) return e;
    if ((e = launch_sort(c, n, x, y, z, mass))) return e;
    return launch_worklist(c, c->act_level ? c->cell_mid : nullptr);
}

// The force kernel's work list from the current cell_start; `mid` as in k_cell_sources.
cudaError_t launch_worklist(haccsr_ctx *c, const uint32_t *mid)
{
    cudaStream_t st = c->stream;
    cudaError_t e;
    int cell_blocks = (int)((c->n_cells + 255) / 256);
    k_cell_sources<<<c->nz * ((c->nc + kCsRows - 1) / kCsRows), 256, 0, st>>>(
        c->cell_start, c->nc, c->nz, c->n_cells, mid, c->cell_sources, c->stats);
    if (c->n_cells <= kSmallCells) {
        k_items_small<<<1, kScanBlock, 0, st>>>(c->cell_start, c->cell_sources, mid, c->n_cells,
                                                c->max_items, c->items, c->stats);
        return cudaGetLastError();
    }
    k_item_count<<<cell_blocks, 256, 0, st>>>(c->cell_start, c->cell_sources, mid, c->n_cells,
                                              c->item_count, c->stats);
    if ((e = scan_u32(c, c->item_count, 2 * c->n_cells, c->item_start, nullptr))) return e;
    k_emit_items<<<cell_blocks, 256, 0, st>>>(c->cell_start, c->cell_sources, c->item_start, mid,
                                              c->n_cells, c->max_items, c->items, c->stats);
    return cudaGetLastError();
}

cudaError_t launch_kick(haccsr_ctx *c, float dt)
{
    if (c->n > 0)
        k_kick<<<stream_grid(c, c->n, 16), 256, 0, c->stream>>>(c->n, dt, c->ax, c->ay, c->az,
                                                                c->vx, c->vy, c->vz);
    return cudaGetLastError();
}

cudaError_t launch_drift(haccsr_ctx *c, int64_t n, float *x, float *y, float *z, const float *vx,
                         const float *vy, const float *vz, float dt)
{
    if (n > 0)
        k_drift<<<stream_grid(c, n, 16), 256, 0, c->stream>>>(n, dt, c->box_l, x, y, z, vx, vy,
                                                              vz, c->stats);
    return cudaGetLastError();
}

}  // namespace haccsr
