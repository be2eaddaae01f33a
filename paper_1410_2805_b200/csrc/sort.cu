// sort.cu -- counting sort of the particles into chaining-mesh cell order (
// permutation array PAPER.md:239) as three shared-memory-staged partition passes, one per
// cell coordinate (z slab, y row, x cell).
//
// Why staged passes: measured on B200, a store instruction whose lanes hit 32 different
// sectors retires at ~25 G stores/s chip-wide whatever the locality, while runs of >= 24
// consecutive 16-byte records stream near the HBM rate.  So every pass ranks a tile of
// particles by one digit (nc <= 256 values) with shared-memory atomics, lays the tile out in
// digit order in shared memory, and writes it back as runs; no thread ever issues a scattered
// global store.  DESIGN.md section 6.2 has the byte counts.
//
//   P0 k_count_rows : read y,z -> histogram of (cz,cy) rows in shared memory (nc^2 bins)
//   scan            : row_start[nc^2+1]; slab_start[cz] = row_start[cz*nc]
//   P1 k_part_z     : read x,y,z,(m) -> tmpA partitioned by cz            (runs of ~T/nc)
//   P2 k_part_y     : tmpA -> tmpB partitioned by (cz,cy), slab-aligned tiles
//   P3 k_sort_rows  : every CTA owns a contiguous run of rows holding ~n/grid particles:
//                     sort each row by cx in shared memory, write sorted float4, perm and
//                     the row's cell_start entries (rows longer than a tile: count pass +
//                     tile passes with CTA-private cursors)
//
// All three passes are software-pipelined: the loads of the next tile are issued before the
// current tile is written out, so the HBM reads overlap the write-out and the next ranking.
//
// Records are 16 bytes {x,y,z,w}: w = mass, and the original index travels in a second array;
// with unit masses w carries the index bits and the second array is not touched.
#include <cstddef>

#include "ctx.h"
#include "mesh.cuh"


namespace haccsr {

constexpr int kSortPer = 8;        // particles per thread per tile
constexpr int kMaxDigits = 256;    // nc <= 256
constexpr int kSortGridMax = 1024; // upper bound of any sort grid (row ownership table)

template <int THREADS, bool MASS>
struct SortSmem {
    static constexpr int kThreads = THREADS;
    static constexpr int kTile = THREADS * kSortPer;
    static constexpr bool kMass = MASS;
    float4 rec[kTile];
    uint32_t idx[MASS ? kTile : 1];
    uint8_t dig[kTile];
    uint32_t cnt[kMaxDigits];    // particles of this tile per digit
    uint32_t off[kMaxDigits];    // exclusive scan of cnt
    uint32_t gbase[kMaxDigits];  // global slot of the digit's first staged element minus off
    uint32_t cur[kMaxDigits];    // P3 long rows: running cursor per cell
    uint32_t tab[kMaxDigits + 4];  // P2: first tile of each slab
    uint32_t tab2[kMaxDigits + 4]; // P2: first slot of each slab
    uint32_t warp_tot[kMaxDigits / 32];
};

// Exclusive scan of s.cnt[0..K) into s.off, K <= 256.  All threads call it; ends synchronised.
template <class S>
__device__ __forceinline__ void tile_scan(S &s, int K)
{
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    uint32_t v = 0, inc = 0;
    if (t < kMaxDigits) {
        v = (t < K) ? s.cnt[t] : 0u;
        inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t u = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += u;
        }
        if (lane == 31) s.warp_tot[w] = inc;
    }
    __syncthreads();
    if (t < kMaxDigits) {
        uint32_t base = 0;
#pragma unroll
        for (int k = 0; k < kMaxDigits / 32; ++k) base += (k < w) ? s.warp_tot[k] : 0u;
        if (t < K) s.off[t] = base + inc - v;
    }
    __syncthreads();
}

// rank[k] = position of the particle among the tile's particles of the same digit
// (s.cnt must be zero on entry; it holds the tile's histogram on exit).
template <class S>
__device__ __forceinline__ void tile_rank(S &s, const int (&d)[kSortPer],
                                          uint32_t (&rank)[kSortPer])
{
#pragma unroll
    for (int k = 0; k < kSortPer; ++k)
        if (d[k] >= 0) rank[k] = atomicAdd(&s.cnt[d[k]], 1u);
    __syncthreads();
}

// Lay the tile out in digit order in shared memory (no barrier: the caller adds one after it
// has also published gbase).
template <class S, bool DIGITS = true>
__device__ __forceinline__ void tile_stage(S &s, const int (&d)[kSortPer],
                                           const uint32_t (&rank)[kSortPer],
                                           const float4 (&r)[kSortPer],
                                           const uint32_t (&ix)[kSortPer])
{
#pragma unroll
    for (int k = 0; k < kSortPer; ++k)
        if (d[k] >= 0) {
            const uint32_t p = s.off[d[k]] + rank[k];
            s.rec[p] = r[k];
            if (S::kMass) s.idx[p] = ix[k];
            if (DIGITS) s.dig[p] = (uint8_t)d[k];  // not needed when the whole tile is one run
        }
}

// Staged element k goes to global slot gbase[digit] + k: consecutive k of one digit are
// consecutive slots, so a warp writes runs.  Clears s.cnt for the next tile; ends synchronised.
template <class S>
__device__ __forceinline__ void tile_writeout(S &s, int K, int n_tile,
                                              float4 *__restrict__ out_rec,
                                              uint32_t *__restrict__ out_idx)
{
    if (threadIdx.x < K) s.cnt[threadIdx.x] = 0;
    for (int k = threadIdx.x; k < n_tile; k += S::kThreads) {
        const uint32_t dst = s.gbase[s.dig[k]] + (uint32_t)k;
        out_rec[dst] = s.rec[k];
        if (S::kMass) out_idx[dst] = s.idx[k];
    }
    __syncthreads();
}

// The row's final layout: sorted float4 {x,y,z,m} and perm (sorted slot -> original index).
template <class S, bool LINEAR = false>
__device__ __forceinline__ void tile_writeout_final(S &s, int K, int n_tile,
                                                    float4 *__restrict__ sorted,
                                                    uint32_t *__restrict__ perm,
                                                    uint32_t linear_base = 0)
{
    if (threadIdx.x < K) s.cnt[threadIdx.x] = 0;
    for (int k = threadIdx.x; k < n_tile; k += S::kThreads) {
        // LINEAR: the tile is a whole row, staged element k is slot linear_base + k
        const uint32_t dst = (LINEAR ? linear_base : s.gbase[s.dig[k]]) + (uint32_t)k;
        float4 r = s.rec[k];
        uint32_t i;
        if (S::kMass) {
            i = s.idx[k];
        } else {
            i = __float_as_uint(r.w);
            r.w = 1.f;
        }
        sorted[dst] = r;
        perm[dst] = i;
    }
    __syncthreads();
}

// Issue the loads of one tile of 16-byte records (P2, P3); nothing waits on them here.
template <class S>
__device__ __forceinline__ void tile_prefetch(const float4 *__restrict__ in_rec,
                                              const uint32_t *__restrict__ in_idx, uint32_t base,
                                              int n_tile, float4 (&r)[kSortPer],
                                              uint32_t (&ix)[kSortPer])
{
#pragma unroll
    for (int k = 0; k < kSortPer; ++k) {
        const int j = k * S::kThreads + (int)threadIdx.x;
        if (j < n_tile) {
            r[k] = __ldg(in_rec + base + j);
            if (S::kMass) ix[k] = __ldg(in_idx + base + j);
        }
    }
}

// ---------------------------------------------------------------------------------------
// P0: histogram of (cz,cy) rows.  8 B read per particle.  The nc^2 counters live in shared
// memory (one persistent CTA per SM) and are flushed once; meshes too large for that
// (nc > 224) count straight into global memory.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_count_rows(int64_t n, const float *__restrict__ y,
                                                     const float *__restrict__ z, MeshGeom g,
                                                     uint32_t *__restrict__ row_count,
                                                     DeviceStats *stats, int use_smem)
{
    extern __shared__ uint32_t hist[];
    constexpr int U = 4;
    const int n_rows = g.nc * g.nc;
    if (use_smem) {
        for (int i = threadIdx.x; i < n_rows; i += blockDim.x) hist[i] = 0;
        __syncthreads();
    }
    bool bad = false;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * U;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x * U + threadIdx.x; i0 < n; i0 += stride) {
        float py[U], pz[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t i = i0 + (int64_t)u * blockDim.x;
            py[u] = (i < n) ? __ldg(y + i) : 0.f;
            pz[u] = (i < n) ? __ldg(z + i) : 0.f;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (i0 + (int64_t)u * blockDim.x >= n) break;
            const float wy = wrap_pos(py[u], g.box_l, bad), wz = wrap_pos(pz[u], g.box_l, bad);
            const int r = cell_coord(wy, g) + g.nc * cell_coord(wz, g);
            if (use_smem) atomicAdd(&hist[r], 1u);
            else atomicAdd(row_count + r, 1u);
        }
    }
    if (bad) stats->error_flag = HACCSR_EDATA;
    if (use_smem) {
        __syncthreads();
        for (int i = threadIdx.x; i < n_rows; i += blockDim.x) {
            const uint32_t v = hist[i];
            if (v) atomicAdd(row_count + i, v);
        }
    }
}

// After the scan of the row counts: slab cursors, the slab-aligned tile table of P2, the rows
// each CTA of P3 owns (contiguous runs of ~n/grid3 particles) and the sentinel cell_start[nc^3].
__global__ void __launch_bounds__(256) k_sort_setup(int nc, int64_t n, int64_t n_cells, int tile2,
                                                    int grid3,
                                                    const uint32_t *__restrict__ row_start,
                                                    uint32_t *__restrict__ slab_cursor,
                                                    uint32_t *__restrict__ tile_start,
                                                    uint32_t *__restrict__ row_first,
                                                    uint32_t *__restrict__ cell_start)
{
    __shared__ uint32_t tiles[kMaxDigits];
    const int t = threadIdx.x;
    if (t < nc) {
        const uint32_t b = row_start[t * nc], e = row_start[(t + 1) * nc];
        slab_cursor[t] = b;
        tiles[t] = (e - b + (uint32_t)tile2 - 1) / (uint32_t)tile2;
    }
    __syncthreads();
    if (t == 0) {
        uint32_t run = 0;
        for (int k = 0; k < nc; ++k) {
            tile_start[k] = run;
            run += tiles[k];
        }
        tile_start[nc] = run;
        cell_start[n_cells] = (uint32_t)n;
    }
    const int n_rows = nc * nc;
    for (int j = t; j <= grid3; j += blockDim.x) {
        uint32_t first = (uint32_t)n_rows;
        if (j < grid3) {
            const uint32_t lo_slot = (uint32_t)((int64_t)j * n / grid3);
            int lo = 0, hi = n_rows;  // first row with row_start >= lo_slot
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (row_start[mid] >= lo_slot) hi = mid; else lo = mid + 1;
            }
            first = (uint32_t)lo;
        }
        row_first[j] = first;
    }
}

// ---------------------------------------------------------------------------------------
// P1: partition the caller's SoA arrays by z slab.  12 B (+4 with masses) read, 16 (+4) written.
// ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(S::kThreads, S::kThreads >= 1024 ? 1 : 2)
    k_part_z(int64_t n, const float *__restrict__ x, const float *__restrict__ y,
             const float *__restrict__ z, const float *__restrict__ mass, MeshGeom g,
             uint32_t *__restrict__ slab_cursor, float4 *__restrict__ out_rec,
             uint32_t *__restrict__ out_idx, DeviceStats *stats)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S &s = *reinterpret_cast<S *>(smem_raw);
    const int K = g.nc, tid = threadIdx.x;
    const int64_t n_tiles = (n + S::kTile - 1) / S::kTile;
    bool bad = false;
    float4 r[kSortPer];
    uint32_t ix[kSortPer], rank[kSortPer];
    int d[kSortPer];
    auto prefetch = [&](int64_t t) {
        const int64_t base = t * S::kTile;
#pragma unroll
        for (int k = 0; k < kSortPer; ++k) {
            const int64_t i = base + k * S::kThreads + tid;
            if (i < n) {
                r[k].x = __ldg(x + i);
                r[k].y = __ldg(y + i);
                r[k].z = __ldg(z + i);
                if (S::kMass) r[k].w = __ldg(mass + i);
            }
        }
    };
    if (tid < K) s.cnt[tid] = 0;
    __syncthreads();
    if (blockIdx.x < n_tiles) prefetch(blockIdx.x);
    for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int64_t base = t * S::kTile;
        const int n_tile = (int)min((int64_t)S::kTile, n - base);
#pragma unroll
        for (int k = 0; k < kSortPer; ++k) {
            const int64_t i = base + k * S::kThreads + tid;
            d[k] = -1;
            ix[k] = (uint32_t)i;
            if (i < n) {
                r[k].x = wrap_pos(r[k].x, g.box_l, bad);
                r[k].y = wrap_pos(r[k].y, g.box_l, bad);
                r[k].z = wrap_pos(r[k].z, g.box_l, bad);
                if (!S::kMass) r[k].w = __uint_as_float((uint32_t)i);
                d[k] = cell_coord(r[k].z, g);
            }
        }
        tile_rank(s, d, rank);
        uint32_t resv = 0;
        if (tid < K) {
            const uint32_t c = s.cnt[tid];
            if (c) resv = atomicAdd(slab_cursor + tid, c);
        }
        tile_scan(s, K);
        tile_stage(s, d, rank, r, ix);
        if (tid < K) s.gbase[tid] = resv - s.off[tid];
        __syncthreads();
        if (t + gridDim.x < n_tiles) prefetch(t + gridDim.x);
        tile_writeout(s, K, n_tile, out_rec, out_idx);
    }
    if (bad) stats->error_flag = HACCSR_EDATA;
}

// ---------------------------------------------------------------------------------------
// P2: partition each slab by y row.  Tiles never straddle a slab, so a tile has nc digits.
// ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(S::kThreads, S::kThreads >= 1024 ? 1 : 2)
    k_part_y(const float4 *__restrict__ in_rec, const uint32_t *__restrict__ in_idx, MeshGeom g,
             const uint32_t *__restrict__ row_start, const uint32_t *__restrict__ tile_start,
             uint32_t *__restrict__ row_cursor, float4 *__restrict__ out_rec,
             uint32_t *__restrict__ out_idx)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S &s = *reinterpret_cast<S *>(smem_raw);
    const int K = g.nc, tid = threadIdx.x;
    for (int i = tid; i <= K; i += S::kThreads) {
        s.tab[i] = tile_start[i];
        s.tab2[i] = row_start[i * K];
    }
    if (tid < K) s.cnt[tid] = 0;
    __syncthreads();
    const uint32_t n_tiles = s.tab[K];
    float4 r[kSortPer];
    uint32_t ix[kSortPer], rank[kSortPer];
    int d[kSortPer];
    int slab = 0, n_tile = 0;
    uint32_t base = 0;
    auto locate = [&](uint32_t t) {  // last slab whose first tile is <= t (it owns tile t)
        int lo = 0, hi = K - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (s.tab[mid] <= t) lo = mid; else hi = mid - 1;
        }
        slab = lo;
        base = s.tab2[lo] + (t - s.tab[lo]) * (uint32_t)S::kTile;
        n_tile = (int)min((uint32_t)S::kTile, s.tab2[lo + 1] - base);
    };
    if (blockIdx.x < n_tiles) {
        locate(blockIdx.x);
        tile_prefetch<S>(in_rec, in_idx, base, n_tile, r, ix);
    }
    for (uint32_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int cur_slab = slab, cur_n = n_tile;
#pragma unroll
        for (int k = 0; k < kSortPer; ++k)
            d[k] = (k * S::kThreads + tid < cur_n) ? cell_coord(r[k].y, g) : -1;
        tile_rank(s, d, rank);
        uint32_t resv = 0;
        if (tid < K) {
            const uint32_t c = s.cnt[tid];
            if (c) resv = atomicAdd(row_cursor + cur_slab * K + tid, c);
        }
        tile_scan(s, K);
        tile_stage(s, d, rank, r, ix);
        if (tid < K) s.gbase[tid] = resv - s.off[tid];
        __syncthreads();
        if (t + gridDim.x < n_tiles) {
            locate(t + gridDim.x);
            tile_prefetch<S>(in_rec, in_idx, base, n_tile, r, ix);
        }
        tile_writeout(s, K, cur_n, out_rec, out_idx);
    }
}

// ---------------------------------------------------------------------------------------
// P3: order every (cz,cy) row by cx, write the final arrays and the row's nc cell_start
// entries.  CTA j owns the rows [row_first[j], row_first[j+1]): contiguous and holding about
// n/grid particles, so the work is balanced without tickets and the next row is known early.
// A row that fits a tile is sorted in shared memory and written linearly (its loads were
// issued while the previous row was written out); a longer row (halo rows) is counted first
// and then placed tile by tile with CTA-private cursors -- its runs are long because few
// cells hold most of its particles.
// ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(S::kThreads, S::kThreads >= 1024 ? 1 : 2)
    k_sort_rows(const float4 *__restrict__ in_rec, const uint32_t *__restrict__ in_idx, MeshGeom g,
                const uint32_t *__restrict__ row_start, const uint32_t *__restrict__ row_first,
                uint32_t *__restrict__ cell_start, float4 *__restrict__ sorted,
                uint32_t *__restrict__ perm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S &s = *reinterpret_cast<S *>(smem_raw);
    const int K = g.nc, tid = threadIdx.x;
    const uint32_t r_end = row_first[blockIdx.x + 1];
    uint32_t row = row_first[blockIdx.x];
    if (tid < K) s.cnt[tid] = 0;
    __syncthreads();
    if (row >= r_end) return;
    float4 r[kSortPer];
    uint32_t ix[kSortPer], rank[kSortPer];
    int d[kSortPer];
    uint32_t b = row_start[row], e = row_start[row + 1];
    if (e - b <= (uint32_t)S::kTile) tile_prefetch<S>(in_rec, in_idx, b, (int)(e - b), r, ix);
    for (; row < r_end; ++row) {
        const uint32_t nb = e;  // rows are contiguous
        const uint32_t ne = (row + 1 < r_end) ? __ldg(row_start + row + 2) : e;
        const bool next_short = (row + 1 < r_end) && (ne - nb <= (uint32_t)S::kTile);
        if (e - b <= (uint32_t)S::kTile) {
            const int n_tile = (int)(e - b);
#pragma unroll
            for (int k = 0; k < kSortPer; ++k)
                d[k] = (k * S::kThreads + tid < n_tile) ? cell_coord(r[k].x, g) : -1;
            tile_rank(s, d, rank);
            tile_scan(s, K);
            tile_stage<S, false>(s, d, rank, r, ix);
            if (tid < K) cell_start[(size_t)row * K + tid] = b + s.off[tid];
            __syncthreads();
            if (next_short) tile_prefetch<S>(in_rec, in_idx, nb, (int)(ne - nb), r, ix);
            tile_writeout_final<S, true>(s, K, n_tile, sorted, perm, b);
        } else {
            // first tile's loads fly while the whole row is counted
            tile_prefetch<S>(in_rec, in_idx, b, S::kTile, r, ix);
            if (tid < K) s.cur[tid] = 0;
            __syncthreads();
            for (uint32_t i0 = b + tid; i0 < e; i0 += 4 * S::kThreads) {
                float xs[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = i0 + u * S::kThreads;
                    xs[u] = (i < e) ? __ldg(&in_rec[i].x) : -1.f;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (i0 + u * S::kThreads < e) atomicAdd(&s.cur[cell_coord(xs[u], g)], 1u);
            }
            __syncthreads();
            if (tid < K) s.cnt[tid] = s.cur[tid];
            __syncthreads();
            tile_scan(s, K);
            if (tid < K) {
                cell_start[(size_t)row * K + tid] = b + s.off[tid];
                s.cur[tid] = b + s.off[tid];
                s.cnt[tid] = 0;
            }
            __syncthreads();
            for (uint32_t base = b; base < e; base += S::kTile) {
                const int n_tile = (int)min((uint32_t)S::kTile, e - base);
#pragma unroll
                for (int k = 0; k < kSortPer; ++k)
                    d[k] = (k * S::kThreads + tid < n_tile) ? cell_coord(r[k].x, g) : -1;
                tile_rank(s, d, rank);
                tile_scan(s, K);
                tile_stage(s, d, rank, r, ix);
                if (tid < K) {
                    s.gbase[tid] = s.cur[tid] - s.off[tid];
                    s.cur[tid] += s.cnt[tid];
                }
                __syncthreads();
                const uint32_t nxt = base + S::kTile;
                if (nxt < e)
                    tile_prefetch<S>(in_rec, in_idx, nxt, (int)min((uint32_t)S::kTile, e - nxt), r,
                                     ix);
                else if (next_short)
                    tile_prefetch<S>(in_rec, in_idx, nb, (int)(ne - nb), r, ix);
                tile_writeout_final(s, K, n_tile, sorted, perm);
            }
        }
        b = nb;
        e = ne;
    }
}

// cell id per ORIGINAL particle, on demand (haccsr_get_mesh): derived from the sorted copy.
__global__ void __launch_bounds__(256) k_cell_ids(int64_t n, const float4 *__restrict__ sorted,
                                                  const uint32_t *__restrict__ perm, MeshGeom g,
                                                  uint32_t *__restrict__ cid)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += stride) {
        const float4 p = sorted[s];
        int cx = cell_coord(p.x, g), cy = cell_coord(p.y, g), cz = cell_coord(p.z, g);
        cid[perm[s]] = (uint32_t)(cx + g.nc * (cy + g.nc * cz));
    }
}

constexpr int kThreads12 = 512;   // P1, P2: 4096-particle tiles, two CTAs per SM
constexpr int kThreads3 = 1024;   // P3: 8192-particle tiles (most rows of the 512^3 box fit)

template <bool MASS>
static cudaError_t run_sort(haccsr_ctx *c, int64_t n, const float *x, const float *y,
                            const float *z, const float *mass, const MeshGeom &g)
{
    using S12 = SortSmem<kThreads12, MASS>;
    using S3 = SortSmem<kThreads3, MASS>;
    cudaStream_t st = c->stream;
    const int grid12 = 2 * c->n_sms, grid3 = c->n_sms < kSortGridMax ? c->n_sms : kSortGridMax;
    static bool configured = false;  // per template instance
    cudaError_t e;
    if (!configured) {
        if ((e = cudaFuncSetAttribute(k_part_z<S12>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)sizeof(S12))))
            return e;
        if ((e = cudaFuncSetAttribute(k_part_y<S12>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)sizeof(S12))))
            return e;
        if ((e = cudaFuncSetAttribute(k_sort_rows<S3>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)sizeof(S3))))
            return e;
        configured = true;
    }
    k_sort_setup<<<1, 256, 0, st>>>(c->nc, n, c->n_cells, S12::kTile, grid3, c->row_start,
                                    c->slab_cursor, c->tile_start, c->row_first, c->cell_start);
    // tmpA aliases the final arrays (dead before P3 writes them); tmpB is workspace of its own
    float4 *a_rec = c->sorted;
    uint32_t *a_idx = c->perm;
    k_part_z<S12><<<grid12, kThreads12, sizeof(S12), st>>>(n, x, y, z, mass, g, c->slab_cursor,
                                                           a_rec, a_idx, c->stats);
    k_part_y<S12><<<grid12, kThreads12, sizeof(S12), st>>>(a_rec, a_idx, g, c->row_start,
                                                           c->tile_start, c->row_cursor,
                                                           c->tmp_pos, c->tmp_idx);
    k_sort_rows<S3><<<grid3, kThreads3, sizeof(S3), st>>>(c->tmp_pos, c->tmp_idx, g, c->row_start,
                                                          c->row_first, c->cell_start, c->sorted,
                                                          c->perm);
    return cudaGetLastError();
}

cudaError_t launch_sort(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                        const float *mass)
{
    cudaStream_t st = c->stream;
    const MeshGeom g = geom_of(c);
    const int n_rows = c->nc * c->nc;
    cudaError_t e;
    if (n == 0) return cudaMemsetAsync(c->cell_start, 0, sizeof(uint32_t) * (c->n_cells + 1), st);
    if ((e = cudaMemsetAsync(c->row_count, 0, sizeof(uint32_t) * (n_rows + 1), st))) return e;
    const size_t hist_bytes = sizeof(uint32_t) * (size_t)n_rows;
    const int use_smem = hist_bytes <= 200 * 1024;
    static bool configured = false;
    if (!configured) {
        if ((e = cudaFuncSetAttribute(k_count_rows, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      200 * 1024)))
            return e;
        configured = true;
    }
    if (use_smem)
        k_count_rows<<<c->n_sms, 1024, hist_bytes, st>>>(n, y, z, g, c->row_count, c->stats, 1);
    else
        k_count_rows<<<c->n_sms * 2, 1024, 0, st>>>(n, y, z, g, c->row_count, c->stats, 0);
    if ((e = scan_u32(c, c->row_count, n_rows, c->row_start, c->row_cursor))) return e;
    return mass ? run_sort<true>(c, n, x, y, z, mass, g) : run_sort<false>(c, n, x, y, z, mass, g);
}

cudaError_t launch_cell_ids(haccsr_ctx *c)
{
    if (c->n > 0) {
        int64_t want = (c->n + 255) / 256, cap = (int64_t)c->n_sms * 8;
        k_cell_ids<<<(int)(want < cap ? want : cap), 256, 0, c->stream>>>(
            c->n, c->sorted, c->perm, geom_of(c), c->cid);
    }
    return cudaGetLastError();
}

}  // namespace haccsr
