// sort.cu -- counting sort of the particles into chaining-mesh cell order (
// permutation array PAPER.md:239) as three shared-memory-staged partition passes, one per
// cell coordinate (z slab, y row, x cell).
//
// Why staged passes: measured on B200, 16-byte stores reach the copy
// rate only as runs of consecutive records; single scattered records retire at ~27 G stores/s
// chip-wide whatever the locality.  So every pass ranks a tile of particles by one digit
// (nc <= 256 values) with shared-memory atomics, lays the tile out in digit order in shared
// memory, and writes it back as runs; no thread ever issues a scattered global store.
//
//   P0 k_count_rows : read y,z -> histogram of (cz,cy) rows in shared memory (nc^2 bins)
//   scan + k_sort_setup : row_start[nc^2+1], the padded row starts row_pad, slab and row
//                     cursors, P2's tile table, P3's row ownership
//   P1 k_part_z     : read x,y,z,(m) -> tmpA partitioned by cz            (runs of ~T/nc)
//   P2 k_part_y     : tmpA -> tmpB partitioned by (cz,cy), slab-aligned tiles
//   P3 k_sort_rows  : every CTA owns a contiguous run of rows holding ~n/grid particles:
//                     sort each row by cx in shared memory, write sorted float4, perm and
//                     the row's cell_start entries (rows longer than a tile: count pass +
//                     tile passes with CTA-private cursors)
//      k_sort_rows_tma : the same pass with its input streamed by TMA bulk copies
//                     (cp.async.bulk + mbarrier ring) and batches of whole rows; used for the
//                     multi-level stepping's [kicked level | rest] split of every cell, and
//                     selectable (HACCSR_P3_TMA=1) for the comparison in DESIGN.md 6.2
//
// All three passes are software-pipelined through registers (the loads of the next tile are
// issued before the current tile is written out).
// In the intermediate arrays every row starts on a multiple of 4 records (`row_pad`, up to 6
// unused slots between rows), which keeps P3's bulk copies 16-byte aligned in the index array.
//
// Records are 16 bytes {x,y,z,w}: w = mass, and the original index travels in a second array;
// with unit masses w carries the index bits and the second array is not touched.
#include <algorithm>
#include <cstddef>
#include <cstdio>
#include <cstdlib>

#include "ctx.h"
#include "mesh.cuh"


namespace haccsr {

constexpr int kSortPer = 8;        // particles per thread per tile
constexpr int kMaxDigits = 256;    // nc <= 256
constexpr int kSortGridMax = 1024; // upper bound of the pass-3 grid (row ownership table)

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
    uint32_t tab2[kMaxDigits + 4]; // P2: first slot of each slab in the intermediate array
    uint32_t tab3[kMaxDigits + 4]; // P2: particles of each slab
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
// DRIFT: the stream map of the SKS sub-cycle fused into this first pass of the
// next binning: x <- wrap(x + dt v) is written back for all three coordinates (the same
// arithmetic as k_drift) and the histogram is taken of the streamed positions; saves the drift
// kernel's launch and the 8 B/particle this pass would re-read.
struct DriftArgs {
    float *x, *y, *z;
    const float *vx, *vy, *vz;
    float dt;
};

// SLAB: the context covers a z window of the mesh (layer_coord); otherwise the whole box.
template <bool DRIFT, bool SLAB>
__global__ void __launch_bounds__(1024) k_count_rows(int64_t n, const float *__restrict__ y,
                                                     const float *__restrict__ z, MeshGeom g,
                                                     uint32_t *__restrict__ row_count,
                                                     DeviceStats *stats, int use_smem,
                                                     DriftArgs dr)
{
    extern __shared__ uint32_t hist[];
    constexpr int U = 4;
    const int n_rows = g.nc * g.nz;
    if (use_smem) {
        for (int i = threadIdx.x; i < n_rows; i += blockDim.x) hist[i] = 0;
        __syncthreads();
    }
    bool bad = false;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * U;
    for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x * U + threadIdx.x; i0 < n; i0 += stride) {
        float py[U], pz[U];
        if (DRIFT) {
            float px[U], v[3][U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int64_t i = i0 + (int64_t)u * blockDim.x;
                if (i < n) {
                    px[u] = dr.x[i];
                    py[u] = dr.y[i];
                    pz[u] = dr.z[i];
                    v[0][u] = __ldg(dr.vx + i);
                    v[1][u] = __ldg(dr.vy + i);
                    v[2][u] = __ldg(dr.vz + i);
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int64_t i = i0 + (int64_t)u * blockDim.x;
                if (i < n) {
                    dr.x[i] = wrap_pos(fmaf(dr.dt, v[0][u], px[u]), g.box_l, bad);
                    dr.y[i] = py[u] = wrap_pos(fmaf(dr.dt, v[1][u], py[u]), g.box_l, bad);
                    dr.z[i] = pz[u] = wrap_pos(fmaf(dr.dt, v[2][u], pz[u]), g.box_l, bad);
                }
            }
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int64_t i = i0 + (int64_t)u * blockDim.x;
                py[u] = (i < n) ? __ldg(y + i) : 0.f;
                pz[u] = (i < n) ? __ldg(z + i) : 0.f;
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (i0 + (int64_t)u * blockDim.x >= n) break;
            const float wy = wrap_pos(py[u], g.box_l, bad), wz = wrap_pos(pz[u], g.box_l, bad);
            const int r = cell_coord(wy, g) +
                          g.nc * (SLAB ? layer_coord(wz, g, bad) : cell_coord(wz, g));
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

// Where row r starts in the sort's intermediate arrays: the dense start plus up to 3 slots of
// slack per row, rounded to a multiple of 4 records, so that every row starts 16-byte aligned
// in the index array too (bulk copies of pass 3) -- a function of row_start alone, and
// row_pad(r+1) - row_pad(r) >= the row's length.
__device__ __forceinline__ uint32_t row_pad_of(uint32_t row_start_r, uint32_t r)
{
    return (row_start_r + 3u * r + 3u) & ~3u;
}

// After the scan of the row counts (row_start): the padded row starts and P2's write cursors
// (every thread one row); block 0 also writes the slab cursors and counts, the slab-aligned
// tile table of P2, the rows each CTA of P3 owns (contiguous runs of ~n/grid3 particles) and
// the sentinel cell_start[nc^3].
// SCAN (meshes of at most 1024 rows, one block of 1024 threads): the exclusive scan of the row
// counts is done here too, one launch instead of two or four.
template <bool SCAN>
__global__ void __launch_bounds__(SCAN ? 1024 : 256) k_sort_setup(int nc, int nz, int64_t n, int64_t n_cells,
                                                    int tile2,
                                                    int grid3,
                                                    const uint32_t *__restrict__ row_count,
                                                    uint32_t *row_start,
                                                    uint32_t *__restrict__ row_pad,
                                                    uint32_t *__restrict__ row_cursor,
                                                    uint32_t *__restrict__ slab_cursor,
                                                    uint32_t *__restrict__ slab_count,
                                                    uint32_t *__restrict__ tile_start,
                                                    uint32_t *__restrict__ row_first,
                                                    uint32_t *__restrict__ cell_start)
{
    __shared__ uint32_t tiles[kMaxDigits];
    __shared__ uint32_t wtot[32];
    const int t = threadIdx.x;
    const int n_rows = nc * nz;
    const int r = blockIdx.x * blockDim.x + t;
    if (SCAN) {   // row_start[r] = sum of the counts of the rows before r; row_start[n_rows] = n
        const uint32_t v = (t < n_rows) ? row_count[t] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, inc, d);
            if ((t & 31) >= d) inc += u;
        }
        if ((t & 31) == 31) wtot[t >> 5] = inc;
        __syncthreads();
        uint32_t base = 0;
        for (int k = 0; k < (t >> 5); ++k) base += wtot[k];
        if (t < n_rows) row_start[t] = base + inc - v;
        if (t == n_rows - 1) row_start[n_rows] = base + inc;
        __syncthreads();
    }
    if (r <= n_rows) {
        const uint32_t p = row_pad_of(row_start[r], (uint32_t)r);
        row_pad[r] = p;
        if (r < n_rows) row_cursor[r] = p;
    }
    if (blockIdx.x != 0) return;
    if (t < nz) {
        const uint32_t b = row_start[t * nc], e = row_start[(t + 1) * nc];
        slab_cursor[t] = row_pad_of(b, (uint32_t)(t * nc));
        slab_count[t] = e - b;
        tiles[t] = (e - b + (uint32_t)tile2 - 1) / (uint32_t)tile2;
    }
    __syncthreads();
    if (t == 0) {
        uint32_t run = 0;
        for (int k = 0; k < nz; ++k) {
            tile_start[k] = run;
            run += tiles[k];
        }
        tile_start[nz] = run;
        cell_start[n_cells] = (uint32_t)n;
    }
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
template <class S, bool SLAB>
__global__ void __launch_bounds__(S::kThreads, S::kThreads >= 1024 ? 1 : 2)
    k_part_z(int64_t n, const float *__restrict__ x, const float *__restrict__ y,
             const float *__restrict__ z, const float *__restrict__ mass, MeshGeom g,
             uint32_t *__restrict__ slab_cursor, float4 *__restrict__ out_rec,
             uint32_t *__restrict__ out_idx, DeviceStats *stats)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S &s = *reinterpret_cast<S *>(smem_raw);
    const int K = g.nz, tid = threadIdx.x;  // digits: the window's layers
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
                d[k] = SLAB ? layer_coord(r[k].z, g, bad) : cell_coord(r[k].z, g);
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
             const uint32_t *__restrict__ row_pad, const uint32_t *__restrict__ slab_count,
             const uint32_t *__restrict__ tile_start, uint32_t *__restrict__ row_cursor,
             float4 *__restrict__ out_rec, uint32_t *__restrict__ out_idx)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S &s = *reinterpret_cast<S *>(smem_raw);
    const int K = g.nc, NS = g.nz, tid = threadIdx.x;  // rows per slab, slabs
    for (int i = tid; i <= NS; i += S::kThreads) {
        s.tab[i] = tile_start[i];
        s.tab2[i] = row_pad[i * K];              // slabs start where their first row starts
        s.tab3[i] = (i < NS) ? slab_count[i] : 0u;
    }
    if (tid < K) s.cnt[tid] = 0;
    __syncthreads();
    const uint32_t n_tiles = s.tab[NS];
    float4 r[kSortPer];
    uint32_t ix[kSortPer], rank[kSortPer];
    int d[kSortPer];
    int slab = 0, n_tile = 0;
    uint32_t base = 0;
    auto locate = [&](uint32_t t) {  // last slab whose first tile is <= t (it owns tile t)
        int lo = 0, hi = NS - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (s.tab[mid] <= t) lo = mid; else hi = mid - 1;
        }
        slab = lo;
        const uint32_t done = (t - s.tab[lo]) * (uint32_t)S::kTile;
        base = s.tab2[lo] + done;
        n_tile = (int)min((uint32_t)S::kTile, s.tab3[lo] - done);
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
// P3 (register-staged, the production path): order every (cz,cy) row by cx, write the final
// arrays and the row's nc cell_start entries.  CTA j owns the rows [row_first[j],
// row_first[j+1]): contiguous and holding about n/grid particles, so the work is balanced
// without tickets and the next row is known early.  A row that fits a tile is sorted in shared
// memory and written linearly (its loads were issued while the previous row was written out); a
// longer row (halo rows) is counted first and then placed tile by tile with CTA-private cursors
// -- its runs are long because few cells hold most of its particles.
// ---------------------------------------------------------------------------------------
template <class S>
__global__ void __launch_bounds__(S::kThreads, S::kThreads >= 1024 ? 1 : 2)
    k_sort_rows(const float4 *__restrict__ in_rec, const uint32_t *__restrict__ in_idx, MeshGeom g,
                const uint32_t *__restrict__ row_start, const uint32_t *__restrict__ row_pad,
                const uint32_t *__restrict__ row_first, uint32_t *__restrict__ cell_start,
                float4 *__restrict__ sorted, uint32_t *__restrict__ perm)
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
    // [b, e): the row's slots in the final (dense) arrays; pb: where it starts in the input
    uint32_t b = row_start[row], e = row_start[row + 1], pb = row_pad[row];
    if (e - b <= (uint32_t)S::kTile) tile_prefetch<S>(in_rec, in_idx, pb, (int)(e - b), r, ix);
    for (; row < r_end; ++row) {
        const uint32_t nb = e;  // rows are contiguous in the final arrays
        const bool have_next = row + 1 < r_end;
        const uint32_t ne = have_next ? __ldg(row_start + row + 2) : e;
        const uint32_t npb = have_next ? __ldg(row_pad + row + 1) : pb;
        const bool next_short = have_next && (ne - nb <= (uint32_t)S::kTile);
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
            if (next_short) tile_prefetch<S>(in_rec, in_idx, npb, (int)(ne - nb), r, ix);
            tile_writeout_final<S, true>(s, K, n_tile, sorted, perm, b);
        } else {
            // first tile's loads fly while the whole row is counted
            tile_prefetch<S>(in_rec, in_idx, pb, S::kTile, r, ix);
            if (tid < K) s.cur[tid] = 0;
            __syncthreads();
            const uint32_t len = e - b;
            for (uint32_t i0 = tid; i0 < len; i0 += 4 * S::kThreads) {
                float xs[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t i = i0 + u * S::kThreads;
                    xs[u] = (i < len) ? __ldg(&in_rec[pb + i].x) : -1.f;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (i0 + u * S::kThreads < len) atomicAdd(&s.cur[cell_coord(xs[u], g)], 1u);
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
            for (uint32_t done = 0; done < len; done += S::kTile) {
                const int n_tile = (int)min((uint32_t)S::kTile, len - done);
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
                const uint32_t nxt = done + S::kTile;
                if (nxt < len)
                    tile_prefetch<S>(in_rec, in_idx, pb + nxt,
                                     (int)min((uint32_t)S::kTile, len - nxt), r, ix);
                else if (next_short)
                    tile_prefetch<S>(in_rec, in_idx, npb, (int)(ne - nb), r, ix);
                tile_writeout_final(s, K, n_tile, sorted, perm);
            }
        }
        b = nb;
        e = ne;
        pb = npb;
    }
}

// ---------------------------------------------------------------------------------------
// P3: order every (cz,cy) row by cx, write the final arrays and the rows' cell_start entries.
// CTA j owns the rows [row_first[j], row_first[j+1]): contiguous, about n/grid particles.
//
// The CTA's input is one contiguous span of the row-partitioned intermediate array, so it is
// streamed with TMA bulk copies (cp.async.bulk, completion on an mbarrier per chunk) into a
// shared-memory ring of kRing chunks of kChunk records: one elected thread issues chunk c as
// soon as chunk c - kRing has been consumed; no registers hold records and nothing else is
// needed to keep the HBM reads in flight under the ranking, scan and write-out phases.  Rows
// are processed in batches of whole rows (<= kBatch input slots, <= kDig cells): count the
// batch's cells with shared-memory atomics (the rank of a record is the atomic's return
// value), exclusive scan = the batch's cell_start entries, place every record's offset at
// its sorted position (inv), and write the batch out LINEARLY by gathering through inv.
// A row longer than a batch (halo rows) is counted first with plain loads and then placed
// tile by tile with CTA-private cell cursors; its runs are long because few cells hold most
// of its particles.
// ---------------------------------------------------------------------------------------
constexpr int kChunk = 1024;   // records per bulk copy
constexpr int kDig = 1024;     // cells per batch (whole rows): one per thread in the scan
constexpr int kRowsMax = kDig / 4;  // nc >= 4

template <bool MASS>
struct RowSmem {
    static constexpr bool kMass = MASS;
    static constexpr int kRing = MASS ? 9 : 12;       // chunks in the ring
    static constexpr int kBatch = MASS ? 6144 : 8192; // input slots per batch / long-row tile
    static constexpr int kPer = kBatch / 1024;        // records per thread per batch
    static constexpr int kRingRecs = kRing * kChunk;
    float4 ring[kRingRecs];
    uint32_t ring_idx[MASS ? kRingRecs : 4];
    uint16_t inv[kBatch];           // sorted position -> offset of the record in the batch span
    uint32_t cnt[2][kDig];          // cell counts -> exclusive scan (double-buffered by batch)
    uint32_t row_pad[kRowsMax + 1]; // the batch's rows in the input (relative to the stream)
    uint32_t row_dst[kRowsMax + 1]; // ... and in the final arrays
    uint32_t lcur[2 * kMaxDigits];  // long rows: running global cursor per digit
    uint32_t lgb[2 * kMaxDigits];   // long rows: global slot of the digit's first staged element
    uint32_t warp_tot[32];
    unsigned long long full[kRing]; // mbarriers: chunk c -> full[c % kRing], parity (c / kRing) & 1
};

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(unsigned long long *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}

__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// TMA bulk copy global -> shared, completion (bytes) signalled on `bar`.
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_gmem, uint32_t bytes,
                                          unsigned long long *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// In-place exclusive scan of cnt[0..nd), nd <= kDig = 1024 threads, one cell each.  Thread t
// returns the count of cell t.  Ends synchronised.
template <class S>
__device__ __forceinline__ uint32_t row_scan(S &s, uint32_t *cnt, int nd)
{
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const uint32_t v = (t < nd) ? cnt[t] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += u;
    }
    if (lane == 31) s.warp_tot[w] = inc;
    __syncthreads();
    uint32_t base = 0;
#pragma unroll
    for (int k = 0; k < 32; ++k) base += (k < w) ? s.warp_tot[k] : 0u;
    if (t < nd) cnt[t] = base + inc - v;
    __syncthreads();
    return v;
}

// ACT (multi-level time stepping): inside every cell the particles of the
// level being kicked (level[original index] == level_k) come first; cell_mid[c] is the end of
// that ACTIVE part.  The force kernel then takes its targets from [cell_start, cell_mid) and
// its sources from whole cells.  Implemented as two digits per cell, active | inactive.
template <class S, bool ACT>
__global__ void __launch_bounds__(1024, 1)
    k_sort_rows_tma(const float4 *__restrict__ in_rec, const uint32_t *__restrict__ in_idx, MeshGeom g,
                const uint32_t *__restrict__ row_start, const uint32_t *__restrict__ row_pad,
                const uint32_t *__restrict__ row_first, uint32_t *__restrict__ cell_start,
                float4 *__restrict__ sorted, uint32_t *__restrict__ perm,
                const uint8_t *__restrict__ level, int level_k, uint32_t *__restrict__ cell_mid)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];  // bulk copies need 16 bytes
    S &s = *reinterpret_cast<S *>(smem_raw);
    const int K = g.nc, tid = threadIdx.x;
    constexpr int DM = ACT ? 2 : 1;  // digits per cell
    // digit of the record in ring slot q that lies in cell `cell` of the batch / row
    auto digit_in_ring = [&](int cell, uint32_t q) -> int {
        if (!ACT) return cell;
        const uint32_t i = S::kMass ? s.ring_idx[q] : __float_as_uint(s.ring[q].w);
        return 2 * cell + (__ldg(level + i) != level_k ? 1 : 0);
    };
    const uint32_t r_end = row_first[blockIdx.x + 1];
    uint32_t row = row_first[blockIdx.x];
    if (row >= r_end) return;
    // the stream: input slots [G0, G1) of this CTA, cut into chunks of kChunk records
    const uint32_t G0 = row_pad[row], G1 = row_pad[r_end];
    const uint32_t n_chunks = (G1 - G0 + kChunk - 1) / kChunk;
    if (tid == 0) {
        for (int k = 0; k < S::kRing; ++k) mbar_init(&s.full[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    s.cnt[0][tid] = 0;
    s.cnt[1][tid] = 0;
    __syncthreads();
    uint32_t issued = 0;  // thread 0: chunks issued so far
    auto produce = [&](uint32_t released) {  // thread 0 only; chunks < released are consumed
        while (issued < n_chunks && issued < released + (uint32_t)S::kRing) {
            const uint32_t slot = issued % (uint32_t)S::kRing;
            const uint32_t g0 = G0 + issued * kChunk;
            const uint32_t len = min(G1 - g0, (uint32_t)kChunk);  // a multiple of 4
            mbar_expect_tx(&s.full[slot], len * (S::kMass ? 20u : 16u));
            bulk_load(&s.ring[slot * kChunk], in_rec + g0, len * 16u, &s.full[slot]);
            if (S::kMass)
                bulk_load(&s.ring_idx[slot * kChunk], in_idx + g0, len * 4u, &s.full[slot]);
            ++issued;
        }
    };
    if (tid == 0) produce(0);
    uint32_t waited = 0;  // every thread: chunks < waited have landed (and were waited for)
    auto wait_upto = [&](uint32_t pos_end) {  // stream positions < pos_end are needed
        const uint32_t need = (pos_end + kChunk - 1) / kChunk;
        while (waited < need) {
            mbar_wait(&s.full[waited % (uint32_t)S::kRing], (waited / (uint32_t)S::kRing) & 1u);
            ++waited;
        }
    };
    auto ring_at = [&](uint32_t pos) -> uint32_t { return pos % (uint32_t)S::kRingRecs; };
    // the final record and index of ring slot q
    auto emit = [&](uint32_t q, uint32_t dst) {
        float4 rec = s.ring[q];
        uint32_t i;
        if (S::kMass) {
            i = s.ring_idx[q];
        } else {
            i = __float_as_uint(rec.w);
            rec.w = 1.f;
        }
        sorted[dst] = rec;
        perm[dst] = i;
    };

    int cb = 0;             // which half of s.cnt the current batch uses (the other is zero)
    uint32_t consumed = 0;  // stream position up to which the ring may be refilled
    int d[S::kPer];
    uint32_t rank[S::kPer];
    while (row < r_end) {
        // ---- batch extent: the longest run of whole rows that fits the ring and the table ----
        const uint32_t p0 = row_pad[row];                 // padded start of the first row
        const uint32_t max_rows = min((uint32_t)(kDig / (K * DM)), r_end - row);
        bool ok = false;
        if ((uint32_t)tid < max_rows) {
            const uint32_t rp_next = __ldg(row_pad + row + tid + 1);
            ok = (rp_next - p0) <= (uint32_t)S::kBatch;  // the row ends inside the batch
            s.row_pad[tid + 1] = rp_next - G0;
            s.row_dst[tid + 1] = __ldg(row_start + row + tid + 1);
        }
        if (tid == 0) {
            s.row_pad[0] = p0 - G0;
            s.row_dst[0] = row_start[row];
        }
        // ok is a prefix (padded starts are monotone).  This barrier also ends the previous
        // batch: every thread has finished reading its ring slots.
        const int n_rows = __syncthreads_count(ok);
        if (tid == 0) produce(consumed / kChunk);
        uint32_t *cnt = s.cnt[cb];
        if (n_rows > 0) {
            const uint32_t span0 = s.row_pad[0], span1 = s.row_pad[n_rows];
            const uint32_t out0 = s.row_dst[0], n_batch = s.row_dst[n_rows] - out0;
            const int nd = n_rows * K * DM;
            wait_upto(span1);
            int r = 0;  // row of this thread's next record (positions grow with k)
#pragma unroll
            for (int k = 0; k < S::kPer; ++k) {
                const uint32_t pos = span0 + tid + 1024u * k;
                d[k] = -1;
                if (pos < span1) {
                    while (r + 1 < n_rows && pos >= s.row_pad[r + 1]) ++r;
                    if (pos - s.row_pad[r] < s.row_dst[r + 1] - s.row_dst[r]) {  // not a pad slot
                        const uint32_t q = ring_at(pos);
                        d[k] = digit_in_ring(r * K + cell_coord(s.ring[q].x, g), q);
                        rank[k] = atomicAdd(&cnt[d[k]], 1u);
                    }
                }
            }
            __syncthreads();
            row_scan(s, cnt, nd);
            if (tid < nd) {
                if (!ACT) cell_start[(size_t)row * K + tid] = out0 + cnt[tid];
                else if (tid & 1) cell_mid[(size_t)row * K + (tid >> 1)] = out0 + cnt[tid];
                else cell_start[(size_t)row * K + (tid >> 1)] = out0 + cnt[tid];
            }
#pragma unroll
            for (int k = 0; k < S::kPer; ++k)
                if (d[k] >= 0) s.inv[cnt[d[k]] + rank[k]] = (uint16_t)(tid + 1024u * k);
            s.cnt[cb ^ 1][tid] = 0;   // the next batch's counters
            __syncthreads();
            for (uint32_t k = tid; k < n_batch; k += 1024)
                emit(ring_at(span0 + s.inv[k]), out0 + k);
            consumed = span1;
            row += n_rows;
            cb ^= 1;
            continue;
        }
        // ---- a row longer than a batch: count it with plain loads, then place it tile by tile
        {
            const uint32_t b = s.row_dst[0], len = s.row_dst[1] - b, pb = p0;
            for (uint32_t i0 = tid; i0 < len; i0 += 4 * 1024) {
                float xs[4];
                uint32_t is[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t i = i0 + k * 1024;
                    xs[k] = (i < len) ? __ldg(&in_rec[pb + i].x) : -1.f;
                    if (ACT && i < len)
                        is[k] = S::kMass ? __ldg(in_idx + pb + i)
                                         : __float_as_uint(__ldg(&in_rec[pb + i].w));
                }
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (i0 + k * 1024 < len) {
                        int dg = cell_coord(xs[k], g);
                        if (ACT) dg = 2 * dg + (__ldg(level + is[k]) != level_k ? 1 : 0);
                        atomicAdd(&cnt[dg], 1u);
                    }
            }
            __syncthreads();
            row_scan(s, cnt, K * DM);
            if (tid < K * DM) {
                if (!ACT) cell_start[(size_t)row * K + tid] = b + cnt[tid];
                else if (tid & 1) cell_mid[(size_t)row * K + (tid >> 1)] = b + cnt[tid];
                else cell_start[(size_t)row * K + (tid >> 1)] = b + cnt[tid];
                s.lcur[tid] = b + cnt[tid];
                cnt[tid] = 0;
            }
            __syncthreads();
            const uint32_t rel0 = pb - G0;
            for (uint32_t done = 0; done < len; done += S::kBatch) {
                const uint32_t n_tile = min((uint32_t)S::kBatch, len - done);
                const uint32_t span0 = rel0 + done, span1 = span0 + n_tile;
                wait_upto(span1);
#pragma unroll
                for (int k = 0; k < S::kPer; ++k) {
                    const uint32_t pos = span0 + tid + 1024u * k;
                    d[k] = -1;
                    if (pos < span1) {
                        const uint32_t q = ring_at(pos);
                        d[k] = digit_in_ring(cell_coord(s.ring[q].x, g), q);
                        rank[k] = atomicAdd(&cnt[d[k]], 1u);
                    }
                }
                __syncthreads();
                const uint32_t c = row_scan(s, cnt, K * DM);
                if (tid < K * DM) {
                    s.lgb[tid] = s.lcur[tid] - cnt[tid];
                    s.lcur[tid] += c;
                }
#pragma unroll
                for (int k = 0; k < S::kPer; ++k)
                    if (d[k] >= 0) s.inv[cnt[d[k]] + rank[k]] = (uint16_t)(tid + 1024u * k);
                __syncthreads();
                if (tid < K * DM) cnt[tid] = 0;
                for (uint32_t k = tid; k < n_tile; k += 1024) {
                    const uint32_t q = ring_at(span0 + s.inv[k]);
                    emit(q, s.lgb[digit_in_ring(cell_coord(s.ring[q].x, g), q)] + k);
                }
                __syncthreads();  // ring slots of the tile are free, cnt is zero again
                consumed = span1;
                if (tid == 0) produce(consumed / kChunk);
            }
            row += 1;
        }
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
        bool bad = false;
        int cx = cell_coord(p.x, g), cy = cell_coord(p.y, g), lz = layer_coord(p.z, g, bad);
        cid[perm[s]] = (uint32_t)(cx + g.nc * (cy + g.nc * lz));
    }
}

constexpr int kThreads12 = 512;   // P1, P2: 4096-particle tiles, two CTAs per SM
constexpr int kThreads3 = 1024;   // P3: 8192-particle tiles, one CTA per SM

// HACCSR_DEBUG=1 in the environment: synchronise after every stage of the sort and name the
// first one that fails on stderr (the stages are asynchronous otherwise).
static bool debug_sync()
{
    static const bool on = getenv("HACCSR_DEBUG") != nullptr;
    return on;
}

static cudaError_t stage_check(cudaStream_t st, const char *stage)
{
    cudaError_t e = cudaGetLastError();
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (debug_sync()) cudaStreamIsCapturing(st, &cap);  // no synchronisation inside a capture
    if (e == cudaSuccess && debug_sync() && cap == cudaStreamCaptureStatusNone)
        e = cudaStreamSynchronize(st);
    if (e != cudaSuccess && debug_sync())
        fprintf(stderr, "haccsr: %s failed: %s\n", stage, cudaGetErrorString(e));
    return e;
}

constexpr size_t kCountRowsSmem = 200 * 1024;

template <bool MASS>
static cudaError_t run_sort(haccsr_ctx *c, int64_t n, const float *x, const float *y,
                            const float *z, const float *mass, const MeshGeom &g)
{
    using S12 = SortSmem<kThreads12, MASS>;
    using S3 = SortSmem<kThreads3, MASS>;
    using S3T = RowSmem<MASS>;
    cudaStream_t st = c->stream;
    const int grid12 = 2 * c->n_sms, grid3 = c->n_sms < kSortGridMax ? c->n_sms : kSortGridMax;
    cudaError_t e;
    const int n_rows = c->nc * c->nz;
    if (n_rows < 1024) {
        k_sort_setup<true><<<1, 1024, 0, st>>>(c->nc, c->nz, n, c->n_cells, S12::kTile, grid3,
                                               c->row_count, c->row_start, c->row_pad,
                                               c->row_cursor, c->slab_cursor, c->slab_count,
                                               c->tile_start, c->row_first, c->cell_start);
    } else {
        if ((e = scan_u32(c, c->row_count, n_rows, c->row_start, nullptr))) return e;
        k_sort_setup<false><<<(n_rows + 256) / 256, 256, 0, st>>>(
            c->nc, c->nz, n, c->n_cells, S12::kTile, grid3, c->row_count, c->row_start, c->row_pad,
            c->row_cursor, c->slab_cursor, c->slab_count, c->tile_start, c->row_first,
            c->cell_start);
    }
    if ((e = stage_check(st, "k_sort_setup"))) return e;
    // tmpA aliases the final arrays (dead before P3 writes them); tmpB is workspace of its own
    float4 *a_rec = c->sorted;
    uint32_t *a_idx = c->perm;
    if (c->nz < c->nc)
        k_part_z<S12, true><<<grid12, kThreads12, sizeof(S12), st>>>(
            n, x, y, z, mass, g, c->slab_cursor, a_rec, a_idx, c->stats);
    else
        k_part_z<S12, false><<<grid12, kThreads12, sizeof(S12), st>>>(
            n, x, y, z, mass, g, c->slab_cursor, a_rec, a_idx, c->stats);
    if ((e = stage_check(st, "k_part_z"))) return e;
    k_part_y<S12><<<grid12, kThreads12, sizeof(S12), st>>>(a_rec, a_idx, g, c->row_pad,
                                                           c->slab_count, c->tile_start,
                                                           c->row_cursor, c->tmp_pos, c->tmp_idx);
    if ((e = stage_check(st, "k_part_y"))) return e;
    if (c->act_level) {
        // multi-level stepping: the TMA-streamed variant that also splits every cell into
        // [kicked level | rest] (cell_mid)
        k_sort_rows_tma<S3T, true><<<grid3, kThreads3, sizeof(S3T), st>>>(
            c->tmp_pos, c->tmp_idx, g, c->row_start, c->row_pad, c->row_first, c->cell_start,
            c->sorted, c->perm, c->act_level, c->act_k, c->cell_mid);
    } else if (getenv("HACCSR_P3_TMA")) {
        // the same pass with TMA-streamed input, kept selectable for the measurement in
        // DESIGN.md section 6.2 (8 % slower than the register-staged kernel)
        k_sort_rows_tma<S3T, false><<<grid3, kThreads3, sizeof(S3T), st>>>(
            c->tmp_pos, c->tmp_idx, g, c->row_start, c->row_pad, c->row_first, c->cell_start,
            c->sorted, c->perm, nullptr, 0, nullptr);
    } else {
        k_sort_rows<S3><<<grid3, kThreads3, sizeof(S3), st>>>(c->tmp_pos, c->tmp_idx, g,
                                                              c->row_start, c->row_pad,
                                                              c->row_first, c->cell_start,
                                                              c->sorted, c->perm);
    }
    return stage_check(st, "k_sort_rows");
}

// The opt-in for more than 48 KB of dynamic shared memory is a per-device attribute of each
// kernel: haccsr_create calls this once per context with the context's device current.
cudaError_t configure_sort_kernels()
{
    cudaError_t e;
    auto dyn = cudaFuncAttributeMaxDynamicSharedMemorySize;
#define HACCSR_OPT_IN(kernel, bytes) \
    if ((e = cudaFuncSetAttribute(kernel, dyn, (int)(bytes))) != cudaSuccess) return e
    HACCSR_OPT_IN((k_count_rows<false, false>), kCountRowsSmem);
    HACCSR_OPT_IN((k_count_rows<false, true>), kCountRowsSmem);
    HACCSR_OPT_IN((k_count_rows<true, false>), kCountRowsSmem);
    HACCSR_OPT_IN((k_count_rows<true, true>), kCountRowsSmem);
    HACCSR_OPT_IN((k_part_z<SortSmem<kThreads12, false>, false>), sizeof(SortSmem<kThreads12, false>));
    HACCSR_OPT_IN((k_part_z<SortSmem<kThreads12, true>, false>), sizeof(SortSmem<kThreads12, true>));
    HACCSR_OPT_IN((k_part_z<SortSmem<kThreads12, false>, true>), sizeof(SortSmem<kThreads12, false>));
    HACCSR_OPT_IN((k_part_z<SortSmem<kThreads12, true>, true>), sizeof(SortSmem<kThreads12, true>));
    HACCSR_OPT_IN((k_part_y<SortSmem<kThreads12, false>>), sizeof(SortSmem<kThreads12, false>));
    HACCSR_OPT_IN((k_part_y<SortSmem<kThreads12, true>>), sizeof(SortSmem<kThreads12, true>));
    HACCSR_OPT_IN((k_sort_rows<SortSmem<kThreads3, false>>), sizeof(SortSmem<kThreads3, false>));
    HACCSR_OPT_IN((k_sort_rows<SortSmem<kThreads3, true>>), sizeof(SortSmem<kThreads3, true>));
    HACCSR_OPT_IN((k_sort_rows_tma<RowSmem<false>, false>), sizeof(RowSmem<false>));
    HACCSR_OPT_IN((k_sort_rows_tma<RowSmem<true>, false>), sizeof(RowSmem<true>));
    HACCSR_OPT_IN((k_sort_rows_tma<RowSmem<false>, true>), sizeof(RowSmem<false>));
    HACCSR_OPT_IN((k_sort_rows_tma<RowSmem<true>, true>), sizeof(RowSmem<true>));
#undef HACCSR_OPT_IN
    return cudaSuccess;
}

cudaError_t launch_sort(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                        const float *mass)
{
    cudaStream_t st = c->stream;
    const MeshGeom g = geom_of(c);
    const int n_rows = c->nc * c->nz;
    cudaError_t e;
    if (n == 0) return cudaMemsetAsync(c->cell_start, 0, sizeof(uint32_t) * (c->n_cells + 1), st);
    if ((e = cudaMemsetAsync(c->row_count, 0, sizeof(uint32_t) * (n_rows + 1), st))) return e;
    const size_t hist_bytes = sizeof(uint32_t) * (size_t)n_rows;
    const int use_smem = hist_bytes <= kCountRowsSmem;
    const int grid0 = use_smem ? c->n_sms : c->n_sms * 2;
    const size_t smem0 = use_smem ? hist_bytes : 0;
    const bool slab = c->nz < c->nc;
    DriftArgs dr = {};
    if (c->pre_drift)  // hacc_sr_subcycle: the pending stream map rides in this pass (x, y, z
        dr = {const_cast<float *>(x), const_cast<float *>(y), const_cast<float *>(z),  // writable)
              c->vx, c->vy, c->vz, c->pre_drift_dt};
#define HACCSR_P0(D, SL) \
    k_count_rows<D, SL><<<grid0, 1024, smem0, st>>>(n, y, z, g, c->row_count, c->stats, use_smem, dr)
    if (c->pre_drift) {
        if (slab) HACCSR_P0(true, true); else HACCSR_P0(true, false);
    } else {
        if (slab) HACCSR_P0(false, true); else HACCSR_P0(false, false);
    }
#undef HACCSR_P0
    if ((e = stage_check(st, "k_count_rows"))) return e;
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
