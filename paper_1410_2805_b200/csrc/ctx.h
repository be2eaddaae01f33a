// ctx.h -- internal layout of a haccsr context and the launchers of each pipeline stage.
// Not part of the ABI.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/haccsr.h"

namespace haccsr {

// ---- work-list geometry -------------------------------------------
constexpr int kWarpTargets1 = 32;    // T=1 item: up to 32 targets, one per lane
constexpr int kMaxT = 4;             // targets per lane of the widest force-kernel variant
constexpr int kChunkTargets = 32 * kMaxT;  // dense cells are cut into chunks of this many targets
constexpr uint32_t kMinSplitSources = 1024;  // a source chunk is never shorter than this ...
constexpr uint32_t kSmallSplitSources = 256; // ... except in small problems (bin.cu)
constexpr uint32_t kLargeSplitSources = 2048; // ... and twice as long in large ones (bin.cu)
constexpr uint32_t kTargetItems = 1u << 20;  // aim for at most ~1M split-induced items
constexpr int kMaxNc = 256;          // largest mesh (cells per dimension)
constexpr int kScanBlock = 1024;     // threads per scan block
constexpr int kScanItems = 4;        // elements per thread
constexpr int kScanTile = kScanBlock * kScanItems;

// One work item of the force kernel, 16 bytes.
//   x = cell id
//   y = first target (offset inside the cell)
//   z = first source (offset inside the cell's flat 27-neighbour source list)
//   w = [31:24] number of targets - 1 (0..127), [23:0] unused; source count comes from
//       sources_per_split (last chunk clipped to the cell's total), bit 23 = split flag.
struct __align__(16) WorkItem {
    uint32_t cell, t_begin, s_begin, packed;
};

struct DeviceStats {  // lives in the workspace; copied out by haccsr_get_stats
    unsigned long long n_eval;
    uint32_t n_items;
    uint32_t n_split_items;
    uint32_t max_cell_count;
    uint32_t sources_per_split;
    uint32_t n_dense_items; // the first n_dense_items items have 33..128 targets (T = 2..4);
                            // the rest, every cell's items of at most 32 targets (T = 1), follow
    uint32_t pad_;
    // counters of one force evaluation, zeroed together: 24 bytes from n_recheck_tiles
    unsigned long long n_recheck_tiles;
    uint32_t item_cursor;   // k_force: next item
    uint32_t sparse_cursor; // k_force_sparse: next sparse item, counted from the front
    uint32_t dense_done;    // k_force: dense items finished
    uint32_t steal_cursor;  // k_force: sparse items taken from the BACK of the list by warps
                            // that ran out of dense items while others still had some
    int32_t error_flag;     // HACCSR_EDATA when a non-finite position was seen
};

}  // namespace haccsr

// A call that is repeated with the same arguments (every step of a time stepper) is captured
// once as a CUDA graph and replayed: one launch instead of ~20.
struct GraphKey {   // compared with memcmp: always zero-filled first
    uint32_t kind;
    int32_t i[7];
    int64_t n;
    uint64_t p[16];
    float f[12];
};
struct GraphSlot {
    GraphKey key;
    cudaGraphExec_t exec;
    uint64_t stamp;
};
constexpr int kGraphSlots = 8;

struct haccsr_ctx {
    int64_t n_max = 0;
    int64_t n = 0;
    int nc = 0;
    int nz = 0;                 // cell layers of the z window (== nc: the whole periodic box)
    int cz0 = 0;                // global index of window layer 0
    int64_t n_cells = 0;        // nc * nc * nz
    float box_l = 0.f;
    bool scale_exact = false;   // nc/L exactly representable in float32
    cudaStream_t stream = nullptr;
    int device = 0;             // the device current at haccsr_create; every call runs on it
    int n_sms = 0;

    // workspace carve-up (device)
    uint32_t *cell_start = nullptr;   // [n_cells+1]
    uint32_t *row_count = nullptr;    // [nc^2+1]    particles per (cz,cy) row
    uint32_t *row_start = nullptr;    // [nc^2+1]    exclusive scan of row_count (final layout)
    uint32_t *row_pad = nullptr;      // [nc^2+1]    (row_start[r] + 3 r + 3) & ~3:
                                      //             row starts in the sort's intermediate arrays
    uint32_t *row_cursor = nullptr;   // [nc^2]      sort pass 2 write cursors
    uint32_t *slab_cursor = nullptr;  // [nc]        sort pass 1 write cursors
    uint32_t *slab_count = nullptr;   // [nc]        particles per z slab
    uint32_t *tile_start = nullptr;   // [nc+1]      first slab-aligned tile of each slab
    uint32_t *row_first = nullptr;    // [1025]      first row owned by each CTA of sort pass 3
    uint32_t *cell_sources = nullptr; // [n_cells]   S_c = sum of the 27 neighbour counts
    uint32_t *item_count = nullptr;   // [2*n_cells+1] dense-cell items | sparse-cell items
    uint32_t *item_start = nullptr;   // [2*n_cells+1] exclusive scan of item_count
    uint32_t *scan_blocks = nullptr;  // [(2 nc^3+1)/kScanTile + 4] block sums of the largest scan
    uint32_t *cid = nullptr;          // [n_max] original order; filled on demand (get_mesh)
    uint32_t *cell_mid = nullptr;     // [n_cells]   multi-level stepping: end of the cell's
                                      //             active part (particles of the kicked level)
    // the four particle arrays hold n_max + 3 nc^2 + 8 slots: as intermediates of the sort
    // every row is padded to a multiple of 4 records (even slots, 16-byte aligned indices)
    float4 *tmp_pos = nullptr;        // records partitioned by (cz,cy) row (sort pass 2)
    uint32_t *tmp_idx = nullptr;      // original index, same order (masses given only)
    uint32_t *perm = nullptr;         // [n] sorted slot -> original index
    float4 *sorted = nullptr;         // [n] {x,y,z,m} in cell order
    haccsr::WorkItem *items = nullptr; // [max_items]
    int64_t max_items = 0;
    haccsr::DeviceStats *stats = nullptr;

    // captured calls (api.cu)
    bool use_graphs = true;
    uint64_t graph_clock = 0;
    GraphSlot graphs[kGraphSlots] = {};

    // state
    bool binned = false;
    bool have_force = false;
    bool unit_mass = true;
    bool pre_drift = false;      // hacc_sr_subcycle: the next bin's first pass streams the
    float pre_drift_dt = 0.f;    // positions by this step first (sort.cu, k_count_rows<true>)
    const uint8_t *act_level = nullptr;  // multi-level stepping: per-particle levels and the
    int act_k = 0;                       // level whose particles the next bin puts first
    float *vx = nullptr, *vy = nullptr, *vz = nullptr;
    float *ax = nullptr, *ay = nullptr, *az = nullptr;
};

namespace haccsr {

int64_t max_items_for(int64_t n_max, int64_t n_cells);

// sort.cu
cudaError_t configure_sort_kernels();
cudaError_t launch_sort(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                        const float *mass);
// bin.cu
cudaError_t scan_u32(haccsr_ctx *c, const uint32_t *in, int64_t n, uint32_t *out, uint32_t *copy);
cudaError_t launch_bin(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                       const float *mass);
cudaError_t launch_worklist(haccsr_ctx *c, const uint32_t *mid);
cudaError_t launch_cell_ids(haccsr_ctx *c);
cudaError_t launch_kick(haccsr_ctx *c, float dt);
cudaError_t launch_drift(haccsr_ctx *c, int64_t n, float *x, float *y, float *z, const float *vx,
                         const float *vy, const float *vz, float dt);

// levels.cu (multi-level time stepping)
cudaError_t launch_assign_levels(haccsr_ctx *c, int64_t n, const float *x, const float *y,
                                 const float *z, float d, int l_min, int l_max, uint8_t *level);
cudaError_t launch_accumulate_evals(haccsr_ctx *c, unsigned long long *evals);

// shard.cu
cudaError_t launch_pack_layer(haccsr_ctx *c, int64_t n, const float *x, const float *y,
                              const float *z, const float *mass, int layer, float4 *out,
                              uint32_t capacity, uint32_t *count);
cudaError_t launch_unpack(haccsr_ctx *c, int64_t n, const float4 *in, float *x, float *y,
                          float *z, float *mass);

// force.cu
struct ForceArgs {
    float eps, r_max, dt;
    float poly[6];
    bool kick;
    float *ax, *ay, *az;
    uint32_t *nbr;
    unsigned long long *pair_total;
};
cudaError_t launch_force(haccsr_ctx *c, const ForceArgs &a);

}  // namespace haccsr
