// api.cu -- the C ABI of include/haccsr.h: argument checking, workspace carve-up, state.
#include <cmath>
#include <cstddef>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ctx.h"

using namespace haccsr;

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) & ~(kAlign - 1); }

struct Layout {
    size_t cell_start, row_count, row_start, row_pad, row_cursor, slab_cursor, slab_count,
        tile_start, row_first, cell_sources, cell_mid, item_count, item_start, scan_blocks, cid, perm,
        sorted, items, stats, tmp_pos, tmp_idx, total;
    int64_t max_items;
};

// nz: cell layers of the context's z window (nc for the whole box, nz_own + 2 for a slab)
bool layout_for(int64_t n_max, int nc, int nz, Layout &l)
{
    if (n_max < 1 || n_max >= (int64_t(1) << 31) || nc < 4 || nc > 256) return false;
    if (nz < 3 || nz > nc) return false;
    const int64_t cells = (int64_t)nc * nc * nz;
    l.max_items = max_items_for(n_max, cells);
    size_t o = 0;
    auto take = [&](size_t bytes) {
        size_t at = o;
        o = align_up(o + bytes);
        return at;
    };
    l.cell_start = take(sizeof(uint32_t) * (cells + 1));
    const int64_t rows = (int64_t)nc * nz;
    l.row_count = take(sizeof(uint32_t) * (rows + 1));
    l.row_start = take(sizeof(uint32_t) * (rows + 1));
    l.row_pad = take(sizeof(uint32_t) * (rows + 1));
    l.row_cursor = take(sizeof(uint32_t) * rows);
    l.slab_cursor = take(sizeof(uint32_t) * nz);
    l.slab_count = take(sizeof(uint32_t) * nz);
    l.tile_start = take(sizeof(uint32_t) * (nz + 1));
    l.row_first = take(sizeof(uint32_t) * 1025);
    l.cell_sources = take(sizeof(uint32_t) * cells);
    l.cell_mid = take(sizeof(uint32_t) * cells);
    l.item_count = take(sizeof(uint32_t) * (2 * cells + 1));
    l.item_start = take(sizeof(uint32_t) * (2 * cells + 1));
    l.scan_blocks = take(sizeof(uint32_t) * ((2 * cells + 1) / kScanTile + 4));
    l.cid = take(sizeof(uint32_t) * n_max);
    // intermediates of the sort: every row starts on a multiple of 4 records (row_pad_of)
    const int64_t n_pad = n_max + 3 * rows + 8;
    l.perm = take(sizeof(uint32_t) * n_pad);
    l.sorted = take(sizeof(float4) * n_pad);
    l.items = take(sizeof(WorkItem) * l.max_items);
    l.stats = take(sizeof(DeviceStats));
    l.tmp_pos = take(sizeof(float4) * n_pad);
    l.tmp_idx = take(sizeof(uint32_t) * n_pad);
    l.total = o;
    return true;
}

inline int cuda_status(cudaError_t e) { return e == cudaSuccess ? HACCSR_OK : HACCSR_ECUDA; }

// Every ABI call runs on the device the context was created on, whatever device the calling
// thread has current, and restores the caller's device on return.
class DeviceGuard {
public:
    explicit DeviceGuard(const haccsr_ctx *c)
    {
        ok_ = cudaGetDevice(&prev_) == cudaSuccess;
        want_ = c ? c->device : prev_;
        if (ok_ && prev_ != want_) ok_ = cudaSetDevice(want_) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (ok_ && prev_ != want_) cudaSetDevice(prev_);
    }
    bool ok() const { return ok_; }

private:
    int prev_ = 0, want_ = 0;
    bool ok_ = false;
};

// Smallest accepted softening: the self pair and coincident pairs go through the arithmetic
// with u = eps and rely on f * 0 = 0, so q^3 = eps^(-3/2) must stay finite and eps must not
// be flushed to zero (include/haccsr.h).
constexpr float kMinEps = 1e-20f;

// Argument checks of a force evaluation that do not depend on the mesh state.
int check_force_params(haccsr_ctx *c, float eps, float r_max, const float *poly, float *ax,
                       float *ay, float *az)
{
    if (!c || !poly || !ax || !ay || !az) return HACCSR_EINVAL;
    if (!(eps >= kMinEps) || !std::isfinite(eps)) return HACCSR_EINVAL;
    if (!(r_max > 0.f) || !((double)r_max <= (double)c->box_l / (double)c->nc))
        return HACCSR_EINVAL;
    for (int k = 0; k < 6; ++k)
        if (!std::isfinite(poly[k])) return HACCSR_EINVAL;
    return HACCSR_OK;
}

inline GraphKey make_key(uint32_t kind, int64_t n)
{
    GraphKey k;
    std::memset(&k, 0, sizeof(k));
    k.kind = kind;
    k.n = n;
    return k;
}

inline uint64_t key_ptr(const void *p) { return (uint64_t) reinterpret_cast<uintptr_t>(p); }

// Run `enqueue` (which only enqueues work on the context's stream and returns a status) as a
// cached CUDA graph: replay it if this exact call was captured before, else capture,
// instantiate and launch it.  Falls back to plain enqueueing when graphs are switched off
// (HACCSR_GRAPHS=0), when the stream cannot be captured (the legacy default stream) or is
// already being captured by the caller.
template <class F>
int run_graphed(haccsr_ctx *c, const GraphKey &key, F enqueue)
{
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (!c->use_graphs || cudaStreamIsCapturing(c->stream, &cap) != cudaSuccess ||
        cap != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return enqueue();
    }
    for (GraphSlot &g : c->graphs)
        if (g.exec && std::memcmp(&g.key, &key, sizeof(key)) == 0) {
            g.stamp = ++c->graph_clock;
            return cuda_status(cudaGraphLaunch(g.exec, c->stream));
        }
    GraphSlot *victim = &c->graphs[0];  // an empty slot, else the least recently used one
    for (GraphSlot &g : c->graphs)
        if (!g.exec || (victim->exec && g.stamp < victim->stamp)) {
            victim = &g;
            if (!g.exec) break;
        }
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
        cudaGetLastError();
        return enqueue();
    }
    const int s = enqueue();
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (s != HACCSR_OK || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return s != HACCSR_OK ? s : HACCSR_ECUDA;
    }
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ei = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess || !exec) {
        cudaGetLastError();
        return enqueue();  // nothing ran during the capture: enqueue it for real
    }
    if (victim->exec) cudaGraphExecDestroy(victim->exec);
    victim->key = key;
    victim->exec = exec;
    victim->stamp = ++c->graph_clock;
    return cuda_status(cudaGraphLaunch(exec, c->stream));
}

int check_force_args(haccsr_ctx *c, float eps, float r_max, const float *poly, float *ax,
                     float *ay, float *az)
{
    const int s = check_force_params(c, eps, r_max, poly, ax, ay, az);
    if (s) return s;
    return c->binned ? HACCSR_OK : HACCSR_ESTATE;
}

int run_force(haccsr_ctx *c, float eps, float r_max, const float *poly, float dt, bool kick,
              float *ax, float *ay, float *az, uint32_t *nbr, uint64_t *pair_total)
{
    int s = check_force_args(c, eps, r_max, poly, ax, ay, az);
    if (s) return s;
    if (kick && !(c->vx && c->vy && c->vz)) return HACCSR_ESTATE;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    ForceArgs a;
    a.eps = eps;
    a.r_max = r_max;
    a.dt = dt;
    for (int k = 0; k < 6; ++k) a.poly[k] = poly[k];
    a.kick = kick;
    a.ax = ax; a.ay = ay; a.az = az;
    a.nbr = nbr;
    a.pair_total = reinterpret_cast<unsigned long long *>(pair_total);
    GraphKey key = make_key(kick ? 2u : 3u, c->n);
    const void *ptrs[] = {ax, ay, az, nbr, pair_total, c->vx, c->vy, c->vz};
    for (int k = 0; k < 8; ++k) key.p[k] = key_ptr(ptrs[k]);
    key.f[0] = eps; key.f[1] = r_max; key.f[2] = dt;
    for (int k = 0; k < 6; ++k) key.f[3 + k] = poly[k];
    key.i[0] = c->unit_mass;
    s = run_graphed(c, key, [&] { return cuda_status(launch_force(c, a)); });
    if (s) return s;
    c->ax = ax; c->ay = ay; c->az = az;
    c->have_force = true;
    return HACCSR_OK;
}

}  // namespace

extern "C" {

int haccsr_abi_version(void) { return 2; }

size_t haccsr_workspace_bytes(int64_t n_max, int nc)
{
    Layout l;
    return layout_for(n_max, nc, nc, l) ? l.total : 0;
}

size_t haccsr_workspace_bytes_slab(int64_t n_max, int nc, int nz_own)
{
    Layout l;
    if (nz_own < 1 || nz_own > nc - 2) return 0;
    return layout_for(n_max, nc, nz_own + 2, l) ? l.total : 0;
}

static int create_ctx(haccsr_ctx **out, int64_t n_max, float box_L, int nc, int nz, int cz0,
                      void *workspace, size_t workspace_bytes, void *cuda_stream);

int haccsr_create(haccsr_ctx **out, int64_t n_max, float box_L, int nc, void *workspace,
                  size_t workspace_bytes, void *cuda_stream)
{
    return create_ctx(out, n_max, box_L, nc, nc, 0, workspace, workspace_bytes, cuda_stream);
}

int haccsr_create_slab(haccsr_ctx **out, int64_t n_max, float box_L, int nc, int cz_lo,
                       int nz_own, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (out) *out = nullptr;
    if (nc < 4 || nz_own < 1 || nz_own > nc - 2 || cz_lo < 0 || cz_lo >= nc) return HACCSR_EINVAL;
    // the window: one passive layer below the owned layers, one above (periodic in z)
    return create_ctx(out, n_max, box_L, nc, nz_own + 2, (cz_lo + nc - 1) % nc, workspace,
                      workspace_bytes, cuda_stream);
}

static int create_ctx(haccsr_ctx **out, int64_t n_max, float box_L, int nc, int nz, int cz0,
                      void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return HACCSR_EINVAL;
    *out = nullptr;
    Layout l;
    if (!layout_for(n_max, nc, nz, l)) return HACCSR_EINVAL;
    if (!(box_L > 0.f) || !std::isfinite(box_L)) return HACCSR_EINVAL;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & (kAlign - 1)))
        return HACCSR_EINVAL;
    if (workspace_bytes < l.total) return HACCSR_ENOMEM;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HACCSR_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return HACCSR_ECUDA;
    haccsr_ctx *c = new (std::nothrow) haccsr_ctx();
    if (!c) return HACCSR_ENOMEM;
    c->n_max = n_max;
    c->nc = nc;
    c->nz = nz;
    c->cz0 = cz0;
    c->n_cells = (int64_t)nc * nc * nz;
    c->box_l = box_L;
    const double scale = (double)nc / (double)box_L;
    c->scale_exact = ((double)(float)scale == scale);
    c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    c->device = dev;
    const char *env = std::getenv("HACCSR_GRAPHS");
    c->use_graphs = !(env && env[0] == '0');
    c->n_sms = sms;
    char *w = static_cast<char *>(workspace);
    c->cell_start = reinterpret_cast<uint32_t *>(w + l.cell_start);
    c->row_count = reinterpret_cast<uint32_t *>(w + l.row_count);
    c->row_start = reinterpret_cast<uint32_t *>(w + l.row_start);
    c->row_pad = reinterpret_cast<uint32_t *>(w + l.row_pad);
    c->row_cursor = reinterpret_cast<uint32_t *>(w + l.row_cursor);
    c->slab_cursor = reinterpret_cast<uint32_t *>(w + l.slab_cursor);
    c->slab_count = reinterpret_cast<uint32_t *>(w + l.slab_count);
    c->tile_start = reinterpret_cast<uint32_t *>(w + l.tile_start);
    c->row_first = reinterpret_cast<uint32_t *>(w + l.row_first);
    c->cell_sources = reinterpret_cast<uint32_t *>(w + l.cell_sources);
    c->cell_mid = reinterpret_cast<uint32_t *>(w + l.cell_mid);
    c->item_count = reinterpret_cast<uint32_t *>(w + l.item_count);
    c->item_start = reinterpret_cast<uint32_t *>(w + l.item_start);
    c->scan_blocks = reinterpret_cast<uint32_t *>(w + l.scan_blocks);
    c->cid = reinterpret_cast<uint32_t *>(w + l.cid);
    c->perm = reinterpret_cast<uint32_t *>(w + l.perm);
    c->sorted = reinterpret_cast<float4 *>(w + l.sorted);
    c->items = reinterpret_cast<WorkItem *>(w + l.items);
    c->max_items = l.max_items;
    c->stats = reinterpret_cast<DeviceStats *>(w + l.stats);
    c->tmp_pos = reinterpret_cast<float4 *>(w + l.tmp_pos);
    c->tmp_idx = reinterpret_cast<uint32_t *>(w + l.tmp_idx);
    if (configure_sort_kernels() != cudaSuccess ||
        cudaMemsetAsync(c->stats, 0, sizeof(DeviceStats), c->stream) != cudaSuccess) {
        delete c;
        return HACCSR_ECUDA;
    }
    *out = c;
    return HACCSR_OK;
}

int haccsr_destroy(haccsr_ctx *ctx)
{
    if (!ctx) return HACCSR_EINVAL;
    {
        DeviceGuard guard(ctx);
        if (guard.ok()) cudaStreamSynchronize(ctx->stream);
        for (GraphSlot &g : ctx->graphs)
            if (g.exec) cudaGraphExecDestroy(g.exec);
    }
    delete ctx;
    return HACCSR_OK;
}

int hacc_sr_bin(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                const float *mass, float *vx, float *vy, float *vz)
{
    if (!c || n < 0 || n > c->n_max) return HACCSR_EINVAL;
    if (n > 0 && (!x || !y || !z)) return HACCSR_EINVAL;
    const int nv = (vx != nullptr) + (vy != nullptr) + (vz != nullptr);
    if (nv != 0 && nv != 3) return HACCSR_EINVAL;
    c->n = n;
    c->unit_mass = (mass == nullptr);
    c->vx = vx; c->vy = vy; c->vz = vz;
    c->have_force = false;
    c->binned = false;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    GraphKey key = make_key(1u, n);
    const void *ptrs[] = {x, y, z, mass, vx, vy, vz, c->act_level};
    for (int k = 0; k < 8; ++k) key.p[k] = key_ptr(ptrs[k]);
    key.i[0] = c->act_k;
    key.i[1] = c->pre_drift;
    key.f[0] = c->pre_drift_dt;
    const int s = run_graphed(c, key, [&] { return cuda_status(launch_bin(c, n, x, y, z, mass)); });
    if (s) return s;
    c->binned = true;
    return HACCSR_OK;
}

int hacc_sr_force(haccsr_ctx *c, float eps, float r_max, const float *poly, float *ax, float *ay,
                  float *az, uint32_t *nbr_count, uint64_t *pair_total)
{
    return run_force(c, eps, r_max, poly, 0.f, false, ax, ay, az, nbr_count, pair_total);
}

int hacc_sr_force_kick(haccsr_ctx *c, float eps, float r_max, const float *poly, float dt,
                       float *ax, float *ay, float *az, uint32_t *nbr_count,
                       uint64_t *pair_total)
{
    return run_force(c, eps, r_max, poly, dt, true, ax, ay, az, nbr_count, pair_total);
}

int hacc_sr_kick(haccsr_ctx *c, float dt)
{
    if (!c) return HACCSR_EINVAL;
    if (!c->have_force || !(c->vx && c->vy && c->vz)) return HACCSR_ESTATE;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    return cuda_status(launch_kick(c, dt));
}

int hacc_sr_drift(haccsr_ctx *c, int64_t n, float *x, float *y, float *z, const float *vx,
                  const float *vy, const float *vz, float dt)
{
    if (!c || n < 0) return HACCSR_EINVAL;
    if (n > 0 && (!x || !y || !z || !vx || !vy || !vz)) return HACCSR_EINVAL;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    return cuda_status(launch_drift(c, n, x, y, z, vx, vy, vz, dt));
}

int hacc_sr_subcycle(haccsr_ctx *c, int64_t n, float *x, float *y, float *z, const float *mass,
                     float *vx, float *vy, float *vz, float eps, float r_max, const float *poly,
                     float dt, int n_sub, float *ax, float *ay, float *az)
{
    // every argument is checked before the first kernel is enqueued: an error return leaves
    // the caller's arrays untouched
    if (!c || n_sub < 1 || !std::isfinite(dt)) return HACCSR_EINVAL;
    if (n < 0 || n > c->n_max) return HACCSR_EINVAL;
    if (!vx || !vy || !vz) return HACCSR_EINVAL;
    if (n > 0 && (!x || !y || !z)) return HACCSR_EINVAL;
    int s = check_force_params(c, eps, r_max, poly, ax, ay, az);
    if (s) return s;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    // S(dt/2) K(dt) [S(dt) K(dt)]^(n_sub-1) S(dt/2): every stream that is followed by a kick
    // rides in the first pass of that kick's binning (k_count_rows<true>); the whole map is
    // one CUDA graph
    GraphKey key = make_key(4u, n);
    const void *ptrs[] = {x, y, z, mass, vx, vy, vz, ax, ay, az};
    for (int k = 0; k < 10; ++k) key.p[k] = key_ptr(ptrs[k]);
    key.f[0] = eps; key.f[1] = r_max; key.f[2] = dt;
    for (int k = 0; k < 6; ++k) key.f[3 + k] = poly[k];
    key.i[0] = n_sub;
    s = run_graphed(c, key, [&] {
        int st = HACCSR_OK;
        for (int k = 0; k < n_sub && st == HACCSR_OK; ++k) {
            c->pre_drift = true;
            c->pre_drift_dt = (k == 0) ? 0.5f * dt : dt;
            st = hacc_sr_bin(c, n, x, y, z, mass, vx, vy, vz);
            c->pre_drift = false;
            if (st) break;
            st = hacc_sr_force_kick(c, eps, r_max, poly, dt, ax, ay, az, nullptr, nullptr);
        }
        if (st == HACCSR_OK) st = hacc_sr_drift(c, n, x, y, z, vx, vy, vz, 0.5f * dt);
        return st;
    });
    c->pre_drift = false;
    if (s) return s;
    // the state the calls above leave behind (they do not run when the graph is replayed)
    c->n = n;
    c->unit_mass = (mass == nullptr);
    c->vx = vx; c->vy = vy; c->vz = vz;
    c->ax = ax; c->ay = ay; c->az = az;
    c->binned = true;
    c->have_force = true;
    return HACCSR_OK;
}

int hacc_sr_subcycle_multilevel(haccsr_ctx *c, int64_t n, float *x, float *y, float *z,
                                const float *mass, float *vx, float *vy, float *vz, float eps,
                                float r_max, const float *poly, float T, float d, int l_min,
                                int l_max, float *ax, float *ay, float *az, uint8_t *level,
                                uint64_t *evals)
{
    // every argument is checked before the first kernel is enqueued
    if (!c || !std::isfinite(T) || !(d > 0.f) || !std::isfinite(d) || !level) return HACCSR_EINVAL;
    if (c->nz < c->nc) return HACCSR_EINVAL;  // rho0 is the mean of the WHOLE box: not on a slab
    if (l_min < 1 || l_max < l_min || l_max > 64 || (l_min & (l_min - 1)) || (l_max & (l_max - 1)))
        return HACCSR_EINVAL;
    if (n < 0 || n > c->n_max || !vx || !vy || !vz) return HACCSR_EINVAL;
    if (n > 0 && (!x || !y || !z)) return HACCSR_EINVAL;
    int s = check_force_params(c, eps, r_max, poly, ax, ay, az);
    if (s) return s;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    int lm = 0;
    while ((1 << lm) < l_max) ++lm;
    unsigned long long *ev = reinterpret_cast<unsigned long long *>(evals);
    GraphKey key = make_key(5u, n);
    const void *ptrs[] = {x, y, z, mass, vx, vy, vz, ax, ay, az, level, evals};
    for (int k = 0; k < 12; ++k) key.p[k] = key_ptr(ptrs[k]);
    key.f[0] = eps; key.f[1] = r_max; key.f[2] = T; key.f[3] = d;
    for (int k = 0; k < 6; ++k) key.f[4 + k] = poly[k];
    key.i[0] = l_min;
    key.i[1] = l_max;
    s = run_graphed(c, key, [&] {
        int st;
        if (ev && cudaMemsetAsync(ev, 0, sizeof(*ev), c->stream) != cudaSuccess)
            return (int)HACCSR_ECUDA;
        // levels from the cell occupancies at the beginning of the long step
        if ((st = hacc_sr_bin(c, n, x, y, z, mass, vx, vy, vz))) return st;
        if (launch_assign_levels(c, n, x, y, z, d, l_min, l_max, level) != cudaSuccess)
            return (int)HACCSR_ECUDA;
        const float half = 0.5f * T / (float)l_max;
        for (int h = 1; h <= 2 * l_max; ++h) {
            int v2 = 0;
            while (!((h >> v2) & 1)) ++v2;
            const int k = lm - v2;   // the level whose SKS midpoints fall on this half stream
            if (k < 0) {             // nobody is kicked: a plain stream
                if ((st = hacc_sr_drift(c, n, x, y, z, vx, vy, vz, half))) return st;
                continue;
            }
            // the half stream rides in the binning's first pass; the mesh of the streamed
            // positions has the particles of level k first in every cell
            c->act_level = level;
            c->act_k = k;
            c->pre_drift = true;
            c->pre_drift_dt = half;
            st = hacc_sr_bin(c, n, x, y, z, mass, vx, vy, vz);
            c->act_level = nullptr;
            c->pre_drift = false;
            if (st) return st;
            if (ev && launch_accumulate_evals(c, ev) != cudaSuccess) return (int)HACCSR_ECUDA;
            if ((st = run_force(c, eps, r_max, poly, T / (float)(1 << k), true, ax, ay, az,
                                nullptr, nullptr)))
                return st;
        }
        return (int)HACCSR_OK;
    });
    c->act_level = nullptr;
    c->pre_drift = false;
    if (s) return s;
    c->n = n;
    c->unit_mass = (mass == nullptr);
    c->vx = vx; c->vy = vy; c->vz = vz;
    c->ax = ax; c->ay = ay; c->az = az;
    c->binned = true;
    c->have_force = true;
    return HACCSR_OK;
}

int hacc_sr_pack_layer(haccsr_ctx *c, int64_t n, const float *x, const float *y, const float *z,
                       const float *mass, int cz_layer, float *out_records, int64_t capacity,
                       uint32_t *count)
{
    if (!c || n < 0 || capacity < 0 || capacity >= (int64_t(1) << 32) || !count)
        return HACCSR_EINVAL;
    if (cz_layer < 0 || cz_layer >= c->nc) return HACCSR_EINVAL;
    if (n > 0 && (!x || !y || !z)) return HACCSR_EINVAL;
    if (capacity > 0 && !out_records) return HACCSR_EINVAL;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    return cuda_status(launch_pack_layer(c, n, x, y, z, mass, cz_layer,
                                         reinterpret_cast<float4 *>(out_records),
                                         (uint32_t)capacity, count));
}

int hacc_sr_unpack(haccsr_ctx *c, int64_t n, const float *records, float *x, float *y, float *z,
                   float *mass)
{
    if (!c || n < 0) return HACCSR_EINVAL;
    if (n > 0 && (!records || !x || !y || !z)) return HACCSR_EINVAL;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    return cuda_status(
        launch_unpack(c, n, reinterpret_cast<const float4 *>(records), x, y, z, mass));
}

int haccsr_get_mesh(haccsr_ctx *c, const uint32_t **cell_start, const uint32_t **perm,
                    const float **sorted_pos, const uint32_t **cell_id)
{
    if (!c) return HACCSR_EINVAL;
    if (!c->binned) return HACCSR_ESTATE;
    if (cell_start) *cell_start = c->cell_start;
    if (perm) *perm = c->perm;
    if (sorted_pos) *sorted_pos = reinterpret_cast<const float *>(c->sorted);
    if (cell_id) {
        DeviceGuard guard(c);
        if (!guard.ok() || launch_cell_ids(c) != cudaSuccess) return HACCSR_ECUDA;
        *cell_id = c->cid;
    }
    return HACCSR_OK;
}

int haccsr_get_stats(haccsr_ctx *c, haccsr_stats *out)
{
    if (!c || !out) return HACCSR_EINVAL;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    DeviceStats d;
    if (cudaMemcpyAsync(&d, c->stats, sizeof(d), cudaMemcpyDeviceToHost, c->stream) !=
        cudaSuccess)
        return HACCSR_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HACCSR_ECUDA;
    out->n = c->n;
    out->n_cells = c->n_cells;
    out->n_eval = d.n_eval;
    out->n_items = d.n_items;
    out->n_split_items = d.n_split_items;
    out->max_cell_count = d.max_cell_count;
    out->sources_per_split = d.sources_per_split;
    out->n_recheck_tiles = d.n_recheck_tiles;
    return HACCSR_OK;
}

int haccsr_sync(haccsr_ctx *c)
{
    if (!c) return HACCSR_EINVAL;
    DeviceGuard guard(c);
    if (!guard.ok()) return HACCSR_ECUDA;
    int32_t flag = 0;
    if (cudaMemcpyAsync(&flag, &c->stats->error_flag, sizeof(flag), cudaMemcpyDeviceToHost,
                        c->stream) != cudaSuccess)
        return HACCSR_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HACCSR_ECUDA;
    if (flag != 0) {
        cudaMemsetAsync(&c->stats->error_flag, 0, sizeof(flag), c->stream);
        return flag;
    }
    return HACCSR_OK;
}

const char *haccsr_strerror(int s)
{
    switch (s) {
    case HACCSR_OK: return "ok";
    case HACCSR_EINVAL: return "invalid argument";
    case HACCSR_ESTATE: return "call out of order (bin -> force -> kick)";
    case HACCSR_ENOMEM: return "workspace too small";
    case HACCSR_ECUDA: return "CUDA runtime error (is there a device?)";
    case HACCSR_EDATA: return "non-finite particle position";
    default: return "unknown status";
    }
}

}  // extern "C"
