// force.cu -- the short-range force kernel (Eq. 12) with the kick
// fused into its epilogue.
//
// Design:
//   * persistent warps pull 16-byte work items (cell, target chunk, source chunk) from a
//     global counter -- the paper's dynamic work queue at warp granularity;
//   * a warp holds 32*T targets in registers (T = 1 sparse cells, up to T = 4 dense cells) and
//     streams
//     the cell's flat 27-neighbour source list through a private, double-buffered
//     shared-memory tile in SoA form, "pre-generated into a contiguous array",
//     with the periodic image shift applied while staging;
//   * the pair arithmetic is packed two sources at a time in fma.rn.f32x2 / add.f32x2 /
//     mul.f32x2 (one issue slot for two FMAs), rsqrt on the SFU, the polynomial re-centred in
//     u = s + eps and negated so that f = q^2*q - Q(u) is one FMA, Horner form;
//   * the cutoff is a select.  Pairs whose float32 u lies within +-8 ulp of the
//     cutoff are left out of the fast path and decided in FP64 by a rare per-tile fix-up pass,
//     so that the interacting-pair set is exactly {s < r_max^2} for the float32 inputs.
#include <cstddef>
#include <cstdlib>

#include "ctx.h"

namespace haccsr {

// Launch shape and unrolling were chosen by measurement on configs[3]:
// 16 warps x 1 CTA per SM beats 8 x 2 by 1 %, four 4-source groups per iteration of the T >= 3
// pair loop beat one by 3 % (for T <= 2 four beat two by 0.3-0.7 % once the T = 1 items had
// their own 32-warp kernel; in round 1's single kernel two were better), 64-source tiles beat 128.
constexpr int kWarpsPerBlock = 16;
constexpr int kBlocksPerSm = 1;
constexpr int kUnrollLo = 4;       // 4-source groups per iteration of the pair loop, T <= 2
constexpr int kUnrollHi = 4;       // same, T >= 3
constexpr int kSrcPerLane = 2;     // sources each lane stages per tile
constexpr int kTile = 32 * kSrcPerLane;  // sources per shared-memory tile
constexpr uint32_t kBandHalf = 8;  // guard band: +-8 float32 ulps of (r_max^2 + eps)
constexpr int kSegs = 18;          // 9 rows x (main piece, x-wrap piece)
constexpr float kFar = 1.0e9f;     // padding sources / idle target lanes live out here

struct ForceParams {
    const float4 *sorted;
    const uint32_t *cell_start;
    const uint32_t *perm;
    const WorkItem *items;
    DeviceStats *stats;
    float *ax, *ay, *az;
    float *vx, *vy, *vz;  // null unless kick
    uint32_t *nbr;
    unsigned long long *pair_total;
    double rm2;        // exact cutoff r_max^2 (double of the float32 r_max)
    float box_l;
    float eps;
    float cut_lo;      // float with bit pattern lo_bits: u < cut_lo  =>  surely inside
    uint32_t lo_bits;  // bits(fl(r_max^2+eps)) - kBandHalf
    float dt;
    float nq[6];       // -Q_k, Q(u) = P(u - eps); the fix-up path evaluates the same form
    int nc;
    int nz, cz0;       // the context's z window (nz == nc: the whole periodic box)
    int split_sparse;  // the sparse cells' items are left to k_force_sparse
};

struct __align__(16) WarpTile {
    float sx[2][kTile], sy[2][kTile], sz[2][kTile], sm[2][kTile];
    uint32_t seg_off[kSegs + 2];
    uint32_t seg_base[kSegs];
    uint32_t seg_shift[kSegs];
};

__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float2 dup2(float a) { return make_float2(a, a); }

// u = dx^2 + dy^2 + dz^2 + eps in the fixed order shared by the fast and the fix-up path.
__device__ __forceinline__ float u_of(float dx, float dy, float dz, float eps)
{
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmaf_rn(dx, dx, eps)));
}

// f_SR for one pair from u (scalar form of the packed arithmetic below).
__device__ __forceinline__ float fsr_of(float u, const float *nq)
{
    float q = rsqrt_approx(u);
    float h = nq[5];
    h = __fmaf_rn(h, u, nq[4]);
    h = __fmaf_rn(h, u, nq[3]);
    h = __fmaf_rn(h, u, nq[2]);
    h = __fmaf_rn(h, u, nq[1]);
    h = __fmaf_rn(h, u, nq[0]);
    return __fmaf_rn(__fmul_rn(q, q), q, h);
}

template <int T, bool MASS, bool COUNT>
__device__ __forceinline__ void process_item(const ForceParams &p, WarpTile &w, const WorkItem it,
                                             const int lane)
{
    const int nc = p.nc;
    const uint32_t cell = it.cell;
    const int cx = (int)(cell % (uint32_t)nc);
    const int cy = (int)((cell / (uint32_t)nc) % (uint32_t)nc);
    // lz: layer inside the context's z window (storage); cz: the global layer (periodic frame)
    const int lz = (int)(cell / ((uint32_t)nc * (uint32_t)nc));
    const int cz = (lz + p.cz0 >= nc) ? lz + p.cz0 - nc : lz + p.cz0;
    const bool whole_box = p.nz == nc;
    const int nt = (int)(it.packed >> 24) + 1;
    const bool split = (it.packed >> 23) & 1u;
    const float L = p.box_l;

    // ---- segment table: lanes 0..17 each describe one contiguous piece of the source list --
    {
        uint32_t len = 0, base = 0, shift = 0;
        if (lane < kSegs) {
            const int row = lane % 9, piece = lane / 9;
            int qy = cy + (row % 3) - 1, qz = cz + (row / 3) - 1;
            // where the neighbour row is stored: a slab's targets have both z neighbours
            // inside the window, the whole box wraps
            int ql = lz + (row / 3) - 1;
            qy += (qy < 0) ? nc : 0;
            qy -= (qy >= nc) ? nc : 0;
            qz += (qz < 0) ? nc : 0;
            qz -= (qz >= nc) ? nc : 0;
            if (whole_box) ql = qz;
            // frame rule: a coordinate is shifted by -L when it is in the top layers and the
            // target cell is in the top layer, or when it is the top layer wrapping to cell 0
            const uint32_t shy = ((qy == nc - 1 && cy == 0) || (cy == nc - 1 && qy >= nc - 2));
            const uint32_t shz = ((qz == nc - 1 && cz == 0) || (cz == nc - 1 && qz >= nc - 2));
            const uint32_t rowbase = (uint32_t)nc * (uint32_t)(qy + nc * ql);
            int c0, c1;  // cell range [c0, c1)
            uint32_t shx;
            if (cx == 0) {
                if (piece == 0) { c0 = 0; c1 = 2; shx = 0; }
                else { c0 = nc - 1; c1 = nc; shx = 1; }
            } else if (cx == nc - 1) {
                if (piece == 0) { c0 = nc - 2; c1 = nc; shx = 1; }
                else { c0 = 0; c1 = 1; shx = 0; }
            } else {
                if (piece == 0) { c0 = cx - 1; c1 = cx + 2; shx = 0; }
                else { c0 = 0; c1 = 0; shx = 0; }
            }
            base = __ldg(p.cell_start + rowbase + c0);
            len = __ldg(p.cell_start + rowbase + c1) - base;
            shift = shx | (shy << 1) | (shz << 2);
        }
        uint32_t inc = len;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        __syncwarp();  // previous item's readers of the table are done
        if (lane < kSegs) {
            w.seg_off[lane] = inc - len;
            w.seg_base[lane] = base;
            w.seg_shift[lane] = shift;
        }
        if (lane == kSegs) {
            w.seg_off[kSegs] = inc;        // total sources of the cell
            w.seg_off[kSegs + 1] = 0xffffffffu;
        }
        __syncwarp();
    }
    const uint32_t s_total = w.seg_off[kSegs];
    const uint32_t sps = p.stats->sources_per_split;
    const uint32_t s_begin = it.s_begin;
    const uint32_t s_end = min(s_total, s_begin + (split ? sps : s_total));

    // ---- targets: T per lane, in the frame of the target cell --------------------------------
    const uint32_t t_base = __ldg(p.cell_start + cell) + it.t_begin;
    const float tsx = (cx == nc - 1) ? L : 0.f, tsy = (cy == nc - 1) ? L : 0.f,
                tsz = (cz == nc - 1) ? L : 0.f;
    // T == 1 only: a cell with at most 16 (8, 4, 2) targets runs 2 (4, 8, 16) copies of its
    // targets side by side in the warp, each copy against its own slice of every source tile,
    // and the copies' sums are combined by shuffles at the end -- otherwise most lanes of a
    // sparse cell's warp would idle.
    const int sub = (T == 1) ? (nt <= 2 ? 4 : nt <= 4 ? 3 : nt <= 8 ? 2 : nt <= 16 ? 1 : 0)
                             : 0;  // log2(copies)
    const int tlane = (T == 1) ? (lane & (31 >> sub)) : lane;          // this lane's target
    const int slice = (T == 1) ? (lane >> (5 - sub)) : 0;              // its slice of a tile
    float xi[T], yi[T], zi[T];   // shifted target positions
    float2 nx[T], ny[T], nz[T];  // (-x, -x) ...
    float Ax[T], Ay[T], Az[T];
    uint32_t cnt[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        const int idx = tlane + 32 * t;
        if (idx < nt) {
            float4 q = __ldg(p.sorted + t_base + idx);
            xi[t] = q.x - tsx;
            yi[t] = q.y - tsy;
            zi[t] = q.z - tsz;
        } else {
            xi[t] = yi[t] = zi[t] = -kFar;
        }
        nx[t] = dup2(-xi[t]);
        ny[t] = dup2(-yi[t]);
        nz[t] = dup2(-zi[t]);
        cnt[t] = 0;
    }

    // the loop constants stay in the constant bank / uniform registers: pinning them in
    // ordinary registers was measured 6 % slower (register-file read pressure of FFMA2)
    const float2 eps2 = dup2(p.eps);
    const float2 n5 = dup2(p.nq[5]), n4 = dup2(p.nq[4]), n3 = dup2(p.nq[3]), n2 = dup2(p.nq[2]),
                 n1 = dup2(p.nq[1]), n0 = dup2(p.nq[0]);
    const float cut_lo = p.cut_lo;
    const uint32_t lo_bits = p.lo_bits;

    // only a target cell in the first or last layer of a dimension sees shifted images: every
    // other item stores its sources as they are (measured: configs[3] -0.8 %)
    const bool has_shift = cx == 0 || cx == nc - 1 || cy == 0 || cy == nc - 1 || cz == 0 ||
                           cz == nc - 1;
    // ---- staging: two sources per lane per tile --------------------------------------------
    int cur = 0;  // monotone segment pointer of this lane
    float4 gs[kSrcPerLane];    // staged sources (raw, as loaded)
    uint32_t gshift = 0;       // 3 image-shift bits per staged source, applied when stored
    auto stage_load = [&](uint32_t f0) {
        gshift = 0;
#pragma unroll
        for (int k = 0; k < kSrcPerLane; ++k) {
            const uint32_t f = f0 + 32u * k + lane;
            gs[k] = make_float4(kFar, kFar, kFar, 0.f);
            if (f < s_end) {
                while (f >= w.seg_off[cur + 1]) ++cur;
                const uint32_t src = w.seg_base[cur] + (f - w.seg_off[cur]);
                gshift |= w.seg_shift[cur] << (3 * k);
                gs[k] = __ldg(p.sorted + src);
            }
        }
    };
    auto stage_store = [&](int b) {
        if (has_shift) {
#pragma unroll
            for (int k = 0; k < kSrcPerLane; ++k) {
                const uint32_t sh = gshift >> (3 * k);
                w.sx[b][lane + 32 * k] = gs[k].x - ((sh & 1u) ? L : 0.f);
                w.sy[b][lane + 32 * k] = gs[k].y - ((sh & 2u) ? L : 0.f);
                w.sz[b][lane + 32 * k] = gs[k].z - ((sh & 4u) ? L : 0.f);
                if (MASS) w.sm[b][lane + 32 * k] = gs[k].w;
            }
        } else {
#pragma unroll
            for (int k = 0; k < kSrcPerLane; ++k) {
                w.sx[b][lane + 32 * k] = gs[k].x;
                w.sy[b][lane + 32 * k] = gs[k].y;
                w.sz[b][lane + 32 * k] = gs[k].z;
                if (MASS) w.sm[b][lane + 32 * k] = gs[k].w;
            }
        }
    };

    int buf = 0;
    unsigned long long recheck = 0;
    float2 ax2[T], ay2[T], az2[T];  // running sums over the even / odd sources of the chunk
#pragma unroll
    for (int t = 0; t < T; ++t) ax2[t] = ay2[t] = az2[t] = make_float2(0.f, 0.f);
    if (s_begin < s_end) stage_load(s_begin);
    for (uint32_t f0 = s_begin; f0 < s_end; f0 += kTile) {
        stage_store(buf);
        __syncwarp();
        if (f0 + kTile < s_end) stage_load(f0 + kTile);
        const int ntile = (int)min((uint32_t)kTile, s_end - f0);
        const int ngroups = (ntile + 3) >> 2;

        bool near = false;
        const float4 *X4 = reinterpret_cast<const float4 *>(w.sx[buf]);
        const float4 *Y4 = reinterpret_cast<const float4 *>(w.sy[buf]);
        const float4 *Z4 = reinterpret_cast<const float4 *>(w.sz[buf]);
        const float4 *M4 = reinterpret_cast<const float4 *>(w.sm[buf]);
        // groups of this lane's slice (all of them unless T == 1 runs target copies); a tile
        // is padded to 64 far-away sources, so a slice may run past ngroups
        const int gper = (T == 1) ? ((ngroups + (1 << sub) - 1) >> sub) : ngroups;
        const int g0 = (T == 1) ? slice * gper : 0;
#pragma unroll(T >= 3 ? kUnrollHi : kUnrollLo)
        for (int g = 0; g < gper; ++g) {
            const float4 X = X4[g0 + g], Y = Y4[g0 + g], Z = Z4[g0 + g];
            float4 M = make_float4(1.f, 1.f, 1.f, 1.f);
            if (MASS) M = M4[g0 + g];
#pragma unroll
            for (int t = 0; t < T; ++t) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float2 sx2 = h ? make_float2(X.z, X.w) : make_float2(X.x, X.y);
                    const float2 sy2 = h ? make_float2(Y.z, Y.w) : make_float2(Y.x, Y.y);
                    const float2 sz2 = h ? make_float2(Z.z, Z.w) : make_float2(Z.x, Z.y);
                    const float2 m2 = h ? make_float2(M.z, M.w) : make_float2(M.x, M.y);
                    const float2 dx = __fadd2_rn(sx2, nx[t]);
                    const float2 dy = __fadd2_rn(sy2, ny[t]);
                    const float2 dz = __fadd2_rn(sz2, nz[t]);
                    float2 u = __ffma2_rn(dx, dx, eps2);
                    u = __ffma2_rn(dy, dy, u);
                    u = __ffma2_rn(dz, dz, u);
                    float2 q = make_float2(rsqrt_approx(u.x), rsqrt_approx(u.y));
                    float2 hh = __ffma2_rn(n5, u, n4);
                    hh = __ffma2_rn(hh, u, n3);
                    hh = __ffma2_rn(hh, u, n2);
                    hh = __ffma2_rn(hh, u, n1);
                    hh = __ffma2_rn(hh, u, n0);
                    float2 f = __ffma2_rn(__fmul2_rn(q, q), q, hh);
                    if (MASS) f = __fmul2_rn(f, m2);
                    const bool in0 = u.x < cut_lo, in1 = u.y < cut_lo;
                    f.x = in0 ? f.x : 0.f;
                    f.y = in1 ? f.y : 0.f;
                    near |= (__float_as_uint(u.x) - lo_bits) < 2u * kBandHalf;
                    near |= (__float_as_uint(u.y) - lo_bits) < 2u * kBandHalf;
                    if (COUNT) cnt[t] += (uint32_t)in0 + (uint32_t)in1;
                    ax2[t] = __ffma2_rn(f, dx, ax2[t]);
                    ay2[t] = __ffma2_rn(f, dy, ay2[t]);
                    az2[t] = __ffma2_rn(f, dz, az2[t]);
                }
            }
        }
        // ---- rare: a pair of this tile sits in the guard band; decide it in FP64 -----------
        if (__any_sync(0xffffffffu, near)) {
            ++recheck;
            const int j1 = min(ntile, 4 * (g0 + gper));
            for (int j = 4 * g0; j < j1; ++j) {
                const float xj = w.sx[buf][j], yj = w.sy[buf][j], zj = w.sz[buf][j];
                const float mj = MASS ? w.sm[buf][j] : 1.f;
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    const float dx = __fadd_rn(xj, -xi[t]);
                    const float dy = __fadd_rn(yj, -yi[t]);
                    const float dz = __fadd_rn(zj, -zi[t]);
                    const float u = u_of(dx, dy, dz, p.eps);
                    if ((__float_as_uint(u) - lo_bits) < 2u * kBandHalf) {
                        const double ex = (double)xj - (double)xi[t];
                        const double ey = (double)yj - (double)yi[t];
                        const double ez = (double)zj - (double)zi[t];
                        const double s = ex * ex + ey * ey + ez * ez;
                        if (s < p.rm2) {
                            const float f = fsr_of(u, p.nq) * mj;
                            ax2[t].x = __fmaf_rn(f, dx, ax2[t].x);
                            ay2[t].x = __fmaf_rn(f, dy, ay2[t].x);
                            az2[t].x = __fmaf_rn(f, dz, az2[t].x);
                            if (COUNT) cnt[t] += 1u;
                        }
                    }
                }
            }
        }
        buf ^= 1;
    }

#pragma unroll
    for (int t = 0; t < T; ++t) {
        Ax[t] = ax2[t].x + ax2[t].y;
        Ay[t] = ay2[t].x + ay2[t].y;
        Az[t] = az2[t].x + az2[t].y;
    }
    if (T == 1 && sub) {  // combine the target copies
        for (int d = 16; d >= (32 >> sub); d >>= 1) {
            Ax[0] += __shfl_xor_sync(0xffffffffu, Ax[0], d);
            Ay[0] += __shfl_xor_sync(0xffffffffu, Ay[0], d);
            Az[0] += __shfl_xor_sync(0xffffffffu, Az[0], d);
            if (COUNT) cnt[0] += __shfl_xor_sync(0xffffffffu, cnt[0], d);
        }
    }

    // ---- epilogue: accelerations in original particle order, fused kick ------------------
    unsigned long long my_pairs = 0;
#pragma unroll
    for (int t = 0; t < T; ++t) {
        const int idx = lane + 32 * t;
        if (idx < nt) {
            const uint32_t o = __ldg(p.perm + t_base + idx);
            if (!split) {
                p.ax[o] = Ax[t];
                p.ay[o] = Ay[t];
                p.az[o] = Az[t];
                if (p.vx) {
                    p.vx[o] = __fmaf_rn(p.dt, Ax[t], p.vx[o]);
                    p.vy[o] = __fmaf_rn(p.dt, Ay[t], p.vy[o]);
                    p.vz[o] = __fmaf_rn(p.dt, Az[t], p.vz[o]);
                }
            } else {
                atomicAdd(p.ax + o, Ax[t]);
                atomicAdd(p.ay + o, Ay[t]);
                atomicAdd(p.az + o, Az[t]);
                if (p.vx) {
                    atomicAdd(p.vx + o, p.dt * Ax[t]);
                    atomicAdd(p.vy + o, p.dt * Ay[t]);
                    atomicAdd(p.vz + o, p.dt * Az[t]);
                }
            }
            if (COUNT) {
                // the self pair (d = 0, u = eps) went through the arithmetic once, in the
                // source chunk that starts the list's row of the own cell: chunk 0 holds it
                // only if the own cell's piece lies in it, so subtract where it was counted
                uint32_t c = cnt[t];
                const uint32_t self_f = w.seg_off[4] + (t_base + idx - w.seg_base[4]);
                if (self_f >= s_begin && self_f < s_end) c -= 1u;
                if (p.nbr) {
                    if (!split) p.nbr[o] = c; else atomicAdd(p.nbr + o, c);
                }
                my_pairs += c;
            }
        }
    }
    if (COUNT && p.pair_total) {
#pragma unroll
        for (int d = 16; d; d >>= 1) my_pairs += __shfl_xor_sync(0xffffffffu, my_pairs, d);
        if (lane == 0 && my_pairs) atomicAdd(p.pair_total, my_pairs);
    }
    if (lane == 0 && recheck) atomicAdd(&p.stats->n_recheck_tiles, recheck);
}

template <bool MASS, bool COUNT>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, kBlocksPerSm) k_force(const ForceParams p)
{
    __shared__ WarpTile tiles[kWarpsPerBlock];
    const int lane = threadIdx.x & 31;
    WarpTile &w = tiles[threadIdx.x >> 5];
    const uint32_t n_all = p.stats->n_items;
    const uint32_t n_items = p.split_sparse ? p.stats->n_dense_items : n_all;
    for (;;) {
        uint32_t k = 0;
        if (lane == 0) k = atomicAdd(&p.stats->item_cursor, 1u);
        k = __shfl_sync(0xffffffffu, k, 0);
        if (k >= n_items) break;
        const WorkItem it = p.items[k];
        const uint32_t nt1 = it.packed >> 24;  // targets - 1
        if (nt1 < 32u) process_item<1, MASS, COUNT>(p, w, it, lane);
        else if (nt1 < 64u) process_item<2, MASS, COUNT>(p, w, it, lane);
        else if (nt1 < 96u) process_item<3, MASS, COUNT>(p, w, it, lane);
        else process_item<4, MASS, COUNT>(p, w, it, lane);
        if (p.split_sparse && lane == 0) atomicAdd(&p.stats->dense_done, 1u);
    }
    if (!p.split_sparse) return;
    // Out of dense items while other warps still run theirs (the last items of a halo core
    // take a while): fill the wait with sparse items taken from the back of the list;
    // k_force_sparse, launched next, takes the rest from the front.
    const uint32_t n_sparse = n_all - n_items;
    for (;;) {
        uint32_t s = n_sparse;
        if (lane == 0 && *(volatile uint32_t *)&p.stats->dense_done < n_items)
            s = atomicAdd(&p.stats->steal_cursor, 1u);
        s = __shfl_sync(0xffffffffu, s, 0);
        if (s >= n_sparse) break;
        process_item<1, MASS, COUNT>(p, w, p.items[n_all - 1u - s], lane);
    }
}

// The items of the sparse cells (at most 32 particles: one T = 1 item each, listed after the
// dense cells' items) in a kernel of their own.  These items are bound by latency, not by the
// FMA pipe (item claim, segment table, target and tile loads for a ~400-source list:
// DESIGN.md section 7), and the T = 1 path needs half the registers of the T = 4 loop: at 64
// registers 32 warps per SM hide twice as much of it.
constexpr int kSparseWarps = 16, kSparseBlocksPerSm = 2, kSparseClaim = 1;

template <bool MASS, bool COUNT>
__global__ void __launch_bounds__(kSparseWarps * 32, kSparseBlocksPerSm)
    k_force_sparse(const ForceParams p)
{
    __shared__ WarpTile tiles[kSparseWarps];
    const int lane = threadIdx.x & 31;
    WarpTile &w = tiles[threadIdx.x >> 5];
    // what k_force did not take from the back of the list
    const uint32_t first = p.stats->n_dense_items, n_sparse = p.stats->n_items - first;
    const uint32_t n_items = first + n_sparse - min(p.stats->steal_cursor, n_sparse);
    // items are claimed kSparseClaim at a time.  Claiming 4 saves the dependent round trip to L2
    // of three claims in four and gained 9 % on very sparse uniform points (6.8 per cell), but
    // lengthens the kernel's tail: configs[1] lost 2.7 %, the large configs were unchanged; so 1.
    for (;;) {
        uint32_t k0 = 0;
        if (lane == 0) k0 = first + atomicAdd(&p.stats->sparse_cursor, (uint32_t)kSparseClaim);
        k0 = __shfl_sync(0xffffffffu, k0, 0);
        if (k0 >= n_items) break;
        WorkItem mine = {0, 0, 0, 0};   // lane j holds item k0 + j
        if (lane < kSparseClaim && k0 + lane < n_items) mine = p.items[k0 + lane];
#pragma unroll 1
        for (int j = 0; j < kSparseClaim && k0 + j < n_items; ++j) {
            WorkItem it;
            it.cell = __shfl_sync(0xffffffffu, mine.cell, j);
            it.t_begin = __shfl_sync(0xffffffffu, mine.t_begin, j);
            it.s_begin = __shfl_sync(0xffffffffu, mine.s_begin, j);
            it.packed = __shfl_sync(0xffffffffu, mine.packed, j);
            process_item<1, MASS, COUNT>(p, w, it, lane);
        }
    }
}

// Split items combine with atomics, so the outputs start from zero.
__global__ void __launch_bounds__(256) k_zero_outputs(int64_t n, float *__restrict__ ax,
                                                      float *__restrict__ ay,
                                                      float *__restrict__ az,
                                                      uint32_t *__restrict__ nbr,
                                                      unsigned long long *pair_total,
                                                      DeviceStats *stats)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) {   // and the counters of this evaluation
        stats->n_recheck_tiles = 0;
        stats->item_cursor = stats->sparse_cursor = stats->dense_done = stats->steal_cursor = 0;
        if (pair_total) *pair_total = 0;
    }
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        ax[i] = 0.f;
        ay[i] = 0.f;
        az[i] = 0.f;
        if (nbr) nbr[i] = 0u;
    }
}

// Q(u) = P(u - eps): re-centre the polynomial in double, return the NEGATED coefficients.
static void recentre_negate(const float c[6], double eps, float nq[6])
{
    double q[6] = {0, 0, 0, 0, 0, 0};
    // binomial expansion of sum_j c_j (u - eps)^j
    for (int j = 0; j < 6; ++j) {
        double binom = 1.0;  // C(j,k)
        for (int k = 0; k <= j; ++k) {
            if (k > 0) binom = binom * (double)(j - k + 1) / (double)k;
            double pw = 1.0;
            for (int e = 0; e < j - k; ++e) pw *= -eps;
            q[k] += (double)c[j] * binom * pw;
        }
    }
    for (int k = 0; k < 6; ++k) nq[k] = (float)(-q[k]);
}

cudaError_t launch_force(haccsr_ctx *c, const ForceArgs &a)
{
    cudaStream_t st = c->stream;
    cudaError_t e;
    const int64_t n = c->n;
    if (n == 0) {   // empty mesh: C = 0, nothing else to write
        if (a.pair_total && (e = cudaMemsetAsync(a.pair_total, 0, sizeof(unsigned long long), st)))
            return e;
        return cudaSuccess;
    }
    // split items combine with atomics, so the outputs start from zero: one kernel zeroes
    // them, C and the counters of this evaluation (small problems are launch-bound)
    {
        const int64_t want = (n + 1023) / 1024, cap = (int64_t)c->n_sms * 8;
        k_zero_outputs<<<(int)(want < cap ? want : cap), 256, 0, st>>>(n, a.ax, a.ay, a.az, a.nbr,
                                                                       a.pair_total, c->stats);
    }

    ForceParams p;
    p.sorted = c->sorted;
    p.cell_start = c->cell_start;
    p.perm = c->perm;
    p.items = c->items;
    p.stats = c->stats;
    p.ax = a.ax; p.ay = a.ay; p.az = a.az;
    p.vx = a.kick ? c->vx : nullptr;
    p.vy = a.kick ? c->vy : nullptr;
    p.vz = a.kick ? c->vz : nullptr;
    p.nbr = a.nbr;
    p.pair_total = a.pair_total;
    p.rm2 = (double)a.r_max * (double)a.r_max;
    p.box_l = c->box_l;
    p.eps = a.eps;
    const float cut = (float)(p.rm2 + (double)a.eps);
    uint32_t cut_bits;
    memcpy(&cut_bits, &cut, 4);
    p.lo_bits = cut_bits - kBandHalf;
    memcpy(&p.cut_lo, &p.lo_bits, 4);
    p.dt = a.dt;
    recentre_negate(a.poly, (double)a.eps, p.nq);
    p.nc = c->nc;
    p.nz = c->nz;
    p.cz0 = c->cz0;

    // below ~1 M particles the second launch costs more than the occupancy gains (configs[0])
    // (HACCSR_SPARSE_KERNEL=0: never, =2: always -- for measurements and tests)
    const char *env = getenv("HACCSR_SPARSE_KERNEL");
    const bool sparse_kernel =
        env && env[0] == '0' ? false : env && env[0] == '2' ? true : n >= (int64_t(1) << 20);
    p.split_sparse = sparse_kernel ? 1 : 0;
    const bool count = a.nbr || a.pair_total;
    const int grid = c->n_sms * kBlocksPerSm, block = kWarpsPerBlock * 32;
    const int grid_s = c->n_sms * kSparseBlocksPerSm, block_s = kSparseWarps * 32;
#define HACCSR_FORCE(M, C)                                               \
    do {                                                                 \
        k_force<M, C><<<grid, block, 0, st>>>(p);                        \
        if (sparse_kernel) k_force_sparse<M, C><<<grid_s, block_s, 0, st>>>(p); \
    } while (0)
    if (c->unit_mass) {
        if (count) HACCSR_FORCE(false, true); else HACCSR_FORCE(false, false);
    } else {
        if (count) HACCSR_FORCE(true, true); else HACCSR_FORCE(true, false);
    }
#undef HACCSR_FORCE
    return cudaGetLastError();
}

}  // namespace haccsr
