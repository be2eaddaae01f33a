// levels.cu -- multi-level (density-adaptive) time stepping, PAPER.md:214-216 (section 2.5) and
// 315-325 (section 3.1, Eq. 11): "particles in higher density regions will require finer
// short-range time steps.  A local density estimate can be trivially extracted from the same"
// structure "constructed for evaluating the short-range interparticle forces" -- here the
// occupancy of the particle's chaining-mesh cell.  Readings S21-S23 of DESIGN.md section 3.
#include "ctx.h"
#include "mesh.cuh"

namespace haccsr {

// cell (window id) of a particle position, as the sort computes it
__device__ __forceinline__ int64_t cell_of(float x, float y, float z, const MeshGeom &g, bool &bad)
{
    const float wx = wrap_pos(x, g.box_l, bad), wy = wrap_pos(y, g.box_l, bad),
                wz = wrap_pos(z, g.box_l, bad);
    return cell_coord(wx, g) + (int64_t)g.nc * (cell_coord(wy, g) + (int64_t)g.nc * layer_coord(wz, g, bad));
}

// Eq. 11: l = floor((rho/rho0) / d) + 1 kicks, rho/rho0 = n_c * n_cells / n, clipped to
// [l_min, l_max]; level = floor(log2 l) (power-of-two kick counts keep the levels
// synchronised).  The ratio is formed in double, as the definition.
__global__ void __launch_bounds__(256) k_assign_levels(int64_t n, const float *__restrict__ x,
                                                       const float *__restrict__ y,
                                                       const float *__restrict__ z, MeshGeom g,
                                                       const uint32_t *__restrict__ cell_start,
                                                       double cells, double n_total, double d,
                                                       int l_min, int l_max,
                                                       uint8_t *__restrict__ level)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int64_t c = cell_of(x[i], y[i], z[i], g, bad);
        // same expression, same order as the definition: (n_c * cells) / n, then / d
        const double ratio = (double)(cell_start[c + 1] - cell_start[c]) * cells / n_total;
        double lf = floor(ratio / d) + 1.0;
        lf = fmin(fmax(lf, (double)l_min), (double)l_max);
        const int l = (int)lf;
        level[i] = (uint8_t)(31 - __clz(l));
    }
}

__global__ void k_accumulate_evals(unsigned long long *evals, const DeviceStats *stats)
{
    *evals += stats->n_eval;
}

static inline int stream_grid(const haccsr_ctx *c, int64_t n)
{
    const int64_t want = (n + 255) / 256, cap = (int64_t)c->n_sms * 16;
    return (int)(want < cap ? (want > 0 ? want : 1) : cap);
}

cudaError_t launch_assign_levels(haccsr_ctx *c, int64_t n, const float *x, const float *y,
                                 const float *z, float d, int l_min, int l_max, uint8_t *level)
{
    if (n > 0) {
        // the density is relative to the mean of the WHOLE box: nc^3 cells
        const double cells = (double)c->nc * c->nc * c->nc;
        k_assign_levels<<<stream_grid(c, n), 256, 0, c->stream>>>(
            n, x, y, z, geom_of(c), c->cell_start, cells, (double)n, (double)d, l_min, l_max,
            level);
    }
    return cudaGetLastError();
}

cudaError_t launch_accumulate_evals(haccsr_ctx *c, unsigned long long *evals)
{
    k_accumulate_evals<<<1, 1, 0, c->stream>>>(evals, c->stats);
    return cudaGetLastError();
}

}  // namespace haccsr
