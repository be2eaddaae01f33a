// mesh.cuh -- position -> wrapped position -> cell coordinate, shared by the binning kernels.
// Internal to csrc/; nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ctx.h"

namespace haccsr {

struct MeshGeom {
    float box_l;
    float scale;      // nc / L (used only when exact)
    double dscale_nc; // (double) nc
    double dbox_l;    // (double) L
    int nc;
    int exact;
    // the z window of the mesh this context covers: nz cell layers starting at global layer
    // cz0 (periodic).  nz == nc, cz0 == 0: the whole box.  Otherwise an overloaded slab
    // (PAPER.md:112-122): layers 0 and nz-1 of the window hold passive particles only.
    int nz;
    int cz0;
};

// Wrap rule (reading S16): x - L*floor(x/L); a result that is not inside [0,L)
// after rounding becomes 0.  Non-finite input returns 0 and sets *bad.
// The out-of-box case is kept out of line: the streaming kernels then carry two compares and
// a predicated call per coordinate instead of the division and its convergence barriers.
static __device__ __noinline__ float wrap_pos_slow(float x, float box_l, int *bad)
{
    if (!isfinite(x)) {
        *bad = 1;
        return 0.f;
    }
    float w = x - box_l * floorf(x / box_l);
    if (!(w >= 0.f && w < box_l)) w = 0.f;
    return w;
}

__device__ __forceinline__ float wrap_pos(float x, float box_l, bool &bad)
{
    if (x >= 0.f && x < box_l) return x;
    int b = 0;
    const float w = wrap_pos_slow(x, box_l, &b);
    bad |= (b != 0);
    return w;
}

// Exact floor(x*nc/L) (reading S12).  When nc/L is a float32 number the round-down product
// cannot cross an integer upwards, so float2int_rd(fmul_rd) is the exact floor; otherwise the
// same double expression the definition uses.
static __device__ __noinline__ int cell_coord_double(float x, double nc, double box_l)
{
    return (int)floor((double)x * nc / box_l);
}

__device__ __forceinline__ int cell_coord(float x, const MeshGeom &g)
{
    const int c = g.exact ? __float2int_rd(__fmul_rd(x, g.scale))
                          : cell_coord_double(x, g.dscale_nc, g.dbox_l);
    return min(max(c, 0), g.nc - 1);
}


// Window layer of a wrapped z coordinate; a particle outside the window sets bad and is put
// in the last layer.
__device__ __forceinline__ int layer_coord(float z, const MeshGeom &g, bool &bad)
{
    int l = cell_coord(z, g) - g.cz0;
    l += (l < 0) ? g.nc : 0;
    if (l >= g.nz) {
        bad = true;
        l = g.nz - 1;
    }
    return l;
}

inline MeshGeom geom_of(const haccsr_ctx *c)
{
    MeshGeom g;
    g.box_l = c->box_l;
    g.scale = (float)((double)c->nc / (double)c->box_l);
    g.dscale_nc = (double)c->nc;
    g.dbox_l = (double)c->box_l;
    g.nc = c->nc;
    g.exact = c->scale_exact ? 1 : 0;
    g.nz = c->nz;
    g.cz0 = c->cz0;
    return g;
}

}  // namespace haccsr
