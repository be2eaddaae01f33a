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
};

// Wrap rule (reading S16): x - L*floor(x/L); a result that is not inside [0,L)
// after rounding becomes 0.  Non-finite input returns 0 and sets *bad.
__device__ __forceinline__ float wrap_pos(float x, float box_l, bool &bad)
{
    if (x >= 0.f && x < box_l) return x;
    if (!isfinite(x)) {
        bad = true;
        return 0.f;
    }
    float w = x - box_l * floorf(x / box_l);
    if (!(w >= 0.f && w < box_l)) w = 0.f;
    return w;
}

// Exact floor(x*nc/L) (reading S12).  When nc/L is a float32 number the round-down product
// cannot cross an integer upwards, so float2int_rd(fmul_rd) is the exact floor; otherwise the
// same double expression the definition uses.
__device__ __forceinline__ int cell_coord(float x, const MeshGeom &g)
{
    int c;
    if (g.exact)
        c = __float2int_rd(__fmul_rd(x, g.scale));
    else
        c = (int)floor((double)x * g.dscale_nc / g.dbox_l);
    return min(max(c, 0), g.nc - 1);
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
    return g;
}

}  // namespace haccsr
