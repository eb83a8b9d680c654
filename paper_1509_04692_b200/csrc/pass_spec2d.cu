// Colour-pass translation unit: the speculative warp-per-cell kernels for small 2-D systems.  See sweep_spec2d.cuh.
#include "ctx.hpp"
#include "sweep_spec2d.cuh"

namespace {

template <int KIND, int NV>
bool launch_spec(hpmc_ctx* c, int ci, int nactive)
{
    hpmc_launch(c, k_sweep_spec2d<KIND, NV>, (nactive + kSpecWarps - 1) / kSpecWarps, 32 * kSpecWarps, 0,
        c->g, c->mv, c->sf, c->sd, c->ctrl, ci, c->opt_tile_cap, c->pos[c->cur], c->tag[c->cur], c->cell_start, c->k0, c->k1, c->trace,
        c->after_colour ? 1 : 0);
    return true;
}

}  // namespace

bool hpmc_launch_spec2d(hpmc_ctx* c, int ci, int kind, int nv, int nactive)
{
    if (kind == kKindDisk) return launch_spec<kKindDisk, 0>(c, ci, nactive);
    return (nv == 5) ? launch_spec<kKindPolygon, 5>(c, ci, nactive) : launch_spec<kKindPolygon, 0>(c, ci, nactive);
}
