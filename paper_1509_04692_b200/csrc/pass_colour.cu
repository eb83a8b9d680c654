// Colour-pass translation unit: the per-thread global-memory pass (cross-check variant, `hpmc_set_option("path", 1)`), and
// the routing of the launchers declared in ctx.hpp to the translation units that hold each variant.
#include "ctx.hpp"
#include "sweep.cuh"

bool hpmc_launch_tile2d_disk(hpmc_ctx* c, int ci, int shape);
bool hpmc_launch_tile2d_pentagon(hpmc_ctx* c, int ci, int shape);
bool hpmc_launch_tile2d_polygon(hpmc_ctx* c, int ci, int shape);
bool hpmc_launch_warpcell_2d(hpmc_ctx* c, int ci, int kind, int nv, int nactive);
bool hpmc_launch_warpcell_3d(hpmc_ctx* c, int ci, int kind, int nv, int nactive);

bool hpmc_launch_tile2d(hpmc_ctx* c, int ci, int kind, int nv, int shape)
{
    if (kind == kKindDisk) return hpmc_launch_tile2d_disk(c, ci, shape);
    return (nv == 5) ? hpmc_launch_tile2d_pentagon(c, ci, shape) : hpmc_launch_tile2d_polygon(c, ci, shape);
}

bool hpmc_launch_warpcell(hpmc_ctx* c, int ci, int kind, int nv, int nactive)
{
    return (c->g.dim == 3) ? hpmc_launch_warpcell_3d(c, ci, kind, nv, nactive) : hpmc_launch_warpcell_2d(c, ci, kind, nv, nactive);
}

namespace {

template <int KIND, int NV>
bool launch_thread_per_cell(hpmc_ctx* c, int ci, int nactive)
{
    const int TB = 128;
    k_sweep_colour<KIND, NV><<<(nactive + TB - 1) / TB, TB, 0, c->stream>>>(c->g, c->mv, c->sf, c->sd, c->ctrl, ci, c->pos[c->cur],
                                                                           c->quat[c->cur], c->tag[c->cur], c->cell_start, c->k0, c->k1,
                                                                           c->trace);
    return true;
}

}  // namespace

bool hpmc_launch_colour(hpmc_ctx* c, int ci, int kind, int nv, int nactive)
{
    if (kind == kKindDisk) return launch_thread_per_cell<kKindDisk, 0>(c, ci, nactive);
    if (kind == kKindPolygon) return (nv == 5) ? launch_thread_per_cell<kKindPolygon, 5>(c, ci, nactive) : launch_thread_per_cell<kKindPolygon, 0>(c, ci, nactive);
    return launch_thread_per_cell<kKindPolyhedron, 0>(c, ci, nactive);
}
