// Colour-pass translation unit: the warp-per-cell kernels of one dimension.  See sweep_warpcell.cuh.
#include "ctx.hpp"
#include "sweep_warpcell.cuh"

namespace {


template <int KIND, int NV, int DIM>
bool launch_warpcell(hpmc_ctx* c, int ci, int nactive)
{
    if constexpr (KIND == kKindPolyhedron) {
        if (nactive > kOccMinActive3d) {
            hpmc_launch(c, k_sweep_warpcell_occ<KIND, NV, DIM>, (nactive + kW3Warps - 1) / kW3Warps, 32 * kW3Warps, 0,
                c->g, c->mv, c->sf, c->sd, c->ctrl, ci, c->opt_tile_cap, c->pos[c->cur], c->quat[c->cur], c->tag[c->cur], c->cell_start, c->k0,
                c->k1, c->trace, c->after_colour ? 1 : 0);
            return true;
        }
    }
    hpmc_launch(c, k_sweep_warpcell<KIND, NV, DIM>, (nactive + kW3Warps - 1) / kW3Warps, 32 * kW3Warps, 0,
        c->g, c->mv, c->sf, c->sd, c->ctrl, ci, c->opt_tile_cap, c->pos[c->cur], c->quat[c->cur], c->tag[c->cur], c->cell_start, c->k0,
        c->k1, c->trace, c->after_colour ? 1 : 0);
    return true;
}

}  // namespace

bool hpmc_launch_warpcell_3d_nv(hpmc_ctx* c, int ci, int nv, int nactive);

bool hpmc_launch_warpcell_3d(hpmc_ctx* c, int ci, int kind, int nv, int nactive)
{
    if (kind == kKindDisk) return launch_warpcell<kKindDisk, 0, 3>(c, ci, nactive);
    // polyhedra: 8 vertices (cubes, config 3), 20 and 24 (pass_warpcell_3d_nv.cu) have unrolled support functions
    if (nv == 20 || nv == 24) return hpmc_launch_warpcell_3d_nv(c, ci, nv, nactive);
    return (nv == 8) ? launch_warpcell<kKindPolyhedron, 8, 3>(c, ci, nactive) : launch_warpcell<kKindPolyhedron, 0, 3>(c, ci, nactive);
}
