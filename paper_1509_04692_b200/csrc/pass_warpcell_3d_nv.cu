// Colour-pass translation unit: the 3-D warp-per-cell kernels with 20 and 24 unrolled vertices.  See sweep_warpcell.cuh.
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

// Unrolled support functions for the paper's two benchmark polyhedra: 20 vertices (dodecahedra) and 24 (truncated
// octahedra, Fig. 4 and Table 1).  A translation unit of its own so that it compiles beside pass_warpcell_3d.cu.
bool hpmc_launch_warpcell_3d_nv(hpmc_ctx* c, int ci, int nv, int nactive)
{
    return (nv == 20) ? launch_warpcell<kKindPolyhedron, 20, 3>(c, ci, nactive) : launch_warpcell<kKindPolyhedron, 24, 3>(c, ci, nactive);
}
