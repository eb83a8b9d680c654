// Colour-pass translation unit: the 2-D tile kernels (one launch per colour, and the dataflow launch) for ONE particle kind,
// in the three tile shapes.  See sweep_tile2d.cuh.
#include "ctx.hpp"
#include "sweep_tile2d.cuh"

namespace {

template <int KIND, int NV, int WARPS, int R, int MINB>
bool launch_tile2d(hpmc_ctx* c, int ci)
{
    using TL = Tile2D<WARPS, R>;
    const GridParams& g = c->g;
    const int nax = g.n[0] / 2, nay = g.n[1] / 2;
    const int tiles = ((nax + kTileW - 1) / kTileW) * ((nay + TL::TH - 1) / TL::TH);
    if (c->flow_now) {   // all four colours in one persistent dataflow launch (issued for colour index 0 only)
        auto kern = k_sweep_tile2d_flow<KIND, NV, WARPS, R, MINB>;
        static bool attr_set = false;   // per template instance
        if (!attr_set) {
            if (!cuda_ok(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TL::bytes), "flow/attr")) return false;
            attr_set = true;
        }
        const int slots = c->num_sms * MINB;
        kern<<<tiles < slots ? tiles : slots, TL::NT, TL::bytes, c->stream>>>(g, c->mv, c->sf, c->sd, c->ctrl, c->opt_tile_cap,
                                                                                        c->pos[c->cur], c->tag[c->cur], c->cell_start, c->k0,
                                                                                        c->k1, c->trace, c->flow_done);
        return true;
    }
    auto kern = k_sweep_tile2d<KIND, NV, WARPS, R, MINB>;
    static bool attr_set = false;   // per template instance
    if (!attr_set) {
        if (!cuda_ok(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TL::bytes), "tile/attr")) return false;
        attr_set = true;
    }
    kern<<<tiles, TL::NT, TL::bytes, c->stream>>>(g, c->mv, c->sf, c->sd, c->ctrl, ci, c->opt_tile_cap, c->pos[c->cur], c->tag[c->cur],
                                                  c->cell_start, c->k0, c->k1, c->trace);
    return true;
}


template <int KIND, int NV>
bool launch_shape(hpmc_ctx* c, int ci, int shape)
{
    switch (shape) {
        case 1: return launch_tile2d<KIND, NV, 8, 2, 2>(c, ci);    // two rows of cells per warp (the R > 1 code path)
        case 2: return launch_tile2d<KIND, NV, 4, 1, 8>(c, ci);    // 64 registers, 8 CTAs per SM: large grids
        default: return launch_tile2d<KIND, NV, 2, 1, 8>(c, ci);   // small tiles: grids below one wave
    }
}

}  // namespace

bool hpmc_launch_tile2d_disk(hpmc_ctx* c, int ci, int shape) { return launch_shape<kKindDisk, 0>(c, ci, shape); }
