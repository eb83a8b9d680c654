// Colour-pass translation unit: the 2-D tile kernels for one particle kind (pentagon); the body is pass_tile2d.inc.
#include "pass_tile2d.inc"

bool hpmc_launch_tile2d_pentagon(hpmc_ctx* c, int ci, int shape) { return launch_shape<kKindPolygon, 5>(c, ci, shape); }
