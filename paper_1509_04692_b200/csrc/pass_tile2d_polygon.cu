// Colour-pass translation unit: the 2-D tile kernels for one particle kind (polygon); the body is pass_tile2d.inc.
#include "pass_tile2d.inc"

bool hpmc_launch_tile2d_polygon(hpmc_ctx* c, int ci, int shape) { return launch_shape<kKindPolygon, 0>(c, ci, shape); }
