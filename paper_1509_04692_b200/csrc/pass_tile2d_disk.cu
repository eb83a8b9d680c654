// Colour-pass translation unit: the 2-D tile kernels for one particle kind (disk); the body is pass_tile2d.inc.
#include "pass_tile2d.inc"

bool hpmc_launch_tile2d_disk(hpmc_ctx* c, int ci, int shape) { return launch_shape<kKindDisk, 0>(c, ci, shape); }
