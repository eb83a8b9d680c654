// Colour-pass translation unit: whole sweeps of a small 2-D system in one thread-block cluster.  See sweep_cluster2d.cuh.
#include "ctx.hpp"
#include "sweep_cluster2d.cuh"

namespace {

template <int KIND, int NV, int G>
int launch_cluster(hpmc_ctx* c, int64_t n_sweeps, int ncta)
{
    auto kern = k_sweep_cluster2d<KIND, NV, G>;
    const size_t smem = cluster_smem_bytes<G>(c->g.C);
    if (!cuda_ok(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "cluster/smem")) return -1;
    if (ncta > 8 && !cuda_ok(c, cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1), "cluster/nonportable")) return -1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)ncta, 1, 1);
    cfg.blockDim = dim3(kClThreads, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)ncta;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg) != cudaSuccess || nclusters < 1) {
        cudaGetLastError();   // not an error of the context: the caller tries a smaller cluster or another pass
        return 0;
    }
    const int n = (int)n_sweeps;   // the caller keeps it below 2^20
    if (!cuda_ok(c, cudaLaunchKernelEx(&cfg, kern, c->g, c->mv, c->sf, c->sd, c->ctrl, n, c->cur, c->pos[0], c->pos[1], c->tag[0], c->tag[1],
                                       c->counts, c->cell_start, c->k0, c->k1, c->trace),
                 "cluster/launch"))
        return -1;
    return n;
}

}  // namespace

// Runs up to n_sweeps sweeps in one launch of one cluster of `ncta` CTAs.  Returns the number of sweeps enqueued, 0 if a cluster
// of that size cannot be scheduled on this device, -1 after recording a CUDA error.
int hpmc_launch_cluster2d(hpmc_ctx* c, int64_t n_sweeps, int ncta, int kind, int nv)
{
    if (kind == kKindDisk) return launch_cluster<kKindDisk, 0, 8>(c, n_sweeps, ncta);
    return (nv == 5) ? launch_cluster<kKindPolygon, 5, 8>(c, n_sweeps, ncta) : launch_cluster<kKindPolygon, 0, 8>(c, n_sweeps, ncta);
}
