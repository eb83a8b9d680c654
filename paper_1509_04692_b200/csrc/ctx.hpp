// Host-side context of libhpmc.so and the launchers of the colour-pass kernels, shared by the translation units of the
// library: hpmc_api.cu and pass_*.cu are compiled in parallel and linked (no relocatable device code is needed, every
// kernel is self-contained).
#pragma once
#include <string>
#include <vector>

#include "../../include/hpmc.h"
#include "common.cuh"
#include "overlap.cuh"

using namespace hpmc;

struct hpmc_ctx {
    GridParams g{};
    MoveParams mv{};
    ShapeF sf{};
    ShapeD sd{};
    double d_max = 0.0;
    double w[3] = {1, 1, 1};
    uint64_t seed = 0;
    uint32_t k0 = 0, k1 = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    bool cuda_failed = false;
    int64_t launches = 0;
    uint64_t t_host = 0;  // mirror of the device sweep counter
    Control h_ctrl{};     // host landing buffer for the control block

    // caller-owned
    float4* d_pos_bound = nullptr;
    float4* d_quat_bound = nullptr;
    char* d_ws = nullptr;
    size_t ws_bytes = 0;
    bool state_in_bound = false;  // true: next build reads the bound arrays (tag order)
    bool have_sorted = false;

    // carved from the workspace
    float4* pos[2] = {nullptr, nullptr};
    float4* quat[2] = {nullptr, nullptr};
    int* tag[2] = {nullptr, nullptr};
    int cur = 0;
    int2* key_rank = nullptr;
    int* cell_start = nullptr;  // C+1 (+ padding)
    int* counts = nullptr;      // per-cell histogram, all zero between builds
    int* arrived = nullptr;     // per-cell arrival counter of k_scatter_sort, all zero between builds
    int* tile_sums = nullptr;   // per-tile totals of the scan
    unsigned int* flow_done = nullptr;   // per (colour, tile) stamps of the dataflow pass
    int num_sms = 0;
    int device = 0;                      // CUDA device of the context (the one current at hpmc_create); every entry point switches to it
    uint32_t attr_done = 0;              // cudaFuncSetAttribute(MaxDynamicSharedMemorySize) done for this context: bit per tile shape / flow
    bool after_colour = false;           // the last launch on the stream was a colour pass of the current cell list (PDL: its successor may
                                         // read the cell list before waiting)
    bool flow_now = false;               // this sweep's colour passes go out as one dataflow launch
    Control* ctrl = nullptr;
    int n_cap = 0;                                  // particles the workspace holds (N of hpmc_create); g.N <= n_cap varies with a distributed state
    bool cell_valid = false;                        // cell_start describes the arrays of `cur` (false after a route / append / load)
    bool dist = false;                              // distributed state: tags are global ids, the bound arrays are not used
    unsigned char* d_inactive = nullptr;            // workspace slot of the inactive-region mask (g.inactive points here while any layer is flagged)
    std::vector<unsigned char> inactive_h;          // host copy (survives a re-bind)

    uint2* trace = nullptr;
    int64_t trace_words = 0;

    // compute partition (hpmc_set_partition): this context runs the colour-pass tiles of tile rows [ty0, ty1) only
    int part_rank = 0, part_n = 1;

    // tuning / test knobs (hpmc_set_option)
    int opt_path = 0;                 // 0 auto, 1 per-thread global path, 2 tile path (2-D only), 3 warp per cell, 4 cluster (small 2-D), 5 speculative warp per cell (2-D)
    int cluster_ctas = -1;            // CTAs per cluster of the whole-sweep pass: -1 = not probed yet, 0 = unavailable on this device
    int opt_tile_cap = 1 << 30;       // staging capacity limit of the tile kernel (tests force the overflow path)
    int opt_tile_shape = 0;           // 0 = by grid size, 1..3 = fixed (see pick_tile_shape)
    int opt_flow = -1;                // 2-D tile pass as one dataflow launch per sweep: -1 = when it pays (auto), 0 = never, 1 = always
    int opt_small_build = 1;          // 1: systems with few cells build their cell list in one CTA (k_build_small)
    int opt_graph = 1;                // 1: hpmc_sweep(n >= 3) replays a captured two-sweep CUDA graph
    int opt_pdl = 1;                  // 1: the kernels of a sweep are launched with programmatic stream serialization (common.cuh)

    // CUDA graph of two consecutive sweeps (the ping-pong buffers return to where they started), one per parity of `cur`
    cudaGraphExec_t graph_exec[2] = {nullptr, nullptr};
    int64_t graph_launches = 0;       // kernels inside one replay

    // optional per-kernel device timing (hpmc_set_profile): event pairs around the cell-list build (class 0)
    // and around every colour-pass launch (class 1)
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<int> ev_class;     // one per recorded pair
    size_t ev_used = 0;            // events handed out (2 per pair)
    double prof_ms[2] = {0.0, 0.0};
    int64_t prof_n[2] = {0, 0};
};

// Makes the context's device current for the duration of an entry point (the caller's current device may be another one).
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const hpmc_ctx* c)
    {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) cudaSetDevice(c->device);
        else prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline bool cuda_ok(hpmc_ctx* c, cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return true;
    c->cuda_failed = true;
    c->err = std::string("CUDA error in ") + what + ": " + cudaGetErrorString(e);
    return false;
}


// Kernel launch on the context's stream, as a programmatic dependent launch when the option is on (every kernel launched
// through here starts with pdl_launch_dependents(); pdl_wait();).
template <typename... KArgs, typename... Args>
inline cudaError_t hpmc_launch(hpmc_ctx* c, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c->opt_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

constexpr int kTileWHost = 32;   // active cells per tile row (= kTileW of sweep_tile2d.cuh)
// 3-D polyhedron systems with more active cells per colour than two waves of the 168-register warp-per-cell kernel (12 warps per
// SM) are bound by instruction issue and run k_sweep_warpcell_occ (sweep_warpcell.cuh)
constexpr int kOccMinActive3d = 2 * 148 * 12;

// Colour-pass launchers; each returns false after recording a CUDA error in the context.
//   kind: kKindDisk / kKindPolygon / kKindPolyhedron; nv: unrolled vertex count (5 pentagons; 8, 20, 24 polyhedra) or 0 = runtime count
bool hpmc_launch_tile2d(hpmc_ctx* c, int ci, int kind, int nv, int shape);       // pass_tile2d_*.cu (2-D, not polyhedra)
bool hpmc_launch_warpcell(hpmc_ctx* c, int ci, int kind, int nv, int nactive);   // pass_warpcell_*.cu
bool hpmc_launch_spec2d(hpmc_ctx* c, int ci, int kind, int nv, int nactive);     // pass_spec2d.cu
bool hpmc_launch_colour(hpmc_ctx* c, int ci, int kind, int nv, int nactive);     // pass_colour.cu
// whole sweeps of a small 2-D system in one cluster launch (pass_cluster2d.cu): sweeps enqueued, 0 = cluster size unavailable, -1 = error
int hpmc_launch_cluster2d(hpmc_ctx* c, int64_t n_sweeps, int ncta, int kind, int nv);
