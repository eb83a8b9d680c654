// hpmc_count_overlaps_noalloc (include/hpmc.h): the overlap-count validator (S:8(a) row a12) for callers that cannot
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The existing validator
// (hpmc_count_overlaps) reads the cell list that the library keeps in the caller's WORKSPACE (hpmc_workspace_bytes /
// hpmc_bind).  This variant needs neither a workspace nor a bind: its cell list lives in ONE file-scope device array of fixed
// size, g_noalloc_scratch below, which every GPU that loads libhpmc.so holds until the process exits (1.25 MB).
//
//   - Limits: at most kNoAllocMaxN particles and kNoAllocMaxCells cells; larger requests are refused with HPMC_E_ARG.
//   - The entry point calls no cudaMalloc / cudaFree and no allocating library routine: six small kernel launches on the
//     context's stream, nothing else (plus, the first time on a device, one cudaGetSymbolAddress).
//   - Every call on a device shares the array and finds the previous call's contents in it: k_na_clear zeroes what must start
//     at zero (the per-cell counts, the pair counter, the bad-coordinate flag); everything else is fully rewritten for the
//     first n entries before it is read.
//   - Calls whose kernels overlap on the GPU (two contexts with different streams, two host threads) RACE on the array: run
//     them on one stream or order them with events.
//
// In host code the NAME g_noalloc_scratch is a host-side stand-in, not a device address.  The address a kernel can use is
// fetched once per device, with that device current, by cudaGetSymbolAddress (noalloc_scratch_ptr) and passed as a kernel
// argument.
#include <string>

#include "ctx.hpp"
#include "sweep.cuh"

namespace {

constexpr int kNoAllocMaxN = 65536;        // particles per call
constexpr int kNoAllocMaxCells = 131072;   // cells of the context's grid
constexpr int kNaThreads = 256;
constexpr int kNaScanThreads = 1024;

// layout of the scratch array (all offsets multiples of 256 bytes)
struct NaLayout {
    static constexpr size_t head = 0;                                                        // NaHead
    static constexpr size_t counts = 256;                                                    // int[kNoAllocMaxCells + 1] -> cell_start
    static constexpr size_t key_rank = counts + ((sizeof(int) * (kNoAllocMaxCells + 1) + 255) / 256) * 256;   // int2[kNoAllocMaxN]
    static constexpr size_t order = key_rank + sizeof(int2) * kNoAllocMaxN;                  // int[kNoAllocMaxN]
    static constexpr size_t total = order + sizeof(int) * kNoAllocMaxN;
};

struct NaHead {
    unsigned long long pairs;   // overlapping pairs found
    unsigned int bad;           // particles with coordinates outside [-L/2, L/2) or not finite
};

static __device__ __align__(256) unsigned char g_noalloc_scratch[NaLayout::total];

// device address of the array, per device (fetched at the first call on that device)
constexpr int kNaMaxDevices = 64;
void* g_na_ptr[kNaMaxDevices] = {nullptr};

cudaError_t noalloc_scratch_ptr(int device, void** out)
{
    if (device < 0 || device >= kNaMaxDevices) return cudaErrorInvalidDevice;
    if (!g_na_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);   // the current device is `device` (DeviceGuard)
        if (e != cudaSuccess) return e;
        g_na_ptr[device] = p;
    }
    *out = g_na_ptr[device];
    return cudaSuccess;
}

__global__ void __launch_bounds__(kNaThreads) k_na_clear(unsigned char* __restrict__ scratch, int C)
{
    int* counts = reinterpret_cast<int*>(scratch + NaLayout::counts);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i <= C) counts[i] = 0;
    if (i == 0) {
        NaHead* h = reinterpret_cast<NaHead*>(scratch + NaLayout::head);
        h->pairs = 0ull;
        h->bad = 0u;
    }
}

// cell of every particle on the UNSHIFTED grid (as the existing validator: cell list with zero shift) and its arrival rank
__global__ void __launch_bounds__(kNaThreads)
k_na_hist(const __grid_constant__ GridParams g, int n, const float4* __restrict__ pos, unsigned char* __restrict__ scratch)
{
    int* counts = reinterpret_cast<int*>(scratch + NaLayout::counts);
    int2* key_rank = reinterpret_cast<int2*>(scratch + NaLayout::key_rank);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 x = pos[i];
    const float shift[3] = {0.0f, 0.0f, 0.0f};
    bool bad;
    const int cell = cell_of_checked(g, shift, x.x, x.y, x.z, bad);   // clamped into the grid when the precondition is broken
    if (bad) atomicAdd(&reinterpret_cast<NaHead*>(scratch + NaLayout::head)->bad, 1u);
    key_rank[i] = make_int2(cell, atomicAdd(&counts[cell], 1));
}

// exclusive scan of counts[0..C] in place, one CTA: counts becomes cell_start (cell_start[C] = n)
__global__ void __launch_bounds__(kNaScanThreads) k_na_scan(unsigned char* __restrict__ scratch, int C)
{
    __shared__ int s_warp[kNaScanThreads / 32];
    int* counts = reinterpret_cast<int*>(scratch + NaLayout::counts);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = (C + 1 + kNaScanThreads - 1) / kNaScanThreads;
    const int lo = min(tid * per, C + 1), hi = min(lo + per, C + 1);
    int sum = 0;
    for (int i = lo; i < hi; ++i) sum += counts[i];
    int inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    int run = inc - sum;
    for (int w = 0; w < warp; ++w) run += s_warp[w];
    for (int i = lo; i < hi; ++i) {
        const int v = counts[i];
        counts[i] = run;
        run += v;
    }
}

__global__ void __launch_bounds__(kNaThreads) k_na_scatter(int n, unsigned char* __restrict__ scratch)
{
    const int* cell_start = reinterpret_cast<const int*>(scratch + NaLayout::counts);
    const int2* key_rank = reinterpret_cast<const int2*>(scratch + NaLayout::key_rank);
    int* order = reinterpret_cast<int*>(scratch + NaLayout::order);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) order[cell_start[key_rank[i].x] + key_rank[i].y] = i;
}

// a12 on the scratch cell list: pairs (i < j) in 3^d neighbourhoods whose interiors intersect (strict, fp64).  The same pair
// test as k_count_overlaps (sweep.cuh), reading the caller's tag-order arrays through `order`.
template <int KIND>
__global__ void __launch_bounds__(128)
k_na_count(const __grid_constant__ GridParams g, const __grid_constant__ ShapeD S, int n, const float4* __restrict__ pos,
           const float4* __restrict__ quat, unsigned char* __restrict__ scratch)
{
    const int* cell_start = reinterpret_cast<const int*>(scratch + NaLayout::counts);
    const int2* key_rank = reinterpret_cast<const int2*>(scratch + NaLayout::key_rank);
    const int* order = reinterpret_cast<const int*>(scratch + NaLayout::order);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int found = 0;
    if (i < n) {
        const float4 xp = pos[i];
        const int cell = key_rank[i].x;
        const int cx = cell % g.n[0], cy = (cell / g.n[0]) % g.n[1], cz = cell / (g.n[0] * g.n[1]);
        double MA[9];
        double cA = 1.0, sA = 0.0;
        if (KIND != kKindDisk) {
            const float4 qp = quat[i];
            const double nq = sqrt((double)qp.x * qp.x + (double)qp.y * qp.y + (double)qp.z * qp.z + (double)qp.w * qp.w);
            const double w = qp.x / nq, x = qp.y / nq, y = qp.z / nq, z = qp.w / nq;
            if (KIND == kKindPolygon) { cA = w * w - z * z; sA = 2.0 * w * z; }
            if (KIND == kKindPolyhedron) quat_to_matrix<double>(w, x, y, z, MA);
        }
        const int zlo = (g.dim == 3) ? -1 : 0, zhi = (g.dim == 3) ? 1 : 0;
        for (int dz = zlo; dz <= zhi; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    const int nx = (cx + dx + g.n[0]) % g.n[0], ny = (cy + dy + g.n[1]) % g.n[1], nz = (cz + dz + g.n[2]) % g.n[2];
                    const int c2 = nx + g.n[0] * (ny + g.n[1] * nz);
                    for (int s = cell_start[c2]; s < cell_start[c2 + 1]; ++s) {
                        const int j = order[s];
                        if (j <= i) continue;
                        const float4 xq = pos[j];
                        double r[3] = {(double)xq.x - (double)xp.x, (double)xq.y - (double)xp.y, (double)xq.z - (double)xp.z};
                        for (int k = 0; k < g.dim; ++k) {
                            if (r[k] > 0.5 * g.Ld[k]) r[k] -= g.Ld[k];
                            else if (r[k] < -0.5 * g.Ld[k]) r[k] += g.Ld[k];
                        }
                        if (g.dim == 2) r[2] = 0.0;
                        const double d2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
                        if (d2 >= S.dmax2) continue;
                        bool ov = true;
                        if (KIND != kKindDisk) {
                            const float4 qq = quat[j];
                            const double nq = sqrt((double)qq.x * qq.x + (double)qq.y * qq.y + (double)qq.z * qq.z + (double)qq.w * qq.w);
                            const double w = qq.x / nq, x = qq.y / nq, y = qq.z / nq, z = qq.w / nq;
                            if (KIND == kKindPolygon) {
                                ov = polygon_overlap<double, 0>(S, r[0], r[1], cA, sA, w * w - z * z, 2.0 * w * z, 0.0);
                            } else {
                                double MB[9];
                                quat_to_matrix<double>(w, x, y, z, MB);
                                int unused[3];
                                ov = polyhedron_classify<double>(S, MA, MB, V3<double>{r[0], r[1], r[2]}, 0.0, 0.0, unused) != kGjkSeparated;
                            }
                        }
                        if (ov) ++found;
                    }
                }
    }
    found = __reduce_add_sync(0xffffffffu, found);
    if ((threadIdx.x & 31) == 0 && found)
        atomicAdd(&reinterpret_cast<NaHead*>(scratch + NaLayout::head)->pairs, (unsigned long long)found);
}

// the caller's output: the pair count, or -1 when a coordinate broke the in-box precondition
__global__ void k_na_result(const unsigned char* __restrict__ scratch, long long* __restrict__ out)
{
    const NaHead* h = reinterpret_cast<const NaHead*>(scratch + NaLayout::head);
    *out = h->bad ? -1ll : (long long)h->pairs;
}

int na_fail(hpmc_ctx* c, int code, const std::string& msg)
{
    c->err = msg;
    return code;
}

}  // namespace

extern "C" {

int hpmc_count_overlaps_noalloc(hpmc_ctx* c, const float* d_pos4, const float* d_quat4, int64_t n, int64_t* d_count_out)
{
    if (!c) return HPMC_E_ARG;
    DeviceGuard dev_guard(c);
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (n < 0 || n > kNoAllocMaxN)
        return na_fail(c, HPMC_E_ARG, "hpmc_count_overlaps_noalloc: n = " + std::to_string(n) + " exceeds the static scratch (at most " +
                                          std::to_string(kNoAllocMaxN) + " particles); use hpmc_bind + hpmc_count_overlaps");
    if (c->g.C > kNoAllocMaxCells)
        return na_fail(c, HPMC_E_ARG, "hpmc_count_overlaps_noalloc: the grid has " + std::to_string(c->g.C) + " cells, the static scratch holds " +
                                          std::to_string(kNoAllocMaxCells) + "; use hpmc_bind + hpmc_count_overlaps");
    if (!d_count_out || (n > 0 && !d_pos4) || (n > 0 && c->sd.kind != kKindDisk && !d_quat4))
        return na_fail(c, HPMC_E_ARG, "hpmc_count_overlaps_noalloc: NULL device pointer");
    if (((uintptr_t)d_pos4 & 15u) || ((uintptr_t)d_quat4 & 15u) || ((uintptr_t)d_count_out & 7u))
        return na_fail(c, HPMC_E_ARG, "hpmc_count_overlaps_noalloc: state arrays must be 16-byte aligned, the output 8-byte aligned");
    void* vp = nullptr;
    if (!cuda_ok(c, noalloc_scratch_ptr(c->device, &vp), "noalloc/cudaGetSymbolAddress")) return HPMC_E_CUDA;
    unsigned char* scratch = static_cast<unsigned char*>(vp);
    const GridParams& g = c->g;
    const float4* pos = reinterpret_cast<const float4*>(d_pos4);
    const float4* quat = reinterpret_cast<const float4*>(d_quat4);
    const int nn = (int)n;
    cudaStream_t st = c->stream;
    GridParams gn = g;        // the context's grid with this call's particle count
    gn.N = nn;
    gn.inactive = nullptr;
    k_na_clear<<<(g.C + 1 + kNaThreads - 1) / kNaThreads, kNaThreads, 0, st>>>(scratch, g.C);
    if (nn > 0) {
        const int nb = (nn + kNaThreads - 1) / kNaThreads;
        k_na_hist<<<nb, kNaThreads, 0, st>>>(gn, nn, pos, scratch);
        k_na_scan<<<1, kNaScanThreads, 0, st>>>(scratch, g.C);
        k_na_scatter<<<nb, kNaThreads, 0, st>>>(nn, scratch);
        const int nc = (nn + 127) / 128;
        if (c->sd.kind == kKindDisk) k_na_count<kKindDisk><<<nc, 128, 0, st>>>(gn, c->sd, nn, pos, quat, scratch);
        else if (c->sd.kind == kKindPolygon) k_na_count<kKindPolygon><<<nc, 128, 0, st>>>(gn, c->sd, nn, pos, quat, scratch);
        else k_na_count<kKindPolyhedron><<<nc, 128, 0, st>>>(gn, c->sd, nn, pos, quat, scratch);
        c->launches += 4;
    }
    k_na_result<<<1, 1, 0, st>>>(scratch, reinterpret_cast<long long*>(d_count_out));
    c->launches += 2;
    if (!cuda_ok(c, cudaGetLastError(), "hpmc_count_overlaps_noalloc")) return HPMC_E_CUDA;
    return HPMC_OK;
}

}  // extern "C"
