// Cell-list builder (S:8(a) rows a1-a3): sweep header, cell id, histogram, exclusive scan, scatter into
// the cell-sorted SoA, canonical in-cell order (ascending tag, R8), plus the un-sort for get_state (a13).
// "A bucket sort efficiently assigns particles to cells, and a massively parallel bucket sort on the GPU
// is trivial to implement with atomic operations".
#pragma once
#include "common.cuh"

namespace hpmc {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;

// mode 0: header of the device sweep counter t, then t++ and sweeps++   (a real sweep)
// mode 1: header of t_override, nothing advanced                         (debug cell list)
// mode 2: zero shift, nothing advanced                                   (validator)
__global__ void k_prepare(const __grid_constant__ GridParams g, Control* __restrict__ ctrl, int* __restrict__ counts,
                          uint32_t k0, uint32_t k1, int mode, unsigned long long t_override)
{
    const int stride = gridDim.x * blockDim.x;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= g.C; i += stride) counts[i] = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const unsigned long long t = (mode == 0) ? ctrl->t : t_override;
        SweepHeader h;
        make_header(g, k0, k1, t, mode == 2, h);
        h.pad = 0;
        ctrl->hdr = h;
        if (mode == 0) {
            ctrl->t = t + 1ull;
            ctrl->sweeps += 1ull;
        }
    }
}

// a2 + first half of a3: cell id and slot inside the cell (arrival order; made canonical by k_cell_sort)
__global__ void k_hist(const __grid_constant__ GridParams g, const Control* __restrict__ ctrl,
                       const float4* __restrict__ pos, int* __restrict__ counts, int2* __restrict__ key_rank)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.N) return;
    const float shift[3] = {ctrl->hdr.shift[0], ctrl->hdr.shift[1], ctrl->hdr.shift[2]};
    const float4 x = pos[p];
    int cx, cy, cz;
    const int c = cell_of(g, shift, x.x, x.y, x.z, cx, cy, cz);
    const int rank = atomicAdd(&counts[c], 1);
    key_rank[p] = make_int2(c, rank);
}

__device__ __forceinline__ int warp_inclusive_scan(int v)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) >= o) v += n;
    }
    return v;
}

// exclusive scan of one value per thread across a block of kScanThreads; returns the block total in `total`
__device__ __forceinline__ int block_exclusive_scan(int v, int& total)
{
    __shared__ int warp_sums[kScanThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int inc = warp_inclusive_scan(v);
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    int offset = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        const int s = warp_sums[w];
        if (w < wid) offset += s;
        tot += s;
    }
    total = tot;
    __syncthreads();
    return offset + inc - v;
}

// scan pass 1: per-tile totals
__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const int* __restrict__ counts, int n, int* __restrict__ tile_sums)
{
    const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    int s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i)
        if (base + i < n) s += counts[base + i];
    int total;
    block_exclusive_scan(s, total);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

// scan pass 2: exclusive scan of the tile totals by ONE block
__global__ void __launch_bounds__(kScanThreads) k_scan_spine(int* __restrict__ tile_sums, int ntiles)
{
    __shared__ int carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < ntiles; base += kScanThreads) {
        const int i = base + threadIdx.x;
        const int v = (i < ntiles) ? tile_sums[i] : 0;
        int total;
        const int ex = block_exclusive_scan(v, total);
        const int carry = carry_s;
        if (i < ntiles) tile_sums[i] = carry + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + total;
        __syncthreads();
    }
}

// scan pass 3: in-place exclusive scan of each tile plus its offset; element n (= C) receives the grand total
__global__ void __launch_bounds__(kScanThreads) k_scan_final(int* __restrict__ counts, int n, const int* __restrict__ tile_sums)
{
    const int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    int v[kScanItems];
    int s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = (base + i < n) ? counts[base + i] : 0;
        s += v[i];
    }
    int total;
    int run = block_exclusive_scan(s, total) + tile_sums[blockIdx.x];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (base + i <= n) counts[base + i] = run;   // index n gets the total (all later v are 0)
        run += v[i];
    }
}

// second half of a3: scatter into the cell-sorted SoA.  src_tag == nullptr: source is the caller's tag-order pos4/quat4;
// otherwise the source is the other sorted buffer (2-D: poses only).
__global__ void k_scatter(int N, int dim, const float4* __restrict__ src_pos, const float4* __restrict__ src_quat,
                          const int* __restrict__ src_tag, const int2* __restrict__ key_rank,
                          const int* __restrict__ cell_start, float4* __restrict__ dst_pos, float4* __restrict__ dst_quat,
                          int* __restrict__ dst_tag)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int2 kr = key_rank[p];
    const int dst = cell_start[kr.x] + kr.y;
    const float4 P = src_pos[p];
    if (dim == 2) {
        if (src_tag) dst_pos[dst] = P;
        else {
            const float4 Q = src_quat[p];
            dst_pos[dst] = make_float4(P.x, P.y, Q.x, Q.w);
        }
    } else {
        dst_pos[dst] = P;
        dst_quat[dst] = src_quat[p];
    }
    dst_tag[dst] = src_tag ? src_tag[p] : p;
}

// R8: members of a cell in ascending tag, whatever order the atomics produced
__global__ void k_cell_sort(int C, int dim, const int* __restrict__ cell_start, float4* __restrict__ pos, float4* __restrict__ quat,
                            int* __restrict__ tag)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const int s = cell_start[c], e = cell_start[c + 1];
    for (int i = s + 1; i < e; ++i) {
        const int ti = tag[i];
        int j = i - 1;
        if (tag[j] <= ti) continue;
        const float4 pi = pos[i];
        float4 qi = pi;
        if (dim == 3) qi = quat[i];
        while (j >= s && tag[j] > ti) {
            tag[j + 1] = tag[j];
            pos[j + 1] = pos[j];
            if (dim == 3) quat[j + 1] = quat[j];
            --j;
        }
        tag[j + 1] = ti;
        pos[j + 1] = pi;
        if (dim == 3) quat[j + 1] = qi;
    }
}

// a13: back to tag order
__global__ void k_unsort(int N, int dim, const float4* __restrict__ pos, const float4* __restrict__ quat, const int* __restrict__ tag,
                         float4* __restrict__ out_pos, float4* __restrict__ out_quat)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int t = tag[p];
    float4 x, q;
    load_state(dim, pos, quat, p, x, q);
    if (out_pos) out_pos[t] = x;
    if (out_quat) out_quat[t] = q;
}

// debug: cell id of every particle in tag order, from the (cell, rank) pairs of the last build
__global__ void k_cell_of_tag(int N, const int2* __restrict__ key_rank, const int* __restrict__ src_tag, int* __restrict__ out)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    out[src_tag ? src_tag[p] : p] = key_rank[p].x;
}

}  // namespace hpmc
