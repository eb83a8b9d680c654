// Cell-list builder (S:8(a) rows a1-a3): sweep header, cell id, histogram, exclusive scan, scatter into
// the cell-sorted SoA, canonical in-cell order (ascending tag, R8), plus the un-sort for get_state (a13).
// "A bucket sort efficiently assigns particles to cells, and a massively parallel bucket sort on the GPU
// is trivial to implement with atomic operations".
#pragma once
#include "common.cuh"

namespace hpmc {

constexpr int kScanThreads = 512;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;

// Three launches build the cell list of a sweep:
//   k_hist          header (a0, a1) + cell id and arrival rank of every particle (a2, first half of a3)
//   k_scan          single-pass exclusive scan of the per-cell counts (decoupled look-back), zeroes the counts for the
//                   next build, advances the sweep counter
//   k_scatter_sort  scatter into the cell-sorted SoA; the last particle to arrive in a cell puts the cell's members in
//                   ascending tag order (R8)
// mode 0: header of the device sweep counter t; k_scan then does t++ and sweeps++   (a real sweep)
// mode 1: header of t_override, nothing advanced                                     (debug cell list)
// mode 2: zero shift, nothing advanced                                               (validator)

// a0-a2 + first half of a3.  Every block derives the same header from the (unchanged) sweep counter; block 0 stores it for
// the kernels that follow.  `counts` is all zero on entry (bind, then k_scan after every use).
__global__ void k_hist(const __grid_constant__ GridParams g, Control* __restrict__ ctrl, const float4* __restrict__ pos,
                       int* __restrict__ counts, int2* __restrict__ key_rank, uint32_t k0, uint32_t k1, int mode,
                       unsigned long long t_override)
{
    __shared__ SweepHeader sh;
    if (threadIdx.x == 0) {
        const unsigned long long t = (mode == 0) ? ctrl->t : t_override;
        make_header(g, k0, k1, t, mode == 2, sh);
        sh.pad = 0;
        if (blockIdx.x == 0) ctrl->hdr = sh;
    }
    __syncthreads();
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.N) return;
    const float shift[3] = {sh.shift[0], sh.shift[1], sh.shift[2]};
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

// tile state of the single-pass scan: value (low 32 bits) | epoch << 34 | status << 32; status 1 = tile aggregate,
// 2 = inclusive prefix.  The epoch makes words of earlier launches invalid without clearing the array.
__device__ __forceinline__ unsigned long long scan_pack(unsigned int value, unsigned int status, unsigned long long epoch)
{
    return (unsigned long long)value | ((unsigned long long)status << 32) | (epoch << 34);
}

// second quarter of a3: cell_start[i] = sum of counts[0..i) for i = 0..n (n = C: the grand total), one pass.
// Tiles take tickets so that every predecessor of a tile is already resident (no deadlock in the look-back).
__global__ void __launch_bounds__(kScanThreads)
k_scan(int* __restrict__ counts, int n, int* __restrict__ cell_start, unsigned long long* __restrict__ tile_state,
       Control* __restrict__ ctrl, int ntiles, int mode)
{
    __shared__ int s_tile;
    __shared__ int s_prefix;
    __shared__ unsigned long long s_epoch;
    if (threadIdx.x == 0) {
        s_epoch = ctrl->scan_epoch;                       // read BEFORE taking the ticket (see the last tile below)
        s_tile = (int)atomicAdd(&ctrl->scan_ticket, 1u);
    }
    __syncthreads();
    const int tile = s_tile;
    const unsigned long long epoch = s_epoch & 0x3fffffffull;
    // warp w owns 32*kScanItems consecutive counts; item k of lane l is element k*32 + l of that chunk: every load and
    // store is one coalesced 128-byte line per warp
    __shared__ int s_wsum[kScanThreads / 32];
    const int lane_ = threadIdx.x & 31, warp_ = threadIdx.x >> 5;
    const int wbase = tile * kScanTile + warp_ * (32 * kScanItems) + lane_;
    int v[kScanItems], ex[kScanItems];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int idx = wbase + 32 * k;
        v[k] = (idx <= n) ? counts[idx] : 0;
    }
    int carry = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int idx = wbase + 32 * k;
        if (idx <= n) counts[idx] = 0;                    // ready for the next build
        const int inc = warp_inclusive_scan(v[k]);
        ex[k] = carry + inc - v[k];
        carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane_ == 0) s_wsum[warp_] = carry;
    __syncthreads();
    int woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        const int t = s_wsum[w];
        if (w < warp_) woff += t;
        total += t;
    }
    if (threadIdx.x < 32) {                               // warp 0: publish, look back 32 tiles at a time
        volatile unsigned long long* st = tile_state;
        const int lane = threadIdx.x;
        int prefix = 0;
        if (lane == 0) st[tile] = scan_pack((unsigned)total, tile == 0 ? 2u : 1u, epoch);
        for (int j = tile - 1; j >= 0; j -= 32) {
            const int idx = j - lane;
            unsigned long long w = scan_pack(0u, 2u, epoch);          // before tile 0: an inclusive prefix of zero
            if (idx >= 0)
                do { w = st[idx]; } while ((w >> 34) != epoch || ((w >> 32) & 3ull) == 0ull);
            const unsigned incl = __ballot_sync(0xffffffffu, ((w >> 32) & 3ull) == 2ull);
            const int first = incl ? __ffs(incl) - 1 : 31;            // nearest tile that already knows its inclusive prefix
            prefix += __reduce_add_sync(0xffffffffu, lane <= first ? (int)(unsigned int)w : 0);
            if (incl) break;
        }
        if (lane == 0) {
            if (tile != 0) st[tile] = scan_pack((unsigned)(prefix + total), 2u, epoch);
            s_prefix = prefix;
            if (tile == ntiles - 1) {                     // every other tile has already read the epoch and its ticket
                ctrl->scan_ticket = 0u;
                ctrl->scan_epoch = (epoch + 1ull) & 0x3fffffffull;
                if (mode == 0) {
                    ctrl->t += 1ull;
                    ctrl->sweeps += 1ull;
                }
            }
        }
    }
    __syncthreads();
    const int off = s_prefix + woff;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int idx = wbase + 32 * k;
        if (idx <= n) cell_start[idx] = off + ex[k];
    }
}

// second half of a3: scatter into the cell-sorted SoA.  src_tag == nullptr: source is the caller's tag-order pos4/quat4;
// otherwise the source is the other sorted buffer (2-D: poses only).  In a cell with several members the LAST particle to
// arrive (counted in `arrived`, which it resets) sorts the members by tag (R8), whatever order the atomics produced.
__global__ void k_scatter_sort(int N, int dim, const float4* __restrict__ src_pos, const float4* __restrict__ src_quat,
                               const int* __restrict__ src_tag, const int2* __restrict__ key_rank,
                               const int* __restrict__ cell_start, int* __restrict__ arrived, float4* dst_pos, float4* dst_quat,
                               int* dst_tag)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int2 kr = key_rank[p];
    const int s = cell_start[kr.x], cnt = cell_start[kr.x + 1] - s;
    const int dst = s + kr.y;
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
    if (cnt < 2) return;
    __threadfence();
    if (atomicAdd(&arrived[kr.x], 1) != cnt - 1) return;
    __threadfence();
    arrived[kr.x] = 0;
    // insertion sort of the cell by tag; loads bypass L1 (other SMs wrote these lines during this kernel)
    for (int i = s + 1; i < s + cnt; ++i) {
        const int ti = __ldcg(&dst_tag[i]);
        int j = i - 1;
        if (__ldcg(&dst_tag[j]) <= ti) continue;
        const float4 pi = __ldcg(&dst_pos[i]);
        float4 qi = pi;
        if (dim == 3) qi = __ldcg(&dst_quat[i]);
        while (j >= s && __ldcg(&dst_tag[j]) > ti) {
            dst_tag[j + 1] = __ldcg(&dst_tag[j]);
            dst_pos[j + 1] = __ldcg(&dst_pos[j]);
            if (dim == 3) dst_quat[j + 1] = __ldcg(&dst_quat[j]);
            --j;
        }
        dst_tag[j + 1] = ti;
        dst_pos[j + 1] = pi;
        if (dim == 3) dst_quat[j + 1] = qi;
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
