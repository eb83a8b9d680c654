// Cell-list builder (S:8(a) rows a1-a3): sweep header, cell id, histogram, exclusive scan, scatter into
// the cell-sorted SoA, canonical in-cell order (ascending tag, R8), plus the un-sort for get_state (a13).
// "A bucket sort efficiently assigns particles to cells, and a massively parallel bucket sort on the GPU
// is trivial to implement with atomic operations".
#pragma once
#include "common.cuh"

namespace hpmc {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;
constexpr int kHistItems = 4;     // particles per thread of k_hist
constexpr int kFusedSpineMax = 1024;   // up to this many scan tiles k_scan_final adds up the preceding tile totals itself (no spine launch)

// Three to five launches build the cell list of a sweep:
//   k_hist          header (a0, a1) + cell id and arrival rank of every particle (a2, first half of a3)
//   k_scan_*        exclusive scan of the per-cell counts (one launch when the grid fits one tile of 16 384 counts, else
//                   reduce / spine / final), zeroes the counts for the next build, advances the sweep counter
//   k_scatter       scatter into the cell-sorted SoA; k_sort_cells then puts the members of every cell in
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
    pdl_launch_dependents();
    pdl_wait();
    __shared__ SweepHeader sh;
    if (threadIdx.x == 0) {
        const unsigned long long t = (mode == 0) ? ctrl->t : t_override;
        make_header(g, k0, k1, t, mode == 2, sh);
        sh.pad = 0;
        if (blockIdx.x == 0) ctrl->hdr = sh;
    }
    __syncthreads();
    const float shift[3] = {sh.shift[0], sh.shift[1], sh.shift[2]};
    // kHistItems particles per thread, a block-wide stride apart (coalesced): their loads and their atomics are in flight together
    const int base = blockIdx.x * (blockDim.x * kHistItems) + threadIdx.x;
    float4 x[kHistItems];
    int c[kHistItems], rank[kHistItems];
#pragma unroll
    for (int j = 0; j < kHistItems; ++j) {
        const int p = base + j * blockDim.x;
        if (p < g.N) x[j] = pos[p];
    }
#pragma unroll
    for (int j = 0; j < kHistItems; ++j) {
        const int p = base + j * blockDim.x;
        if (p < g.N) {
            bool bad;
            c[j] = cell_of_checked(g, shift, x[j].x, x[j].y, (g.dim == 3) ? x[j].z : 0.0f, bad);
            if (bad) atomicAdd(&ctrl->bad_coords, 1u);
            rank[j] = atomicAdd(&counts[c[j]], 1);
        }
    }
#pragma unroll
    for (int j = 0; j < kHistItems; ++j) {
        const int p = base + j * blockDim.x;
        if (p < g.N) key_rank[p] = make_int2(c[j], rank[j]);
    }
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

// second quarter of a3: cell_start[i] = sum of counts[0..i) for i = 0..n (n = C: the grand total).  Warp w of a tile owns
// 32*kScanItems consecutive counts; item k of lane l is element k*32 + l of that chunk, so every load and store is one
// coalesced 128-byte line per warp.  A grid that fits one tile (configs 0, 1, 3) runs k_scan_final alone; larger ones run
// reduce -> spine -> final.  (A single-pass decoupled look-back scan was measured slower here: its inclusive-prefix
// wavefront advances 32 tiles per L2 round trip, 0.77 TB/s on 16.7 M counts.)
__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const int* __restrict__ counts, int n, int* __restrict__ tile_sums)
{
    pdl_launch_dependents();
    pdl_wait();
    __shared__ int s_wsum[kScanThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wbase = blockIdx.x * kScanTile + warp * (32 * kScanItems) + lane;
    int s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int idx = wbase + 32 * k;
        if (idx <= n) s += counts[idx];
    }
    s = __reduce_add_sync(0xffffffffu, s);
    if (lane == 0) s_wsum[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) t += s_wsum[w];
        tile_sums[blockIdx.x] = t;
    }
}

// exclusive scan of the tile totals by ONE block; also advances the sweep counter of a real sweep (mode 0)
__global__ void __launch_bounds__(kScanThreads) k_scan_spine(int* __restrict__ tile_sums, int ntiles, Control* __restrict__ ctrl, int mode)
{
    pdl_launch_dependents();
    pdl_wait();
    __shared__ int carry_s;
    if (threadIdx.x == 0) {
        carry_s = 0;
        if (mode == 0) {
            ctrl->t += 1ull;
            ctrl->sweeps += 1ull;
        }
    }
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

// exclusive scan inside each tile plus the tile's offset; re-zeroes the counts for the next build.  single = 1: the whole grid
// is one tile (no reduce pass ran); single = 2: the reduce pass ran but no spine -- the block sums the preceding tile totals
// itself; in both cases this kernel also advances the sweep counter.  single = 0: tile_sums holds the spine's prefix.
__global__ void __launch_bounds__(kScanThreads)
k_scan_final(int* __restrict__ counts, int n, int* __restrict__ cell_start, const int* __restrict__ tile_sums, int single,
             Control* __restrict__ ctrl, int mode)
{
    pdl_launch_dependents();
    pdl_wait();
    __shared__ int s_wsum[kScanThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wbase = blockIdx.x * kScanTile + warp * (32 * kScanItems) + lane;
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
    if (lane == 0) s_wsum[warp] = carry;
    // offset of this tile: nothing (one tile), the spine's exclusive prefix, or -- fused -- the sum of the preceding tile totals,
    // added up here by the block itself (a few hundred L2-resident values: cheaper than a launch of its own)
    __shared__ int s_tile_off;
    if (single == 2) {
        int part = 0;
        for (int i = threadIdx.x; i < (int)blockIdx.x; i += kScanThreads) part += tile_sums[i];
        part = __reduce_add_sync(0xffffffffu, part);
        __shared__ int s_psum[kScanThreads / 32];
        if (lane == 0) s_psum[warp] = part;
        __syncthreads();
        if (threadIdx.x == 0) {
            int t = 0;
#pragma unroll
            for (int w = 0; w < kScanThreads / 32; ++w) t += s_psum[w];
            s_tile_off = t;
        }
    }
    __syncthreads();
    int off = (single == 1) ? 0 : (single == 2) ? s_tile_off : tile_sums[blockIdx.x];
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w)
        if (w < warp) off += s_wsum[w];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int idx = wbase + 32 * k;
        if (idx <= n) cell_start[idx] = off + ex[k];
    }
    if (single && mode == 0 && threadIdx.x == 0 && blockIdx.x == 0) {
        ctrl->t += 1ull;
        ctrl->sweeps += 1ull;
    }
}

// second half of a3: scatter into the cell-sorted SoA.  src_tag == nullptr: source is the caller's tag-order pos4/quat4;
// otherwise the source is the other sorted buffer (2-D: poses only).  Members of a cell land in arrival order (k_sort_cells).
__global__ void k_scatter(int N, int dim, const float4* __restrict__ src_pos, const float4* __restrict__ src_quat,
                          const int* __restrict__ src_tag, const int2* __restrict__ key_rank, const int* __restrict__ cell_start,
                          float4* __restrict__ dst_pos, float4* __restrict__ dst_quat, int* __restrict__ dst_tag)
{
    pdl_launch_dependents();
    pdl_wait();
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

// last quarter of a3 (R8): one thread per cell puts the members of a multiply-occupied cell in ascending tag, whatever order
// the atomics of k_hist produced.  A launch of its own: the scatter's stores are then visible without fences, the cells of
// neighbouring threads are neighbours in memory, and no thread spins through dependent L2 loads while its warp waits
// (measured on 1 M pentagons: scatter + sort 9.8 + ~5 us against 25 us for the scatter whose last arrival sorted the cell).
// Cells of up to kSortRegs members (all but freak cells) are sorted in registers: every tag is loaded at once, the rank of a
// member is the number of smaller tags in its cell, then every pose is loaded at once and stored at its rank -- two rounds of
// independent loads instead of an insertion sort's chain of dependent global loads and stores (config 3, ~3 members per cell:
// 17 -> 6 us under ncu).
template <int M>
__device__ __forceinline__ void sort_cell_in_registers(int s, int n, int dim, float4* pos, float4* quat, int* tag)
{
    int t[M], r[M];
#pragma unroll
    for (int k = 0; k < M; ++k) t[k] = (k < n) ? tag[s + k] : 0x7fffffff;   // padding ranks behind every member
    bool sorted = true;
#pragma unroll
    for (int k = 0; k < M; ++k) {
        int rk = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) rk += (j != k && t[j] < t[k]) ? 1 : 0;   // tags are distinct
        r[k] = rk;
        sorted = sorted && (k >= n || rk == k);
    }
    if (sorted) return;
    float4 P[M];
#pragma unroll
    for (int k = 0; k < M; ++k)
        if (k < n) P[k] = pos[s + k];
#pragma unroll
    for (int k = 0; k < M; ++k)
        if (k < n) { pos[s + r[k]] = P[k]; tag[s + r[k]] = t[k]; }
    if (dim == 3) {
#pragma unroll
        for (int k = 0; k < M; ++k)
            if (k < n) P[k] = quat[s + k];
#pragma unroll
        for (int k = 0; k < M; ++k)
            if (k < n) quat[s + r[k]] = P[k];
    }
}

// DIM = 3 only takes the register path: 2-D cells hold one particle, sometimes two (the insertion sort is then one compare
// and one swap), and the 1 M-thread launch of config 2 is 5 us slower with the 78 registers of the register path.
template <int DIM>
__global__ void k_sort_cells(int C, const int* __restrict__ cell_start, float4* pos, float4* quat, int* tag)
{
    constexpr int dim = DIM;
    pdl_launch_dependents();
    pdl_wait();
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const int s = cell_start[c], e = cell_start[c + 1];
    const int n = e - s;
    if (n < 2) return;
    if (DIM == 3 && n <= 4) { sort_cell_in_registers<4>(s, n, dim, pos, quat, tag); return; }
    if (DIM == 3 && n <= 8) { sort_cell_in_registers<8>(s, n, dim, pos, quat, tag); return; }
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

// Small systems (configs 0, 1): the whole cell-list build in ONE CTA -- header, histogram in shared memory, scan, scatter,
// in-cell tag sort -- instead of three launches whose latencies and gaps are a third of such a sweep.  Same results as the
// k_hist / k_scan_final / k_scatter / k_sort_cells sequence (the arrival ranks differ, the sorted result does not).  Dynamic shared
// memory: (C + 2) ints.  `counts` and `arrived` are not touched (they stay all-zero).
constexpr int kSmallBuildThreads = 1024;
constexpr int kSmallBuildMaxCells = 11500;    // (C + 2) * 4 bytes of shared memory <= 46 KB
constexpr int kSmallBuildMaxN = 8192;       // measured: config 3 (32 768 particles) is 20 % slower with one CTA, config 1 is 5 % faster

__global__ void __launch_bounds__(kSmallBuildThreads)
k_build_small(const __grid_constant__ GridParams g, Control* __restrict__ ctrl, uint32_t k0, uint32_t k1, int mode,
              unsigned long long t_override, const float4* __restrict__ src_pos, const float4* __restrict__ src_quat,
              const int* __restrict__ src_tag, int2* __restrict__ key_rank, int* __restrict__ cell_start, float4* dst_pos,
              float4* dst_quat, int* dst_tag)
{
    pdl_launch_dependents();
    pdl_wait();
    extern __shared__ int s_off[];            // counts, then exclusive offsets, C + 1 entries
    __shared__ SweepHeader sh;
    __shared__ int s_part[kSmallBuildThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = g.C;                        // entries 0..n
    if (tid == 0) {
        const unsigned long long t = (mode == 0) ? ctrl->t : t_override;
        make_header(g, k0, k1, t, mode == 2, sh);
        sh.pad = 0;
        ctrl->hdr = sh;
        if (mode == 0) {
            ctrl->t = t + 1ull;
            ctrl->sweeps += 1ull;
        }
    }
    for (int i = tid; i <= n; i += kSmallBuildThreads) s_off[i] = 0;
    __syncthreads();
    // a2 + histogram
    const float shift[3] = {sh.shift[0], sh.shift[1], sh.shift[2]};
    for (int p = tid; p < g.N; p += kSmallBuildThreads) {
        const float4 x = src_pos[p];
        bool bad;
        const int c = cell_of_checked(g, shift, x.x, x.y, (g.dim == 3) ? x.z : 0.0f, bad);
        if (bad) atomicAdd(&ctrl->bad_coords, 1u);
        key_rank[p] = make_int2(c, atomicAdd(&s_off[c], 1));
    }
    __syncthreads();
    // exclusive scan of n + 1 counts: each thread owns a run of consecutive entries
    const int per = (n + 1 + kSmallBuildThreads - 1) / kSmallBuildThreads;
    const int lo = tid * per, hi = min(lo + per, n + 1);
    int sum = 0;
    for (int i = lo; i < hi; ++i) sum += s_off[i];
    const int inc = warp_inclusive_scan(sum);
    if (lane == 31) s_part[warp] = inc;
    __syncthreads();
    int run = inc - sum;
    for (int w = 0; w < warp; ++w) run += s_part[w];
    for (int i = lo; i < hi; ++i) {
        const int v = s_off[i];
        s_off[i] = run;
        cell_start[i] = run;
        run += v;
    }
    __syncthreads();
    // scatter (second half of a3)
    for (int p = tid; p < g.N; p += kSmallBuildThreads) {
        const int2 kr = key_rank[p];
        const int dst = s_off[kr.x] + kr.y;
        const float4 P = src_pos[p];
        if (g.dim == 2) {
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
    __syncthreads();
    // R8: members of a cell in ascending tag
    for (int c = tid; c < n; c += kSmallBuildThreads) {
        const int s = s_off[c], e = s_off[c + 1];
        for (int i = s + 1; i < e; ++i) {
            const int ti = dst_tag[i];
            int j = i - 1;
            if (dst_tag[j] <= ti) continue;
            const float4 pi = dst_pos[i];
            float4 qi = pi;
            if (g.dim == 3) qi = dst_quat[i];
            while (j >= s && dst_tag[j] > ti) {
                dst_tag[j + 1] = dst_tag[j];
                dst_pos[j + 1] = dst_pos[j];
                if (g.dim == 3) dst_quat[j + 1] = dst_quat[j];
                --j;
            }
            dst_tag[j + 1] = ti;
            dst_pos[j + 1] = pi;
            if (g.dim == 3) dst_quat[j + 1] = qi;
        }
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
