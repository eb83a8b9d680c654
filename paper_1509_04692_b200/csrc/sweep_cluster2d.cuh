// Whole sweeps of a SMALL 2-D system in ONE launch of ONE thread-block cluster (S:8(a) rows a0-a11; BASELINE.json's
// 4096-disk and 4096-pentagon configs).
//
// Such a system is far below one wave of the GPU: a sweep is ~15 000 trials, microseconds of arithmetic, and what it costs is
// latency -- five dependent launches per sweep (build + four colours) and their drain/launch gaps.  Here one cluster of up
// to 16 CTAs (16 SMs of one GPC, 16 384 threads) runs `n_sweeps` complete sweeps back to back, separated only by hardware
// cluster barriers (barrier.cluster, ~0.2 us; release/acquire at cluster scope orders the global-memory traffic between the
// CTAs), seven per sweep:
//
//   header      every CTA derives the sweep's grid shift and colour order with Philox (a0, a1)
//   histogram   one thread per particle: pinned cell function, arrival rank from an L2 atomic (a2)           | barrier
//   scan        EVERY CTA scans all C+1 counts into its own shared memory: cell_start lookups are local      |
//   scatter     into the other sorted buffer (ping-pong), global memory / L2 (a3)                            | barrier
//   tag sort    one thread per multiply-occupied cell: members in ascending tag (R8)                         | barrier
//   4 colours   a group of G lanes per active cell (G = 8 disks, 16 polygons): the 3x3 neighbourhood is staged in shared
//               memory, then the cell's n_select trials run as in the warp-per-cell pass -- Philox and the trial pose on
//               every lane, the lanes stride over the candidates (a8), ballot-packed queue (a10), one narrow test per lane
//               (a9), group vote, lane 0 writes back (a11)                                                   | barrier each
//
// Results are identical to every other colour-pass variant (same Philox keys, same make_trial, same polygon_separated).
// The state stays in global memory (it is L2-resident by size); only cell_start and the staged neighbourhoods live in shared
// memory.  Neighbourhoods larger than the staging capacity fall back to the per-thread path on the group's first lane.
#pragma once
#include "common.cuh"
#include "overlap.cuh"
#include "sweep.cuh"

namespace hpmc {

constexpr int kClThreads = 1024;          // threads per CTA
constexpr int kClMaxCells = 11500;        // (C + 2) ints of shared memory for cell_start

__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}

__device__ __forceinline__ unsigned cluster_nctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}

template <int G>
struct ClusterUnit {                       // staging of one group of G lanes
    static constexpr int CAP = (G >= 16) ? 2 * G : 3 * G;   // staged poses: the broad phase is at most CAP / G strides of the group
    float4 pose[CAP];
    int gidx[CAP];
    unsigned char queue[CAP];
};

template <int G>
constexpr size_t cluster_smem_bytes(int C)
{
    return sizeof(int) * (size_t)((C + 2 + 3) / 4 * 4) + sizeof(ClusterUnit<G>) * (kClThreads / G);
}

// pos[2] / tag[2]: the two cell-sorted buffers; `cur` holds the state on entry, and after n_sweeps sweeps buffer
// cur ^ (n_sweeps & 1) holds it.  counts: C+1 zeros on entry and on exit.  cell_start_g: the last sweep's CSR on exit.
template <int KIND, int NV, int G>
__global__ void __launch_bounds__(kClThreads, 1)
k_sweep_cluster2d(const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv, const __grid_constant__ ShapeF S,
                  const __grid_constant__ ShapeD SD, Control* __restrict__ ctrl, int n_sweeps, int cur, float4* pos0, float4* pos1,
                  int* tag0, int* tag1, int* __restrict__ counts, int* __restrict__ cell_start_g, uint32_t k0, uint32_t k1,
                  uint2* __restrict__ trace)
{
    using Unit = ClusterUnit<G>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int* s_start = reinterpret_cast<int*>(smem_raw);                                      // C + 1 offsets (every CTA: all of them)
    Unit* s_units = reinterpret_cast<Unit*>(smem_raw + sizeof(int) * (size_t)((g.C + 2 + 3) / 4 * 4));
    __shared__ SweepHeader sh;
    __shared__ int s_part[kClThreads / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rank = (int)cluster_ctarank(), ncta = (int)cluster_nctarank();
    const int T = ncta * kClThreads, gt = rank * kClThreads + tid;       // threads of the cluster, this thread's index
    const int lig = lane & (G - 1), gbase = lane & ~(G - 1);              // lane in group, first lane of the group
    const unsigned gmask = (G == 32) ? 0xffffffffu : (((1u << G) - 1u) << gbase);
    Unit& U = s_units[tid / G];
    const int unit = gt / G, nunits = T / G;
    const int n0 = g.n[0], n1 = g.n[1], nax = n0 >> 1, nay = n1 >> 1, nactive = nax * nay;
    const int C = g.C, N = g.N;
    const unsigned long long t_first = ctrl->t;
    CellCounters cc;

    for (int sweep = 0; sweep < n_sweeps; ++sweep) {
        const float4* src_pos = cur ? pos1 : pos0;
        const int* src_tag = cur ? tag1 : tag0;
        float4* dst_pos = cur ? pos0 : pos1;
        int* dst_tag = cur ? tag0 : tag1;
        // ---- header (a0, a1) -------------------------------------------------------------------------------------------
        if (tid == 0) {
            make_header(g, k0, k1, t_first + (unsigned long long)sweep, false, sh);
            sh.pad = 0;
            if (rank == 0) ctrl->hdr = sh;
        }
        __syncthreads();
        const float shift[3] = {sh.shift[0], sh.shift[1], 0.0f};
        const uint32_t t_lo = sh.t_lo, t_hi16 = sh.t_hi16;
        // ---- histogram (a2): one thread per particle (N <= T) ----------------------------------------------------------
        float4 my_pose = make_float4(0.f, 0.f, 1.f, 0.f);
        int my_tag = 0, my_cell = -1, my_rank = 0;
        if (gt < N) {
            my_pose = __ldcg(&src_pos[gt]);
            my_tag = __ldcg(&src_tag[gt]);
            int cx, cy, cz;
            my_cell = cell_of(g, shift, my_pose.x, my_pose.y, 0.0f, cx, cy, cz);
            my_rank = atomicAdd(&counts[my_cell], 1);
        }
        cluster_barrier();
        // ---- scan: every CTA builds the whole CSR in its own shared memory ----------------------------------------------
        for (int i = tid; i <= C; i += kClThreads) s_start[i] = __ldcg(&counts[i]);
        __syncthreads();
        {
            const int per = (C + 1 + kClThreads - 1) / kClThreads;
            const int lo = tid * per, hi = min(lo + per, C + 1);
            int sum = 0;
            for (int i = lo; i < hi; ++i) sum += s_start[i];
            int inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += n;
            }
            if (lane == 31) s_part[warp] = inc;
            __syncthreads();
            int run = inc - sum;
            for (int w = 0; w < warp; ++w) run += s_part[w];
            for (int i = lo; i < hi; ++i) {
                const int v = s_start[i];
                s_start[i] = run;
                run += v;
            }
        }
        __syncthreads();
        if (rank == 0)
            for (int i = tid; i <= C; i += kClThreads) cell_start_g[i] = s_start[i];   // for the fallback path and later builds
        // ---- scatter (a3) ----------------------------------------------------------------------------------------------------
        if (gt < N) {
            const int dst = s_start[my_cell] + my_rank;
            dst_pos[dst] = my_pose;
            dst_tag[dst] = my_tag;
        }
        cluster_barrier();
        for (int i = gt; i <= C; i += T) counts[i] = 0;                                 // every CTA has read them: ready for the next build
        // ---- R8: members of a cell in ascending tag ------------------------------------------------------------------------
        for (int c = gt; c < C; c += T) {
            const int s = s_start[c], e = s_start[c + 1];
            for (int i = s + 1; i < e; ++i) {
                const int ti = __ldcg(&dst_tag[i]);
                int j = i - 1;
                if (__ldcg(&dst_tag[j]) <= ti) continue;
                const float4 pi = __ldcg(&dst_pos[i]);
                while (j >= s && __ldcg(&dst_tag[j]) > ti) {
                    dst_tag[j + 1] = __ldcg(&dst_tag[j]);
                    dst_pos[j + 1] = __ldcg(&dst_pos[j]);
                    --j;
                }
                dst_tag[j + 1] = ti;
                dst_pos[j + 1] = pi;
            }
        }
        cluster_barrier();
        // ---- the four colours (a4-a11) ------------------------------------------------------------------------------------------
        for (int ci = 0; ci < 4; ++ci) {
            const int gamma = sh.perm[ci];
            const uint32_t c3 = (kTagTrial << 24) | ((uint32_t)gamma << 16) | t_hi16;
            // every lane of a warp runs the same number of rounds (the collectives below are warp-wide)
            const int rounds = (nactive + nunits - 1) / nunits;
            for (int r = 0; r < rounds; ++r) {
                const int idx = r * nunits + unit;
                const bool live = idx < nactive;
                const int ix = live ? idx % nax : 0, iy = live ? idx / nax : 0;
                const int cx = 2 * ix + (gamma & 1), cy = 2 * iy + ((gamma >> 1) & 1);
                const int cell = cx + n0 * cy;
                const long long slot0 = (long long)cell * mv.n_select;
                const bool seam = cx == 0 || cy == 0 || cx >= n0 - 2 || cy >= n1 - 2;
                // staging (a7): lane j of the group owns neighbour cell j = (dy+1)*3 + (dx+1), and cell j + G if that is below 9
                int my_start[2] = {0, 0}, my_cnt[2] = {0, 0};
#pragma unroll
                for (int h = 0; h < ((G >= 9) ? 1 : 2); ++h) {
                    const int j = lig + h * G;
                    if (live && j < 9) {
                        int nx = cx + (j % 3) - 1, ny = cy + (j / 3) - 1;
                        nx += (nx < 0) ? n0 : 0; nx -= (nx >= n0) ? n0 : 0;
                        ny += (ny < 0) ? n1 : 0; ny -= (ny >= n1) ? n1 : 0;
                        const int c = nx + n0 * ny;
                        my_start[h] = s_start[c];
                        my_cnt[h] = s_start[c + 1] - my_start[h];
                    }
                }
                int incl = my_cnt[0];   // inclusive prefix of the first cells inside the group
#pragma unroll
                for (int o = 1; o < G; o <<= 1) {
                    const int n = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lig >= o) incl += n;
                }
                const int total0 = __shfl_sync(0xffffffffu, incl, gbase + G - 1);
                const int total = total0 + ((G >= 9) ? 0 : __shfl_sync(0xffffffffu, my_cnt[1], gbase));   // G = 8: cell 8 sits on lane 0
                const int own_s = __shfl_sync(0xffffffffu, incl - my_cnt[0], gbase + 4);
                const int nmem = __shfl_sync(0xffffffffu, my_cnt[0], gbase + 4);
                const bool staged = total <= Unit::CAP;
                if (live && nmem > 0 && staged) {
                    // a lane copies its cells' members; cells hold a few particles each
                    for (int e = 0; e < my_cnt[0]; ++e) {
                        const int gi = my_start[0] + e, at = incl - my_cnt[0] + e;
                        U.pose[at] = __ldcg(&dst_pos[gi]);
                        U.gidx[at] = gi;
                    }
                    if (G < 9)
                        for (int e = 0; e < my_cnt[1]; ++e) {
                            const int gi = my_start[1] + e, at = total0 + e;
                            U.pose[at] = __ldcg(&dst_pos[gi]);
                            U.gidx[at] = gi;
                        }
                }
                // strides of the broad phase: as many as the fullest neighbourhood of this warp needs (warp-uniform)
                const int nstride = (__reduce_max_sync(0xffffffffu, (live && nmem > 0 && staged) ? total : 0) + G - 1) / G;
                __syncwarp();
                if (live && nmem == 0 && trace && lig == 0)
                    for (int k = 0; k < mv.n_select; ++k) trace[slot0 + k] = make_uint2(0u, 0u);
                if (live && nmem > 0 && !staged && lig == 0)      // neighbourhood above the staging capacity: per-thread path
                    sweep_cell_global<KIND, NV>(g, mv, S, SD, gamma, t_lo, t_hi16, shift, cx, cy, 0, dst_pos, nullptr, dst_tag, cell_start_g,
                                                k0, k1, trace, cc);
                const bool work = live && nmem > 0 && staged;
                if (!__any_sync(0xffffffffu, work)) continue;   // a warp with nothing to do leaves the issue slots to the others
                U4 blk{0u, 0u, 0u, 0u};
                for (int k = 0; k < mv.n_select; ++k) {
                    // a0: lane j of the group draws the Philox block of trial k + j for the next G trials at once, off the
                    // critical path of the sequential trials; the trial then broadcasts its block
                    if ((k & (G - 1)) == 0) blk = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)(k + lig), c3, k0, k1);
                    const int src = gbase + (k & (G - 1));
                    const U4 b0{__shfl_sync(0xffffffffu, blk.x, src), __shfl_sync(0xffffffffu, blk.y, src), __shfl_sync(0xffffffffu, blk.z, src),
                                __shfl_sync(0xffffffffu, blk.w, src)};
                    // phase A: trial pose, identical on every lane of the group (a5, a6)
                    int p = 0, outcome = 0;
                    bool rotate = false;
                    TrialState A{};
                    if (work) {
                        p = own_s + (int)mulhi32(b0.x, (uint32_t)nmem);   // R8
                        const float4 P = U.pose[p];
                        outcome = make_trial<KIND>(g, mv, shift, cell, 2, b0, 0u, make_float4(P.x, P.y, 0.f, 0.f), make_float4(P.z, 0.f, 0.f, P.w),
                                                   A, rotate) ? 1 : 2;
                    }
                    const float4 Tp = make_float4(A.x, A.y, A.qw, A.qz);
                    // broad phase (a8): the group strides over the staged candidates; survivors to the queue (a10)
                    int nq = 0;
                    bool sure = false;
                    for (int st = 0; st < nstride; ++st) {
                        const int q = st * G + lig;
                        bool hit = false;
                        if (outcome == 1 && q < total && q != p) {
                            const float4 B = U.pose[q];
                            const float rx = seam ? min_image(B.x, Tp.x, g.hi[0], g.Ld[0]) : B.x - Tp.x;
                            const float ry = seam ? min_image(B.y, Tp.y, g.hi[1], g.Ld[1]) : B.y - Tp.y;
                            const float d2 = rx * rx + ry * ry;
                            hit = d2 < S.dmax2;                                  // R16
                            if (hit && (KIND == kKindDisk || d2 < S.din2)) sure = true;
                        }
                        const unsigned bal = __ballot_sync(0xffffffffu, hit) & gmask;
                        if (hit) U.queue[nq + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)q;
                        nq += __popc(bal);
                    }
                    bool overlap = (__ballot_sync(0xffffffffu, sure) & gmask) != 0u;
                    __syncwarp();
                    // phase B: narrow phase (a9), one queue entry per lane, group vote (early exit of P:45 at group granularity)
                    if (KIND == kKindPolygon) {
                        const int todo = overlap ? 0 : nq;
                        const int most = __reduce_max_sync(0xffffffffu, todo);          // warp-uniform trip count
                        for (int base = 0; base < most; base += G) {
                            const int e = base + lig;
                            bool ov = false;
                            if (e < todo && !overlap) ov = pair_overlap_2d<KIND, NV>(g, S, Tp, U.pose[U.queue[e]], mv.eps_g, seam);
                            const unsigned vote = __ballot_sync(0xffffffffu, ov) & gmask;   // every lane of the warp votes (no short circuit)
                            overlap = overlap || vote != 0u;
                        }
                    }
                    if (outcome == 1 && overlap) outcome = 3;
                    // phase C: accept / write back (a11)
                    if (work && lig == 0) {
                        if (outcome == 1) {
                            float4 Tw = Tp;
                            if (!rotate) {   // R-wrap
                                Tw.x = __fadd_rn(Tw.x, (Tw.x >= g.hi[0]) ? -g.L[0] : (Tw.x < g.lo[0]) ? g.L[0] : 0.0f);
                                Tw.y = __fadd_rn(Tw.y, (Tw.y >= g.hi[1]) ? -g.L[1] : (Tw.y < g.lo[1]) ? g.L[1] : 0.0f);
                                ++cc.tacc;
                            } else {
                                ++cc.racc;
                            }
                            dst_pos[U.gidx[p]] = Tw;
                            U.pose[p] = Tw;
                        } else if (outcome == 2) {
                            ++cc.trcell;
                        } else {
                            if (rotate) ++cc.rrov; else ++cc.trov;
                        }
                        ++cc.trials;
                        if (trace) trace[slot0 + k] = make_uint2((uint32_t)__ldcg(&dst_tag[U.gidx[p]]), (rotate ? 1u : 0u) | ((uint32_t)outcome << 8));
                    }
                    __syncwarp();
                }
            }
            cluster_barrier();   // this colour's write-backs are visible to every CTA before the next colour stages
        }
        cur ^= 1;
    }
    // counters: per-warp reduce, then atomics; the sweep counter advances once for the whole launch
    {
        CellCounters c = cc;
        c.tacc = __reduce_add_sync(0xffffffffu, c.tacc);
        c.trov = __reduce_add_sync(0xffffffffu, c.trov);
        c.trcell = __reduce_add_sync(0xffffffffu, c.trcell);
        c.racc = __reduce_add_sync(0xffffffffu, c.racc);
        c.rrov = __reduce_add_sync(0xffffffffu, c.rrov);
        c.trials = __reduce_add_sync(0xffffffffu, c.trials);
        if (lane == 0 && c.trials) {
            unsigned long long* set = ctrl->counters[(unsigned)(rank * 32 + warp) & (kCounterSets - 1)];
            if (c.tacc) atomicAdd(&set[0], (unsigned long long)c.tacc);
            if (c.trov) atomicAdd(&set[1], (unsigned long long)c.trov);
            if (c.trcell) atomicAdd(&set[2], (unsigned long long)c.trcell);
            if (c.racc) atomicAdd(&set[3], (unsigned long long)c.racc);
            if (c.rrov) atomicAdd(&set[4], (unsigned long long)c.rrov);
            atomicAdd(&set[5], (unsigned long long)c.trials);
        }
    }
    if (gt == 0) {
        ctrl->t = t_first + (unsigned long long)n_sweeps;
        ctrl->sweeps += (unsigned long long)n_sweeps;
    }
}

}  // namespace hpmc
