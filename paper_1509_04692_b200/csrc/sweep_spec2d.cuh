// Colour pass for SMALL 2-D systems with the trials of a cell evaluated SPECULATIVELY (S:8(a) rows a4-a11; BASELINE.json's
// 4096-disk and 4096-pentagon configs).
//
// Such a system is a fraction of one wave of the GPU and a sweep is a chain of 2^d x n_select dependent trials per cell, each a
// few thousand cycles of dependent instructions on one warp (profiles/r2_cluster.md): the pass is bound by that chain, not by
// issue slots.  Trial k+1 of a cell depends on trial k only through its accept/reject bit, and everything else about it -- the
// Philox block, the member it picks, the move -- is known in advance.  So the warp of a cell takes the trials four at a time
// and evaluates the whole decision tree of a batch at once: node (i, h) is trial i proposed from the state that the history
// h of accept bits of trials 0..i-1 would have left (1 + 2 + 4 + 8 = 15 proposals).  One lane per node builds its node's
// state by replaying the accepted trials of h -- the same fp32 operations in the same order as the sequential pass, so the
// poses are bit-identical -- and its proposal; all (node, candidate) pairs then go through ONE broad phase over the lanes and
// ONE dense narrow phase through a ballot-packed queue; finally the warp walks the tree along the bits that really came out
// and keeps the poses of that path.  The chain of a batch is the chain of ONE trial (plus up to three cheap pose replays);
// the extra pairs (15 nodes instead of 4) run on lanes that the sequential pass leaves idle (7 candidates on 32 lanes).
//
// MEASURED, NOT THE DEFAULT (hpmc_set_option("path", 5) selects it).  On B200, 4096 pentagons: one batch of four trials costs
// 4.4 us per colour pass against 4 x 1.05 us for the sequential warp-per-cell pass (slope of us per sweep over n_select = 4, 8,
// 16).  clock64 around the phases of a batch (cycles, 9-11 staged poses): moves 400, replay + proposal 1600, broad phase over
// 135-165 pairs 2500, narrow phase 600 per warp round (1-2 rounds), tree walk + write-back 1100: each phase is a few hundred
// dependent instructions at ~5 cycles each on a warp that shares its scheduler with one other warp, so the tree costs as much
// as the four trials it replaces.  The idea needs every phase to be several times leaner than a sequential trial to pay.
//
// Results are identical to every other colour-pass variant (same Philox keys, make_trial, pair_overlap_2d, same wrap), which
// the lock-step tests check.  Cells with more than kSpecMaxMem members or neighbourhoods above the staging capacity take
// the per-thread path on lane 0.
#pragma once
#include "common.cuh"
#include "overlap.cuh"
#include "sweep.cuh"

namespace hpmc {

constexpr int kSpecWarps = 4;      // warps (= active cells) per CTA
constexpr int kSpecBatch = 4;      // trials per decision tree
constexpr int kSpecNodes = (1 << kSpecBatch) - 1;
constexpr int kSpecMaxMem = 4;     // members of the own cell
constexpr int kSpecCap = 48;       // staged poses (3 x 3 cells)

struct SpecSmem {
    float4 pose[kSpecCap];                       // staged neighbourhood (x, y, qw, qz); the own cell's members are updated per batch
    float4 node[kSpecNodes][kSpecMaxMem];        // members of the own cell in the state of node (i, h)
    float4 trial[kSpecNodes];                    // proposal of the node (unwrapped)
    int gidx[kSpecCap];
    int off[10], start[10];
    unsigned short queue[kSpecNodes * kSpecCap]; // node << 8 | staged index
    float4 delta[kSpecBatch];                    // the moves of the batch: (u_x, u_y, sin, cos of the half angle)
    __align__(16) int meta[kSpecBatch];          // member | rotate << 8
    unsigned ovmask;                             // bit P: the proposal of node P overlaps something
};

// the pose a move proposes from `cur` (a5): the arithmetic of make_trial on the 2-D pose layout, same roundings
__device__ __forceinline__ float4 spec_apply(const MoveParams& mv, const float4& D, int rotate, const float4& cur)
{
    float4 T = cur;
    if (rotate) {
        rotate_2d(cur.z, cur.w, D.z, D.w, T.z, T.w);   // R6
    } else {
        T.x = __fmaf_rn(mv.d, D.x, cur.x);              // R5: one rounding per axis
        T.y = __fmaf_rn(mv.d, D.y, cur.y);
    }
    return T;
}

// what an accepted trial leaves in the state (a11, R-wrap): at most one add per axis
__device__ __forceinline__ float4 spec_wrapped(const GridParams& g, float4 T, int rotate)
{
    if (!rotate) {
        T.x = __fadd_rn(T.x, (T.x >= g.hi[0]) ? -g.L[0] : (T.x < g.lo[0]) ? g.L[0] : 0.0f);
        T.y = __fadd_rn(T.y, (T.y >= g.hi[1]) ? -g.L[1] : (T.y < g.lo[1]) ? g.L[1] : 0.0f);
    }
    return T;
}

template <int KIND, int NV>
__global__ void __launch_bounds__(32 * kSpecWarps)
k_sweep_spec2d(const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv, const __grid_constant__ ShapeF S,
               const __grid_constant__ ShapeD SD, Control* __restrict__ ctrl, int colour_index, int cap_limit,
               float4* __restrict__ pose, const int* __restrict__ tag, const int* __restrict__ cell_start, uint32_t k0, uint32_t k1,
               uint2* __restrict__ trace, int after_colour)
{
    // programmatic dependent launch: the rule of k_sweep_warpcell
    const bool late_wait = after_colour != 0;
    if (!late_wait) pdl_wait();
    pdl_launch_dependents();
    __shared__ SpecSmem sm_all[kSpecWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    SpecSmem& sm = sm_all[warp];

    const SweepHeader& H = ctrl->hdr;
    const int gamma = H.perm[colour_index];
    const uint32_t t_lo = H.t_lo, t_hi16 = H.t_hi16;
    const float shift[3] = {H.shift[0], H.shift[1], 0.0f};
    const int nax = g.n[0] >> 1, nay = g.n[1] >> 1;
    const int idx = blockIdx.x * kSpecWarps + warp;
    if (idx >= nax * nay) return;   // whole warp; nothing below synchronises across warps
    const int ix = idx % nax, iy = idx / nax;
    const int cx = 2 * ix + (gamma & 1), cy = 2 * iy + ((gamma >> 1) & 1);
    const int cell = cx + g.n[0] * cy;
    const long long slot0 = (long long)cell * mv.n_select;
    const bool seam = cx == 0 || cy == 0 || cx >= g.n[0] - 2 || cy >= g.n[1] - 2;   // see k_sweep_warpcell

    // ---- staging: lane j < 9 owns neighbour cell j = (dy+1)*3 + (dx+1) ----------------------------------------------------
    int my_start = 0, my_cnt = 0;
    if (lane < 9) {
        int nx = cx + (lane % 3) - 1, ny = cy + (lane / 3) - 1;
        nx += (nx < 0) ? g.n[0] : 0; nx -= (nx >= g.n[0]) ? g.n[0] : 0;
        ny += (ny < 0) ? g.n[1] : 0; ny -= (ny >= g.n[1]) ? g.n[1] : 0;
        const int c = nx + g.n[0] * ny;
        my_start = cell_start[c];
        my_cnt = cell_start[c + 1] - my_start;
    }
    int incl = my_cnt;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += n;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 8);
    const int own_s = __shfl_sync(0xffffffffu, incl - my_cnt, 4);
    const int nmem = __shfl_sync(0xffffffffu, my_cnt, 4);
    CellCounters cc;
    if (nmem == 0 || layer_inactive(g, cy)) {   // empty, or in the inactive region: no trials
        if (trace && lane == 0)
            for (int k = 0; k < mv.n_select; ++k) trace[slot0 + k] = make_uint2(0u, 0u);
        return;
    }
    if (total > min(cap_limit, kSpecCap) || nmem > kSpecMaxMem) {   // warp-uniform: does not fit the speculative buffers
        if (late_wait) pdl_wait();
        if (lane == 0)
            sweep_cell_global<KIND, NV>(g, mv, S, SD, gamma, t_lo, t_hi16, shift, cx, cy, 0, pose, nullptr, tag, cell_start, k0, k1, trace, cc);
        flush_counters(ctrl, cc);
        return;
    }
    if (lane <= 9) { sm.off[lane] = (lane < 9) ? incl - my_cnt : total; sm.start[lane] = my_start; }
    // a0: the Philox blocks of the first 32 trials, one per lane, in front of the wait
    const uint32_t c3 = (kTagTrial << 24) | ((uint32_t)gamma << 16) | t_hi16;
    U4 blk = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)lane, c3, k0, k1);
    if (late_wait) pdl_wait();   // the previous colour pass is complete: its poses can be staged
    __syncwarp();
    for (int e = lane; e < total; e += 32) {
        int j = 0;   // largest j with off[j] <= e
#pragma unroll
        for (int s = 8; s >= 1; s >>= 1)
            if (j + s < 9 && sm.off[j + s] <= e) j += s;
        const int gi = sm.start[j] + (e - sm.off[j]);
        sm.pose[e] = __ldcg(&pose[gi]);
        sm.gidx[e] = gi;
    }
    __syncwarp();

    // node of this lane: level i (the trial it proposes) and history h (accept bits of trials 0..i-1)
    const int lvl = 31 - __clz(lane + 1), hist = lane + 1 - (1 << lvl);
    const unsigned magic = 0xFFFFFFFFu / (unsigned)total + 1u;   // pair index / total as one multiply (exact for indices < 2^16)

    for (int kb = 0; kb < mv.n_select; kb += kSpecBatch) {
        const int nb = min(kSpecBatch, mv.n_select - kb), nnodes = (1 << nb) - 1;
        if ((kb & 31) == 0 && kb > 0) blk = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)(kb + lane), c3, k0, k1);
        // ---- the moves of the batch, from their Philox blocks alone (R5-R8): the lane that drew trial kb + j derives it ------
        {
            const int j = lane - (kb & 31);
            if (j >= 0 && j < kSpecBatch) {
                const bool rot = (KIND != kKindDisk) && (blk.y >> 31);                        // R7
                float sn = 0.0f, cs = 1.0f;
                if (rot) small_sincos(0.5f * __fmul_rn(mv.a, usym(blk.z)), mv.a, sn, cs);      // R6
                sm.delta[j] = make_float4(usym(blk.z), usym(blk.w), sn, cs);                   // R5: translation words
                sm.meta[j] = (int)mulhi32(blk.x, (uint32_t)nmem) | (rot ? 256 : 0);            // R8: member | rotate << 8
            }
            if (lane == 0) sm.ovmask = 0u;
        }
        __syncwarp();
        const int4 meta = *reinterpret_cast<const int4*>(sm.meta);
        const int metas[kSpecBatch] = {meta.x, meta.y, meta.z, meta.w};
        // ---- phase A: one lane per node -- replay the history, then propose (a5, a6).  The members' poses stay in registers
        // (a dynamic member index is a chain of selects): the replay is a dependent chain, and shared memory would add its latency
        // to every link of it
        bool inside = false;
        if (lane < nnodes) {
            float4 st[kSpecMaxMem];
#pragma unroll
            for (int q = 0; q < kSpecMaxMem; ++q) st[q] = sm.pose[own_s + min(q, nmem - 1)];
#pragma unroll
            for (int j = 0; j < kSpecBatch - 1; ++j) {
                if (j < lvl && ((hist >> j) & 1)) {   // trial j was accepted in this history: it left its wrapped proposal behind
                    const int m = metas[j] & 255, rot = metas[j] >> 8;
                    float4 cur = st[0];
#pragma unroll
                    for (int q = 1; q < kSpecMaxMem; ++q) cur = (m == q) ? st[q] : cur;
                    const float4 nw = spec_wrapped(g, spec_apply(mv, sm.delta[j], rot, cur), rot);
#pragma unroll
                    for (int q = 0; q < kSpecMaxMem; ++q) st[q] = (m == q) ? nw : st[q];
                }
            }
            const int ml = (lvl == 0) ? metas[0] : (lvl == 1) ? metas[1] : (lvl == 2) ? metas[2] : metas[3];
            const int m = ml & 255;
            float4 cur = st[0];
#pragma unroll
            for (int q = 1; q < kSpecMaxMem; ++q) cur = (m == q) ? st[q] : cur;
            const float4 T = spec_apply(mv, sm.delta[lvl], ml >> 8, cur);
            sm.trial[lane] = T;
            if (nmem > 1) {   // the cell mates are candidates of this node, in this node's state
#pragma unroll
                for (int q = 0; q < kSpecMaxMem; ++q)
                    if (q < nmem) sm.node[lane][q] = st[q];
            }
            int tx, ty, tz;
            inside = (ml >> 8) || cell_of(g, shift, T.x, T.y, 0.0f, tx, ty, tz) == cell;   // a6 (R13); rotations never fail it
        }
        const unsigned in_mask = __ballot_sync(0xffffffffu, inside);
        __syncwarp();
        // ---- broad phase (a8) over all (node, candidate) pairs, four warp rounds in flight at a time; survivors to the queue (a10)
        const int npairs = nnodes * total;
        int nq = 0;
        for (int base = 0; base < npairs; base += 128) {
            bool hit[4];
            int ent[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int pi = base + 32 * r + lane;
                hit[r] = false;
                ent[r] = 0;
                if (pi < npairs) {
                    const int P = (int)__umulhi((unsigned)pi, magic);
                    const int e = pi - P * total;
                    const int li = 31 - __clz(P + 1);
                    const int mi = ((li == 0) ? metas[0] : (li == 1) ? metas[1] : (li == 2) ? metas[2] : metas[3]) & 255;
                    ent[r] = (P << 8) | e;
                    if (((in_mask >> P) & 1u) && e != own_s + mi) {
                        const bool own = e >= own_s && e < own_s + nmem;
                        const float4 B = own ? sm.node[P][e - own_s] : sm.pose[e];
                        const float4 T = sm.trial[P];
                        const float rx = seam ? min_image(B.x, T.x, g.hi[0], g.Ld[0]) : B.x - T.x;
                        const float ry = seam ? min_image(B.y, T.y, g.hi[1], g.Ld[1]) : B.y - T.y;
                        const float d2 = rx * rx + ry * ry;
                        hit[r] = d2 < S.dmax2;                                  // R16
                        if (hit[r] && (KIND == kKindDisk || d2 < S.din2)) {     // decided by the centre distance alone
                            atomicOr(&sm.ovmask, 1u << P);
                            hit[r] = false;
                        }
                    }
                }
            }
            if (KIND != kKindDisk) {
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const unsigned bal = __ballot_sync(0xffffffffu, hit[r]);
                    if (hit[r]) sm.queue[nq + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)ent[r];
                    nq += __popc(bal);
                }
            }
        }
        __syncwarp();
        // ---- narrow phase (a9), one queue entry per lane ------------------------------------------------------------------------
        if (KIND != kKindDisk) {
            for (int base = 0; base < nq; base += 32) {
                const int qi = base + lane;
                if (qi < nq) {
                    const int ent = sm.queue[qi], P = ent >> 8, e = ent & 0xff;
                    if (!((*(volatile unsigned*)&sm.ovmask >> P) & 1u)) {
                        const bool own = e >= own_s && e < own_s + nmem;
                        const float4 B = own ? sm.node[P][e - own_s] : sm.pose[e];
                        if (pair_overlap_2d<KIND, NV>(g, S, sm.trial[P], B, mv.eps_g, seam)) atomicOr(&sm.ovmask, 1u << P);
                    }
                }
                __syncwarp();
            }
        }
        const unsigned ov_mask = *(volatile unsigned*)&sm.ovmask;
        // ---- walk the tree along the bits that came out; accept / write back (a11) ------------------------------------------------
        int h = 0;
        int last_node = -1;      // lane m < nmem: node of the last accepted trial that moved member m
        bool last_rot = false;
#pragma unroll
        for (int i = 0; i < kSpecBatch; ++i) {
            if (i < nb) {
                const int P = (1 << i) - 1 + h;
                const bool rot = (metas[i] >> 8) != 0;
                const int outcome = !((in_mask >> P) & 1u) ? 2 : ((ov_mask >> P) & 1u) ? 3 : 1;
                if (outcome == 1) {
                    h |= 1 << i;
                    if ((metas[i] & 255) == lane) { last_node = P; last_rot = rot; }
                }
                if (lane == 0) {
                    ++cc.trials;
                    cc.tacc += (outcome == 1 && !rot) ? 1u : 0u;
                    cc.racc += (outcome == 1 && rot) ? 1u : 0u;
                    cc.trcell += (outcome == 2) ? 1u : 0u;
                    cc.trov += (outcome == 3 && !rot) ? 1u : 0u;
                    cc.rrov += (outcome == 3 && rot) ? 1u : 0u;
                    if (trace) trace[slot0 + kb + i] = make_uint2((uint32_t)tag[sm.gidx[own_s + (metas[i] & 255)]], (rot ? 1u : 0u) | ((uint32_t)outcome << 8));
                }
            }
        }
        if (lane < nmem && last_node >= 0) {
            const float4 T = spec_wrapped(g, sm.trial[last_node], last_rot);
            pose[sm.gidx[own_s + lane]] = T;
            sm.pose[own_s + lane] = T;
        }
        __syncwarp();
    }
    flush_counters(ctrl, cc);
}

}  // namespace hpmc
