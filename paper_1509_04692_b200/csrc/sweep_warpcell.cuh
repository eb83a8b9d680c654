// Colour pass, warp-per-cell version (S:8(a) rows a4-a11) -- the paper's block-level work queue at warp
// scope.  Used for every 3-D system (spheres, convex polyhedra) and for 2-D systems too small to fill the GPU with one
// lane per cell (config 1: 961 active cells per colour are 31 warps of the tile kernel but 961 warps here, and the serial
// chain of a trial shrinks from a 32-cell warp round to one cell's work).
//
// One warp = one active cell of the current colour.  The warp first stages the particles of the 3^d cells around
// its cell (a7, "neighbour gather staged in shared memory") and then makes the cell's n_select trials one after
// the other (R9):
//
//   A  every lane evaluates the same Philox block and builds the same trial pose (uniform, no divergence), then
//      the lanes stride over the staged candidates for the circumsphere broad phase (a8: "100 particles in
//      the cells around ... only five pass") and append the survivors to a per-warp queue with ballot/popc;
//   B  the queue is drained one entry per lane: polygon separating axes, or fp32 GJK on the Minkowski difference (a9,
//      Eq. (1)-(2)) where lanes whose fp32 verdict is "unsure" (near contact) re-run their pair in fp64; one vote
//      (__any_sync) gives the trial's fate -- the early exit of P:45 at warp granularity;
//   C  lane 0 writes an accepted pose to the staged copy (so trial k+1 sees it) and to global memory (a11).
//
// Cells of one colour never read what another cell of that colour writes, so warps never synchronise
// with each other.  A neighbourhood with more particles than the staging capacity is handled by lane 0 on the
// per-thread global-memory path (sweep_cell_global); results are identical.
#pragma once
#include "common.cuh"
#include "overlap.cuh"
#include "sweep.cuh"

namespace hpmc {

constexpr int kW3Cap = 192;     // staged particles per warp (own cell + 26 neighbours; cubes at phi=0.51: ~83)
constexpr int kW3Warps = 4;     // warps (= active cells) per CTA

struct Warp3dSmem {
    float4 pos[kW3Cap];
    float4 quat[kW3Cap];
    int gidx[kW3Cap];
    int queue[kW3Cap];
    int off[28];
    int start[28];
};

// G: lanes per narrow-phase pair of the polyhedron pass (1 or 2, see support_mpr)
template <int KIND, int NV, int DIM, int G>
__device__ __forceinline__ void warpcell_body(const GridParams& g, const MoveParams& mv, const ShapeF& S, const ShapeD& SD,
                                              Control* __restrict__ ctrl, int colour_index, int cap_limit, float4* __restrict__ pos,
                                              float4* __restrict__ quat, const int* __restrict__ tag, const int* __restrict__ cell_start,
                                              uint32_t k0, uint32_t k1, uint2* __restrict__ trace, int after_colour)
{
    // Programmatic dependent launch (common.cuh).  A colour pass that follows the cell-list build (or anything else): nothing can be
    // read before that has completed, and only then may the next pass be launched.  A later pass starts while the pass
    // before it still runs (which itself started only after the build was complete): header, cell offsets, Philox blocks and
    // the empty-cell exits do not depend on that pass; the poses do, so the wait sits in front of the staging loads.
    // after_colour: the launch before this one in the stream was a colour pass of the same sweep (set by the host)
    const bool late_wait = after_colour != 0;
    if (!late_wait) pdl_wait();
    pdl_launch_dependents();
    __shared__ Warp3dSmem sm_all[kW3Warps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Warp3dSmem& sm = sm_all[warp];

    const SweepHeader& H = ctrl->hdr;
    const int gamma = H.perm[colour_index];
    const uint32_t t_lo = H.t_lo, t_hi16 = H.t_hi16;
    const float shift[3] = {H.shift[0], H.shift[1], DIM == 3 ? H.shift[2] : 0.0f};
    constexpr int NNB = (DIM == 3) ? 27 : 9, OWN = (DIM == 3) ? 13 : 4;   // cells of the 3^d block; index of the own cell
    const int nax = g.n[0] >> 1, nay = g.n[1] >> 1, naz = (DIM == 3) ? (g.n[2] >> 1) : 1;
    const int idx = blockIdx.x * kW3Warps + warp;
    if (idx >= nax * nay * naz) return;   // whole warp; nothing below synchronises across warps
    const int ix = idx % nax, iy = (idx / nax) % nay, iz = idx / (nax * nay);
    const int cx = 2 * ix + (gamma & 1), cy = 2 * iy + ((gamma >> 1) & 1), cz = (DIM == 3) ? 2 * iz + ((gamma >> 2) & 1) : 0;
    const int cell = cx + g.n[0] * (cy + g.n[1] * cz);
    const long long slot0 = (long long)cell * mv.n_select;
    // With the grid shifted by s in [0,w), the box edge lies inside cell n-1, so cell n-1 holds coordinates near both
    // +L/2 and -L/2.  Only cells 0, n-2 and n-1 can therefore see a neighbour across the periodic seam; only there is
    // the precise min_image needed (R21); elsewhere |x_j - x_t| < 2w <= L/2 and the plain fp32 difference is the same value.
    const bool seam = cx == 0 || cy == 0 || cx >= g.n[0] - 2 || cy >= g.n[1] - 2 || (DIM == 3 && (cz == 0 || cz >= g.n[2] - 2));

    // ---- staging: lane j < 3^d owns neighbour cell j = (dz+1)*9 + (dy+1)*3 + (dx+1) --------------------------------
    int my_start = 0, my_cnt = 0;
    if (lane < NNB) {
        int nx = cx + (lane % 3) - 1, ny = cy + ((lane / 3) % 3) - 1, nz = (DIM == 3) ? cz + (lane / 9) - 1 : 0;
        nx += (nx < 0) ? g.n[0] : 0; nx -= (nx >= g.n[0]) ? g.n[0] : 0;
        ny += (ny < 0) ? g.n[1] : 0; ny -= (ny >= g.n[1]) ? g.n[1] : 0;
        if (DIM == 3) { nz += (nz < 0) ? g.n[2] : 0; nz -= (nz >= g.n[2]) ? g.n[2] : 0; }
        const int c = nx + g.n[0] * (ny + g.n[1] * nz);
        my_start = cell_start[c];
        my_cnt = cell_start[c + 1] - my_start;
    }
    int incl = my_cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += n;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    const int own_s = __shfl_sync(0xffffffffu, incl - my_cnt, OWN);
    const int nmem = __shfl_sync(0xffffffffu, my_cnt, OWN);
    CellCounters cc;
    if (nmem == 0 || layer_inactive(g, DIM == 3 ? cz : cy)) {   // empty, or in the inactive region: no trials
        if (trace && lane == 0)
            for (int k = 0; k < mv.n_select; ++k) trace[slot0 + k] = make_uint2(0u, 0u);
        return;
    }
    if (total > min(cap_limit, kW3Cap)) {   // warp-uniform: neighbourhood does not fit the staging buffers
        if (late_wait) pdl_wait();
        if (lane == 0)
            sweep_cell_global<KIND, NV>(g, mv, S, SD, gamma, t_lo, t_hi16, shift, cx, cy, cz, pos, quat, tag, cell_start, k0, k1, trace, cc);
        flush_counters(ctrl, cc);
        return;
    }
    if (lane <= NNB) { sm.off[lane] = incl - my_cnt; sm.start[lane] = my_start; }   // lane 3^d: off = total
    // a0: the Philox blocks of the first 32 trials, one trial per lane, off the critical path of the sequential trials (a trial
    // is a chain of dependent instructions; ten Philox rounds are a quarter of it) -- and in front of the wait
    const uint32_t c3 = (kTagTrial << 24) | ((uint32_t)gamma << 16) | t_hi16;
    U4 blk = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)lane, c3, k0, k1);
    uint32_t blk_uc = 0u;
    if (DIM == 3) blk_uc = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)lane | (1u << 16), c3, k0, k1).x;
    if (late_wait) pdl_wait();   // the previous colour pass is complete: its poses can be staged
    __syncwarp();
    for (int e = lane; e < total; e += 32) {
        int j = 0;   // largest j with off[j] <= e (off is non-decreasing, off[3^d] = total > e)
#pragma unroll
        for (int s = 16; s >= 1; s >>= 1)
            if (j + s < NNB && sm.off[j + s] <= e) j += s;
        const int gi = sm.start[j] + (e - sm.off[j]);
        float4 x4, q4;
        load_state(DIM, pos, quat, gi, x4, q4);
        sm.pos[e] = x4;
        sm.quat[e] = q4;
        sm.gidx[e] = gi;
    }
    __syncwarp();

    for (int k = 0; k < mv.n_select; ++k) {
        // ---- a0: the blocks of the next 32 trials (the first batch was drawn above); trial k broadcasts its block
        if ((k & 31) == 0 && k > 0) {
            blk = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)(k + lane), c3, k0, k1);
            if (DIM == 3) blk_uc = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)(k + lane) | (1u << 16), c3, k0, k1).x;
        }
        const U4 b0{__shfl_sync(0xffffffffu, blk.x, k & 31), __shfl_sync(0xffffffffu, blk.y, k & 31), __shfl_sync(0xffffffffu, blk.z, k & 31),
                    __shfl_sync(0xffffffffu, blk.w, k & 31)};
        const uint32_t uc = (DIM == 3) ? __shfl_sync(0xffffffffu, blk_uc, k & 31) : 0u;
        // ---- phase A: trial pose (a5, a6), identical on every lane ------------------------------------------------------
        const int p = own_s + (int)mulhi32(b0.x, (uint32_t)nmem);   // R8
        const float4 xp = sm.pos[p], qp = sm.quat[p];
        TrialState A;
        bool rotate;
        int outcome = make_trial<KIND>(g, mv, shift, cell, DIM, b0, uc, xp, qp, A, rotate) ? 1 : 2;
        if (lane == 0) ++cc.trials;
        if (outcome == 1) {
            float MA[9];
            if (KIND == kKindPolyhedron) quat_to_matrix<float>(A.qw, A.qx, A.qy, A.qz, MA);
            // ---- broad phase (a8): lanes stride over the staged candidates, survivors go to the queue (a10) --------
            int nq = 0;
            bool sure = false;   // a centre inside the inscribed-sphere bound (or, for spheres, inside the diameter)
            for (int base = 0; base < total; base += 32) {
                const int q = base + lane;
                bool hit = false;
                if (q < total && q != p) {
                    const float4 xq = sm.pos[q];
                    const float rx = seam ? min_image(xq.x, A.x, g.hi[0], g.Ld[0]) : xq.x - A.x;
                    const float ry = seam ? min_image(xq.y, A.y, g.hi[1], g.Ld[1]) : xq.y - A.y;
                    const float rz = (DIM == 3) ? (seam ? min_image(xq.z, A.z, g.hi[2], g.Ld[2]) : xq.z - A.z) : 0.0f;
                    const float d2 = rx * rx + ry * ry + rz * rz;
                    hit = d2 < S.dmax2;                                  // R16
                    if (hit && (KIND == kKindDisk || d2 < S.din2)) sure = true;
                }
                const unsigned bal = __ballot_sync(0xffffffffu, hit);
                if (hit) sm.queue[nq + __popc(bal & ((1u << lane) - 1u))] = q;
                nq += __popc(bal);
            }
            bool overlap = __any_sync(0xffffffffu, sure);
            __syncwarp();
            // ---- phase B: narrow phase (a9), one queue entry per lane ----------------------------------------------
            if (KIND == kKindPolygon) {
                const float4 T = make_float4(A.x, A.y, A.qw, A.qz);
                for (int base = 0; base < nq && !overlap; base += 32) {
                    const int e = base + lane;
                    bool ov = false;
                    if (e < nq) {
                        const int q = sm.queue[e];
                        const float4 xq = sm.pos[q], qq = sm.quat[q];
                        ov = pair_overlap_2d<KIND, NV>(g, S, T, make_float4(xq.x, xq.y, qq.x, qq.w), mv.eps_g, seam);
                    }
                    overlap = __any_sync(0xffffffffu, ov);
                }
            }
            if (KIND == kKindPolyhedron) {
                // G = 2: two lanes per queue entry (support_mpr), the support scans of a XenoCollide iteration split into their A
                // half and their B half
                const int sub = lane & (G - 1);
                const unsigned pair_mask = ((1u << G) - 1u) << (lane & ~(G - 1));
                for (int base = 0; base < nq && !overlap; base += 32 / G) {
                    const int e = base + lane / G;
                    bool ov = false;
                    if (e < nq) {
                        const int q = sm.queue[e];
                        const float4 xq = sm.pos[q], qq = sm.quat[q];
                        const float rx = seam ? min_image(xq.x, A.x, g.hi[0], g.Ld[0]) : xq.x - A.x;
                        const float ry = seam ? min_image(xq.y, A.y, g.hi[1], g.Ld[1]) : xq.y - A.y;
                        const float rz = seam ? min_image(xq.z, A.z, g.hi[2], g.Ld[2]) : xq.z - A.z;
                        float MB[9];
                        quat_to_matrix<float>(qq.x, qq.y, qq.z, qq.w, MB);
                        int portal[3];
                        const int verdict = polyhedron_classify<float, NV, G>(S, MA, MB, V3<float>{rx, ry, rz}, mv.eps_g, kGjkDeepF, portal, sub, pair_mask);
                        if (verdict == kGjkUnsure) {   // near contact: decide in fp64 from the raw fp32 state
                            if (sub == 0) ++cc.f64;
                            ov = polyhedron_overlap_f64<(NV == 8) ? 8 : 0>(SD, make_float4(A.qw, A.qx, A.qy, A.qz), qq, min_image_d(xq.x, A.x, g.Ld[0]),
                                                            min_image_d(xq.y, A.y, g.Ld[1]), min_image_d(xq.z, A.z, g.Ld[2]), (double)mv.eps_g, portal);
                        } else
                            ov = verdict == kGjkOverlap;
                    }
                    overlap = __any_sync(0xffffffffu, ov);
                }
            }
            if (overlap) outcome = 3;
        }
        // ---- phase C: accept / write back (a11) -----------------------------------------------------------------------
        if (lane == 0) {
            if (outcome == 1) {
                const int gi = sm.gidx[p];
                float x = A.x, y = A.y, z = A.z;
                if (!rotate) {   // R-wrap
                    if (x >= g.hi[0]) x = __fsub_rn(x, g.L[0]); else if (x < g.lo[0]) x = __fadd_rn(x, g.L[0]);
                    if (y >= g.hi[1]) y = __fsub_rn(y, g.L[1]); else if (y < g.lo[1]) y = __fadd_rn(y, g.L[1]);
                    if (DIM == 3) { if (z >= g.hi[2]) z = __fsub_rn(z, g.L[2]); else if (z < g.lo[2]) z = __fadd_rn(z, g.L[2]); }
                    ++cc.tacc;
                } else {
                    ++cc.racc;
                }
                const float4 nx4 = make_float4(x, y, z, xp.w), nq4 = make_float4(A.qw, A.qx, A.qy, A.qz);
                store_state(DIM, pos, quat, gi, nx4, nq4, rotate);
                sm.pos[p] = nx4;
                sm.quat[p] = nq4;
            } else if (outcome == 2) {
                ++cc.trcell;
            } else {
                if (rotate) ++cc.rrov; else ++cc.trov;
            }
            if (trace) trace[slot0 + k] = make_uint2((uint32_t)tag[sm.gidx[p]], (rotate ? 1u : 0u) | ((uint32_t)outcome << 8));
        }
        __syncwarp();
    }
    flush_counters(ctrl, cc);
}

#define HPMC_WARPCELL_PARAMS                                                                                                        \
    const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv, const __grid_constant__ ShapeF S,                  \
        const __grid_constant__ ShapeD SD, Control *__restrict__ ctrl, int colour_index, int cap_limit, float4 *__restrict__ pos,   \
        float4 *__restrict__ quat, const int *__restrict__ tag, const int *__restrict__ cell_start, uint32_t k0, uint32_t k1,       \
        uint2 *__restrict__ trace, int after_colour

// The pass as the compiler sizes it (polyhedra: 168 registers, 12 warps per SM): a system of up to a wave or two of active
// cells is a latency chain per warp, and fewer registers would put spills on that chain (config 3: -14 % at 128 registers).
// One lane per pair for the unrolled 8-vertex shape (config 3: two lanes are 1 % slower, the pair shuffle inside the divergent
// loop costs what the halved scan saves), two for the other counts (20, 24 vertices: the scans are most of an iteration).
template <int KIND, int NV, int DIM>
__global__ void __launch_bounds__(32 * kW3Warps) k_sweep_warpcell(HPMC_WARPCELL_PARAMS)
{
    warpcell_body<KIND, NV, DIM, (NV == 8) ? 1 : 2>(g, mv, S, SD, ctrl, colour_index, cap_limit, pos, quat, tag, cell_start, k0, k1, trace, after_colour);
}

// The same pass held to 96 registers (20 warps per SM) for systems with many waves of active cells, where the pass is bound by
// instruction issue and the extra warps fill the slots a dependent chain leaves empty: 96^3 cubes 3.18e8 -> 3.77e8 trial
// moves/s, 131 072 dodecahedra (the paper's per-GPU size) 1.51e8 -> 1.69e8, and with two lanes per pair (instruction
// count is what binds here) 3.86e8 and 1.93e8.  Same arithmetic, same results.
template <int KIND, int NV, int DIM>
__global__ void __launch_bounds__(32 * kW3Warps, 5) k_sweep_warpcell_occ(HPMC_WARPCELL_PARAMS)
{
    warpcell_body<KIND, NV, DIM, 2>(g, mv, S, SD, ctrl, colour_index, cap_limit, pos, quat, tag, cell_start, k0, k1, trace, after_colour);
}
#undef HPMC_WARPCELL_PARAMS

}  // namespace hpmc
