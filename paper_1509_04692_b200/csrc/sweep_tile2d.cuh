// 2-D colour pass, tile version v3 (S:8(a) rows a4-a11).
//
// One CTA = a tile of 32 x (WARPS*R) active cells of the current colour.  The CTA stages every pose of the
// (2*32+1) x (2*WARPS*R+1) cell region around its tile into shared memory (a7: "neighbour gather staged in shared
// memory").  Cells of a row are contiguous in the cell-sorted pose array, so a region row is one contiguous run
// (two at the periodic wrap): 2*RH segment copies, fully coalesced, and a local CSR of 16-bit offsets.
//
// After the staging barrier the warps are independent (active cells of one colour never read each other's writes,
// P:21).  A warp owns R rows of 32 active cells.  It first compacts its NON-EMPTY cells (ballot/popc) so that
// every lane of every round has work, then for each of the n_select trial rounds:
//
//   A  each lane takes up to R cells in turn: Philox block -> member, move type, trial pose (a0, a5), leave-cell test
//      with the pinned cell function (a6), circumsphere broad phase over the three staged row runs of the cell's 3x3
//      block (a8); centres inside the inscribed-disk bound reject on the spot; the remaining hits are appended to the
//      warp's queue in shared memory (a10) as (owner slot, neighbour).
//   B  the queue (~60 R entries) is drained densely, one entry per lane: branch-free separating-axis test (a9); an
//      overlap sets the owner's flag.  This is the paper's block queue at warp scope: lanes do not idle
//      while one neighbour of one trial is in its narrow phase, and R cells per lane keep the last
//      32-entry batch from running nearly empty.
//   C  owners read their flag; accepted poses go to the staged copy (trial k+1 of the cell sees them) and to global
//      memory (a11).
//
// Only tiles whose region touches the periodic seam use the fp64 minimum image (R21): elsewhere every compared pair is
// closer than 2w <= L/2 and the plain fp32 difference is the same number.  A tile whose region holds more particles
// than the staging capacity falls back to the per-thread global path (sweep_cell_global); results are identical.
#pragma once
#include "common.cuh"
#include "overlap.cuh"
#include "sweep.cuh"

namespace hpmc {

constexpr int kTileW = 32;   // active cells per tile row = lanes of a warp
constexpr int kRowSlots = 5; // predicated broad-phase slots per row run of 3 cells (a run holds more in ~0.1 % of the cases)

template <int WARPS, int R>
struct Tile2D {
    static constexpr int NT = 32 * WARPS;
    static constexpr int TH = WARPS * R;                 // active rows per tile
    static constexpr int RW = 2 * kTileW + 1;            // staged cells per region row
    static constexpr int RH = 2 * TH + 1;                // staged region rows
    static constexpr int NCELLS = RW * RH;
    static constexpr int CAP = (NCELLS * 5 / 4 + 63) / 64 * 64;   // staged poses (pentagon fluid: ~1.0 per cell)
    static constexpr int NSEG = 2 * RH;                  // contiguous runs: two per region row (periodic wrap in x)
    static constexpr int QCAP = 32 * R * 3 * kRowSlots;  // narrow-phase queue entries per warp and trial round: every slot of every lane fits
    static constexpr int SLOTS = 32 * R;                 // trial slots per warp and round
    static_assert(NSEG + 1 <= NT, "one thread per segment");
    static_assert(CAP < 65536, "16-bit local offsets");
    // shared-memory carve (bytes)
    static constexpr size_t off_pose = 0;
    static constexpr size_t off_trial = off_pose + sizeof(float4) * (CAP + 8);   // + 8: the predicated candidate slots may read past the end
    static constexpr size_t off_queue = off_trial + sizeof(float4) * SLOTS * WARPS;
    static constexpr size_t off_seg_g = off_queue + sizeof(unsigned) * QCAP * WARPS;
    static constexpr size_t off_seg_l = off_seg_g + sizeof(int) * NSEG;
    static constexpr size_t off_qcount = off_seg_l + sizeof(int) * (NSEG + 1);
    static constexpr size_t off_lstart = off_qcount + sizeof(int) * WARPS;
    static constexpr size_t off_flag = off_lstart + ((sizeof(unsigned short) * (NCELLS + 1) + 15) / 16) * 16;
    static constexpr size_t off_act = off_flag + SLOTS * WARPS;
    static constexpr size_t bytes = off_act + SLOTS * WARPS;
};

// a10: one predicated shared-memory store per candidate slot B .. 3 kRowSlots - 1 of the hit mask `pm`; `qaddr` (shared-memory
// byte address of the lane's next queue entry) advances by one entry per hit.  Four instructions per slot, no branch.
template <int B>
__device__ __forceinline__ void push_bits(unsigned& qaddr, unsigned pm, const unsigned (&base)[3])
{
    if constexpr (B < 3 * kRowSlots) {
        asm volatile("{\n\t.reg .pred q;\n\t.reg .b32 t;\n\tand.b32 t, %1, %2;\n\tsetp.ne.u32 q, t, 0;\n\t"
                     "@q st.shared.u32 [%0], %3;\n\t@q add.u32 %0, %0, 4;\n\t}"
                     : "+r"(qaddr) : "r"(pm), "n"(1u << B), "r"(base[B / kRowSlots] + (unsigned)(B % kRowSlots)) : "memory");
        push_bits<B + 1>(qaddr, pm, base);
    }
}

// out of line so that the colour pass without a trace pays one uniform branch, not a dozen predicated instructions
static __device__ __noinline__ void trace_store(uint2* __restrict__ trace, const int* __restrict__ tag, int gi, long long at, bool rotate, unsigned outcome)
{
    trace[at] = make_uint2((uint32_t)tag[gi], (rotate ? 1u : 0u) | (outcome << 8));
}

// out-of-line copy for the rare direct evaluations (queue overflow, > 32 candidates): keeps the hot loop's code small
template <int KIND, int NV>
__device__ __noinline__ bool pair_overlap_2d_cold(const GridParams& g, const ShapeF& S, float4 A, float4 B, float eps)
{
    return pair_overlap_2d<KIND, NV>(g, S, A, B, eps, true);
}

// a8, common path: kRowSlots fixed candidate slots per row run of the 3x3 block (bit kRowSlots*dy + j), no data-dependent
// loop.  A slot past the end of its run holds a pose of a cell farther along (or the sentinel padding behind the last staged
// pose): any pose within d_max of a trial that stayed in its cell lies in the 3x3 block (w >= d_max (1 + 2^-10), R11), so such
// a slot can only repeat a genuine neighbour (tiny periodic grids) or the particle itself and needs no length predicate; the
// particle's own slots are cleared from both masks after the loop.
//   mask : centres inside the circumsphere range (R16')          sure : some centre inside the inscribed-disk bound
template <int KIND, bool SEAM>
__device__ __forceinline__ void broad_slots(const GridParams& g, const ShapeF& S, const float2* sm_xy, const int (&rs)[3], int p,
                                            const float4& T, unsigned& mask, bool& sure)
{
    // The two comparisons of a slot as sign bits: d2 < c  <=>  d2 - c < 0 (the difference of two distinct floats is never -0, and
    // x - x is +0), shifted into the masks with one funnel shift each -- an FADD (fma pipe) and an SHF instead of a compare and a
    // predicated OR, both on the half-rate alu pipe, which this pass keeps busier than the fma pipe (profiles/r2_final.md).
    // Slots run from the last to the first so that slot (dy, j) ends on bit kRowSlots dy + j.
    unsigned smask = 0u;
    mask = 0u;
#pragma unroll
    for (int dy = 2; dy >= 0; --dy) {
#pragma unroll
        for (int j = kRowSlots - 1; j >= 0; --j) {
            const float2 B = sm_xy[rs[dy] + j];
            float rx = B.x - T.x, ry = B.y - T.y;
            if (SEAM) {
                rx = min_image(B.x, T.x, g.hi[0], g.Ld[0]);
                ry = min_image(B.y, T.y, g.hi[1], g.Ld[1]);
            }
            const float d2 = rx * rx + ry * ry;
            mask = __funnelshift_l(__float_as_uint(__fsub_rn(d2, S.dmax2)), mask, 1);                               // R16
            if (KIND != kKindDisk) smask = __funnelshift_l(__float_as_uint(__fsub_rn(d2, S.din2)), smask, 1);
        }
    }
    // the particle itself: slot p - rs[1] of the middle run, and -- when the cells between are empty, so that the slots of
    // the first run reach into the next staged row -- slot p - rs[0] of the first run (the last run starts behind p)
    const unsigned j0 = (unsigned)(p - rs[0]), j1 = (unsigned)(p - rs[1]);
    const unsigned keep = ~(((j1 < (unsigned)kRowSlots) ? (1u << (kRowSlots + j1)) : 0u) | ((j0 < (unsigned)kRowSlots) ? (1u << j0) : 0u));
    mask &= keep;
    sure = ((KIND == kKindDisk) ? mask : (smask & keep)) != 0u;                          // disks: any hit is an overlap
}

// The work of one tile of colour gamma (see the header of this file).  FLOW: the caller is the persistent dataflow kernel,
// where other CTAs of the same launch wrote some of the poses read here: stage them with L2-coherent loads.
template <int KIND, int NV, int WARPS, int R, bool FLOW>
__device__ __forceinline__ void tile2d_body(const GridParams& g, const MoveParams& mv, const ShapeF& S, const ShapeD& SD,
                                            Control* __restrict__ ctrl, int gamma, int tile, int cap_limit, float4* __restrict__ pose,
                                            const int* __restrict__ tag, const int* __restrict__ cell_start, uint32_t k0, uint32_t k1,
                                            uint2* __restrict__ trace, unsigned char* smem_raw, bool late_wait = false)
{
    using TL = Tile2D<WARPS, R>;
    // staged poses, positions and orientations apart: the broad phase reads only (x, y), and 8-byte elements halve the
    // shared-memory bank conflicts of its per-lane gathers (lane stride ~2 poses) against one 16-byte array
    float2* sm_xy = reinterpret_cast<float2*>(smem_raw + TL::off_pose);                          // (x, y)
    float2* sm_qq = reinterpret_cast<float2*>(smem_raw + TL::off_pose) + (TL::CAP + 8);          // (qw, qz)
    auto ld_pose = [&](int q) { const float2 a = sm_xy[q], b = sm_qq[q]; return make_float4(a.x, a.y, b.x, b.y); };
    auto st_pose = [&](int q, const float4& v) { sm_xy[q] = make_float2(v.x, v.y); sm_qq[q] = make_float2(v.z, v.w); };
    float4* sm_trial = reinterpret_cast<float4*>(smem_raw + TL::off_trial);     // trial pose of every slot
    unsigned* sm_queue = reinterpret_cast<unsigned*>(smem_raw + TL::off_queue);
    int* sm_seg_g = reinterpret_cast<int*>(smem_raw + TL::off_seg_g);           // global start of each segment
    int* sm_seg_l = reinterpret_cast<int*>(smem_raw + TL::off_seg_l);           // local start of each segment (+ total)
    unsigned short* sm_lstart = reinterpret_cast<unsigned short*>(smem_raw + TL::off_lstart);   // local CSR over region cells
    unsigned char* sm_flag = smem_raw + TL::off_flag;
    unsigned char* sm_act = smem_raw + TL::off_act;

    const SweepHeader& H = ctrl->hdr;
    const uint32_t t_lo = H.t_lo, t_hi16 = H.t_hi16;
    const float shift[3] = {H.shift[0], H.shift[1], 0.0f};
    const int gx = gamma & 1, gy = (gamma >> 1) & 1;
    const int n0 = g.n[0], n1 = g.n[1];
    const int nax = n0 >> 1, nay = n1 >> 1;
    const int tiles_x = (nax + kTileW - 1) / kTileW;
    const int tx = tile % tiles_x, ty = tile / tiles_x;
    const int ix0 = tx * kTileW, iy0 = ty * TL::TH;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // region = cells [cx0-1, cx0-1+RW) x [cy0-1, cy0-1+RHv) (unwrapped), clipped to what the valid active cells need
    const int cx0 = 2 * ix0 + gx, cy0 = 2 * iy0 + gy;
    const int RW = 2 * min(kTileW, nax - ix0) + 1, RHv = 2 * min(TL::TH, nay - iy0) + 1;
    const int ncells = RW * RHv;
    int xs = cx0 - 1;                       // first region column, wrapped
    xs += (xs < 0) ? n0 : 0;
    const int split = min(RW, n0 - xs);     // columns before the periodic wrap in x
    // the region touches the seam iff it contains cell n-1 (which holds coordinates near both box edges) or wraps
    const bool seam = (cx0 - 1 < 0) || (cx0 - 1 + RW - 1 >= n0 - 1) || (cy0 - 1 < 0) || (cy0 - 1 + RHv - 1 >= n1 - 1);

    // ---- staging 1: the contiguous runs of the region rows -------------------------------------------------------
    // global start and length of segment i (two per region row: before and after the periodic wrap in x)
    auto segment = [&](int i, int& gb, int& len) {
        const int ry = i >> 1, second = i & 1;
        gb = 0; len = 0;
        if (i < TL::NSEG && ry < RHv) {
            int cy = cy0 - 1 + ry;
            cy += (cy < 0) ? n1 : 0;
            cy -= (cy >= n1) ? n1 : 0;
            const int first = second ? 0 : xs, ncol = second ? RW - split : split;
            if (ncol > 0) {
                gb = cell_start[cy * n0 + first];
                len = cell_start[cy * n0 + first + ncol] - gb;
            }
        }
    };
    int ntot;
    if constexpr (TL::NSEG <= 32) {
        // every warp works out all segments for itself (lane i: segment i; exclusive scan by shuffles) and writes the same
        // values to shared memory: no block barrier and no idle warps before the poses can be staged
        int gb, len;
        segment(lane, gb, len);
        int inc = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int n = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += n;
        }
        ntot = __shfl_sync(0xffffffffu, inc, 31);
        if (lane < TL::NSEG) { sm_seg_g[lane] = gb; sm_seg_l[lane] = inc - len; }
        if (lane == 0) sm_seg_l[TL::NSEG] = ntot;
        __syncwarp();
    } else {
        if (tid < TL::NSEG) {
            int gb, len;
            segment(tid, gb, len);
            sm_seg_g[tid] = gb;
            sm_seg_l[tid] = len;
        }
        __syncthreads();
        if (warp == 0) {   // exclusive scan of the segment lengths
            int carry = 0;
#pragma unroll
            for (int b = 0; b < (TL::NSEG + 31) / 32; ++b) {
                const int i = b * 32 + lane;
                const int v = (i < TL::NSEG) ? sm_seg_l[i] : 0;
                int inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int n = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += n;
                }
                __syncwarp();
                if (i < TL::NSEG) sm_seg_l[i] = carry + inc - v;
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) sm_seg_l[TL::NSEG] = carry;
        }
        __syncthreads();
        ntot = sm_seg_l[TL::NSEG];
    }
    const bool staged = ntot <= min(cap_limit, TL::CAP);   // block-uniform
    CellCounters cc;
    if (late_wait) pdl_wait();   // the segment table came from the cell list alone; the poses need the previous colour pass complete

    if (!staged) {
        // overflow: more particles around this tile than the staging buffers hold -> per-thread global path
#pragma unroll 1
        for (int j = 0; j < R; ++j) {
            const int ay = warp * R + j;
            if (ix0 + lane < nax && iy0 + ay < nay)
                sweep_cell_global<KIND, NV>(g, mv, S, SD, gamma, t_lo, t_hi16, shift, cx0 + 2 * lane, cy0 + 2 * ay, 0, pose, nullptr, tag,
                                            cell_start, k0, k1, trace, cc);
        }
        flush_counters(ctrl, cc);
        return;
    }

    // ---- staging 2: local CSR (16-bit) and the poses, coalesced ---------------------------------------------------
    for (int ry = warp; ry < RHv; ry += WARPS) {   // one region row per warp at a time: no index division, coalesced
        int cy = cy0 - 1 + ry;
        cy += (cy < 0) ? n1 : 0;
        cy -= (cy >= n1) ? n1 : 0;
        const int* row_start = cell_start + cy * n0;
        const int g0 = sm_seg_g[2 * ry], g1 = sm_seg_g[2 * ry + 1];
        const int l0 = sm_seg_l[2 * ry], l1 = sm_seg_l[2 * ry + 1], l2 = sm_seg_l[2 * ry + 2];
        if (split == RW) {   // block-uniform: the row does not wrap in x (every tile but those on the box edge): one segment
            const int delta = l0 - g0;
            for (int rx = lane; rx < RW; rx += 32) sm_lstart[ry * RW + rx] = (unsigned short)(row_start[xs + rx] + delta);
        } else {
            for (int rx = lane; rx < RW; rx += 32) {
                const bool second = rx >= split;
                const int cx = second ? rx - split : xs + rx;
                sm_lstart[ry * RW + rx] = (unsigned short)(row_start[cx] - (second ? g1 : g0) + (second ? l1 : l0));
            }
        }
        for (int e = lane; e < l1 - l0; e += 32) st_pose(l0 + e, FLOW ? __ldcg(&pose[g0 + e]) : pose[g0 + e]);
        for (int e = lane; e < l2 - l1; e += 32) st_pose(l1 + e, FLOW ? __ldcg(&pose[g1 + e]) : pose[g1 + e]);
    }
    if (tid == 0) sm_lstart[ncells] = (unsigned short)ntot;
    if (tid < 8) st_pose(ntot + tid, make_float4(3.0e18f, 3.0e18f, 1.0f, 0.0f));   // sentinels behind the last staged pose
    __syncthreads();

    // ---- this warp's non-empty active cells, compacted: sm_act[slot] = j*32 + lane of the cell ---------------------
    unsigned char* my_act = sm_act + warp * TL::SLOTS;
    unsigned char* my_flag = sm_flag + warp * TL::SLOTS;
    float4* my_trial = sm_trial + warp * TL::SLOTS;
    unsigned* my_queue = sm_queue + warp * TL::QCAP;
    int n_act = 0;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        const int ay = warp * R + j;
        const bool valid = (ix0 + lane < nax) && (iy0 + ay < nay);
        int nmem = 0;
        if (valid) {
            const int lc = (2 * ay + 1) * RW + 2 * lane + 1;
            nmem = layer_inactive(g, cy0 + 2 * ay) ? 0 : (int)sm_lstart[lc + 1] - (int)sm_lstart[lc];   // an inactive row makes no trials
            if (nmem == 0 && trace) {
                const long long slot0 = (long long)((cx0 + 2 * lane) + n0 * (cy0 + 2 * ay)) * mv.n_select;
                for (int k = 0; k < mv.n_select; ++k) trace[slot0 + k] = make_uint2(0u, 0u);
            }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, nmem > 0);
        if (nmem > 0) my_act[n_act + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)(j * 32 + lane);
        n_act += __popc(bal);
    }
    __syncwarp();
    const int nrounds = (n_act + 31) >> 5;
    const uint32_t c3 = (kTagTrial << 24) | ((uint32_t)gamma << 16) | t_hi16;

    for (int k = 0; k < mv.n_select; ++k) {
        int qn = 0;   // entries in this warp's queue (warp-uniform)
        // per-slot state kept in registers between phases A and C: member index | rotate<<16 | outcome<<17 | sure<<19
        unsigned st[R];
        // ---- phase A: trial generation (a0, a5, a6) + broad phase (a8) + queue fill (a10) ------------------------
#pragma unroll
        for (int s = 0; s < R; ++s) {
            st[s] = 0u;
            if (s < nrounds) {   // warp-uniform
                const int slot = s * 32 + lane;
                unsigned mask = 0u, outcome = 0u;
                int rs[3] = {0, 0, 0}, p = 0;
                bool sure = false, rotate = false;
                float4 T = make_float4(0.f, 0.f, 1.f, 0.f);
                if (slot < n_act) {
                    const int id = my_act[slot];
                    const int ay = warp * R + (id >> 5), al = id & 31;
                    const int rxl = 2 * al + 1, ryl = 2 * ay + 1;
                    const int cell = (cx0 + 2 * al) + n0 * (cy0 + 2 * ay);
                    const int lc = ryl * RW + rxl;
                    const int own_s = sm_lstart[lc], nmem = (int)sm_lstart[lc + 1] - own_s;
                    const U4 b0 = philox4x32_10_rk((uint32_t)cell, t_lo, (uint32_t)k, c3, g.philox_rk);
                    p = own_s + (int)mulhi32(b0.x, (uint32_t)nmem);                 // R8
                    const float4 P = ld_pose(p);
                    TrialState A;
                    const bool inside = make_trial<KIND>(g, mv, shift, cell, 2, b0, 0u, make_float4(P.x, P.y, 0.f, 0.f),
                                                         make_float4(P.z, 0.f, 0.f, P.w), A, rotate);
                    T = make_float4(A.x, A.y, A.qw, A.qz);
                    my_trial[slot] = T;
                    my_flag[slot] = 0;
                    outcome = inside ? 1u : 2u;
                    if (inside) {
                        // a8: the three row runs of the 3x3 block hold <= kRowSlots poses each in all but rare cases: fixed,
                        // predicated candidate slots (bit kRowSlots*dy + j), no data-dependent loop in the common path
                        bool extra = false;
#pragma unroll
                        for (int dy = 0; dy < 3; ++dy) {
                            const int row = (ryl + dy - 1) * RW + rxl;
                            rs[dy] = sm_lstart[row - 1];
                            extra |= (int)sm_lstart[row + 2] - rs[dy] > kRowSlots;
                        }
                        if (seam) broad_slots<KIND, true>(g, S, sm_xy, rs, p, T, mask, sure);
                        else broad_slots<KIND, false>(g, S, sm_xy, rs, p, T, mask, sure);
                        if (extra) {   // a row run with more than kRowSlots poses: the rest one by one
#pragma unroll 1
                            for (int dy = 0; dy < 3; ++dy) {
                                const int row = (ryl + dy - 1) * RW + rxl;
                                for (int q = rs[dy] + kRowSlots; q < (int)sm_lstart[row + 2] && !sure; ++q) {
                                    if (q == p) continue;
                                    const float4 B = ld_pose(q);
                                    const float rx = min_image(B.x, T.x, g.hi[0], g.Ld[0]), ry = min_image(B.y, T.y, g.hi[1], g.Ld[1]);
                                    const float d2 = rx * rx + ry * ry;
                                    if (d2 >= S.dmax2) continue;
                                    sure = (KIND == kKindDisk || d2 < S.din2) ? true : pair_overlap_2d_cold<KIND, NV>(g, S, T, B, mv.eps_g);
                                }
                            }
                        }
                    }
                }
                if (KIND != kKindDisk) {
                    // a10: the lanes append their surviving candidates to the warp's queue -- positions from a warp prefix sum
                    // of the hit counts, then one predicated store per candidate slot (all lanes in step, no per-lane loop).
                    // A trial that is already decided ("sure", or left its cell) queues nothing: the early exit of P:45.
                    const unsigned pm = (outcome == 1u && !sure) ? mask : 0u;
                    const int cnt = __popc(pm);
                    int inc = cnt;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int n = __shfl_up_sync(0xffffffffu, inc, o);
                        inc += (lane >= o) ? n : 0;
                    }
                    // shared-memory address of this lane's first entry; the queue holds every slot of every lane (QCAP), no overflow
                    unsigned qaddr = (unsigned)__cvta_generic_to_shared(my_queue) + 4u * (unsigned)(qn + inc - cnt);
                    qn += __shfl_sync(0xffffffffu, inc, 31);
                    const unsigned base[3] = {((unsigned)slot << 16) + (unsigned)rs[0], ((unsigned)slot << 16) + (unsigned)rs[1],
                                              ((unsigned)slot << 16) + (unsigned)rs[2]};
                    push_bits<0>(qaddr, pm, base);   // entry = owner slot << 16 | staged index of the neighbour
                }
                st[s] = (unsigned)p | (rotate ? 1u << 16 : 0u) | (outcome << 17) | (sure ? 1u << 19 : 0u);
            }
        }
        __syncwarp();
        // ---- phase B: dense narrow phase (a9) --------------------------------------------------------------------------
        if (KIND != kKindDisk) {
            const int nq = qn;
            for (int e = lane; e < nq; e += 32) {
                const unsigned ent = my_queue[e];
                const int o = (int)(ent >> 16), q = (int)(ent & 0xffffu);
                if (pair_overlap_2d<KIND, NV>(g, S, my_trial[o], ld_pose(q), mv.eps_g, seam)) my_flag[o] = 1;
            }
            __syncwarp();
        }
        // ---- phase C: accept / write back (a11) ---------------------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < R; ++s) {
            const unsigned outcome0 = (st[s] >> 17) & 3u;
            if (outcome0 != 0u) {
                const int slot = s * 32 + lane;
                const int p = (int)(st[s] & 0xffffu);
                const bool rotate = (st[s] >> 16) & 1u;
                unsigned outcome = outcome0;
                if (outcome == 1u && (((st[s] >> 19) & 1u) || my_flag[slot])) outcome = 3u;
                const bool acc = outcome == 1u;
                if (acc || trace) {   // global index of the particle: only a write-back or the trace needs it
                    const int id = my_act[slot];
                    const int ay = warp * R + (id >> 5), al = id & 31;
                    const int seg = 2 * (2 * ay + 1) + ((2 * al + 1) >= split ? 1 : 0);
                    const int gi = sm_seg_g[seg] + (p - sm_seg_l[seg]);
                    if (acc) {
                        float4 T = my_trial[slot];
                        // R-wrap: at most one add per axis (x + (-L) is the same fp32 operation as x - L).  Only a cell on the box
                        // edge can hold a position outside [-L/2, L/2), and its tile is a seam tile (block-uniform)
                        if (!rotate && seam) {
                            T.x = __fadd_rn(T.x, (T.x >= g.hi[0]) ? -g.L[0] : (T.x < g.lo[0]) ? g.L[0] : 0.0f);
                            T.y = __fadd_rn(T.y, (T.y >= g.hi[1]) ? -g.L[1] : (T.y < g.lo[1]) ? g.L[1] : 0.0f);
                        }
                        pose[gi] = T;
                        st_pose(p, T);
                    }
                    if (trace) trace_store(trace, tag, gi, (long long)((cx0 + 2 * al) + n0 * (cy0 + 2 * ay)) * mv.n_select + k, rotate, outcome);
                }
                cc.tacc += (acc && !rotate) ? 1u : 0u;
                cc.racc += (acc && rotate) ? 1u : 0u;
                cc.trcell += (outcome == 2u) ? 1u : 0u;
                cc.nrot += rotate ? 1u : 0u;
            }
        }
        __syncwarp();
    }
    // per-lane tallies, summed over the warp by flush_counters (modulo 2^32, so a lane's negative share is harmless)
    cc.trials = (lane == 0) ? (unsigned)(n_act * mv.n_select) : 0u;   // every non-empty cell makes exactly n_select trials (R9)
    cc.trov = cc.trials - cc.nrot - cc.tacc - cc.trcell;              // neither accepted nor out of its cell: overlapped
    cc.rrov = cc.nrot - cc.racc;
    flush_counters(ctrl, cc);
}

// One launch = one colour: one tile per CTA.
template <int KIND, int NV, int WARPS, int R, int MINB>
__global__ void __launch_bounds__(32 * WARPS, MINB)
k_sweep_tile2d(const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv, const __grid_constant__ ShapeF S,
               const __grid_constant__ ShapeD SD, Control* __restrict__ ctrl, int colour_index, int cap_limit,
               float4* __restrict__ pose, const int* __restrict__ tag, const int* __restrict__ cell_start, uint32_t k0,
               uint32_t k1, uint2* __restrict__ trace, int tile0, int after_colour)
{
    // programmatic dependent launch: see k_sweep_warpcell for the rule (first colour pass: wait, then let the next one launch;
    // later passes: launch the next at once and wait only in front of the pose staging)
    const bool late_wait = after_colour != 0;
    if (!late_wait) pdl_wait();
    pdl_launch_dependents();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // tile0: first tile of this launch (0 unless the context runs a partition of the tile rows, hpmc_set_partition)
    tile2d_body<KIND, NV, WARPS, R, false>(g, mv, S, SD, ctrl, ctrl->hdr.perm[colour_index], tile0 + (int)blockIdx.x, cap_limit, pose, tag,
                                           cell_start, k0, k1, trace, smem_raw, late_wait);
}

// One launch = all four colours of a sweep, as a dataflow over (colour, tile) tickets.  A colour pass ends with a tail in
// which the last tiles run on a nearly empty GPU (a tile is four sequential trial rounds, ~20 us), and the next launch cannot
// start before it drains: ~16 of the 70 us of a pass on 1M pentagons.  But a tile of colour c+1 only needs the tiles of
// colour c that overlap its staged region -- the 3x3 tiles around it (they wrote poses it reads, and they read poses it will
// write) -- so persistent CTAs take tickets in (colour, tile) order and a tile waits just for those nine `done` stamps.  Every
// ticket a tile waits for is lower than its own, hence already held by a running or finished CTA: no deadlock.  Stamps are
// the sweep counter + 1, so the array is never cleared between sweeps.
template <int KIND, int NV, int WARPS, int R, int MINB>
__global__ void __launch_bounds__(32 * WARPS, MINB)
k_sweep_tile2d_flow(const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv, const __grid_constant__ ShapeF S,
                    const __grid_constant__ ShapeD SD, Control* __restrict__ ctrl, int cap_limit, float4* __restrict__ pose,
                    const int* __restrict__ tag, const int* __restrict__ cell_start, uint32_t k0, uint32_t k1,
                    uint2* __restrict__ trace, unsigned int* __restrict__ done)
{
    using TL = Tile2D<WARPS, R>;
    pdl_wait();   // no early launch of the successor: this persistent grid fills every SM
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // launch constants live in shared memory, not in registers across the tile body (64 registers: every one counts there)
    __shared__ int s_ticket, s_ntiles, s_tiles_x, s_tiles_y;
    __shared__ unsigned s_stamp;
    volatile unsigned int* vdone = done;
    if (threadIdx.x == 0) {
        const int nax = g.n[0] >> 1, nay = g.n[1] >> 1;
        s_tiles_x = (nax + kTileW - 1) / kTileW;
        s_tiles_y = (nay + TL::TH - 1) / TL::TH;
        s_ntiles = s_tiles_x * s_tiles_y;
        // stamp of this sweep: 1 + (t mod (2^32 - 1)).  Never 0 (the cleared state), and different from the stamp of the sweep
        // before, which is what every entry holds when the sweep starts -- also across the 2^32 wrap of the counter
        s_stamp = (unsigned)((((unsigned long long)ctrl->hdr.t_hi16 << 32) | ctrl->hdr.t_lo) % 0xFFFFFFFFull) + 1u;
        s_ticket = (int)atomicAdd(&ctrl->flow_ticket, 1u);
    }
    __syncthreads();
    for (;;) {
        const int ticket = s_ticket;                       // written before the barrier that ends the previous iteration
        const int ntiles = s_ntiles;
        if (ticket >= 4 * ntiles) break;
        const int ci = ticket / ntiles, tile = ticket - ci * ntiles;
        if (ci > 0 && threadIdx.x < 9) {                   // the nine tiles of the previous colour around this one
            const int tiles_x = s_tiles_x, tiles_y = s_tiles_y;
            const unsigned stamp = s_stamp;
            const int tx = tile % tiles_x, ty = tile / tiles_x;
            int nx = tx + (int)(threadIdx.x % 3) - 1, ny = ty + (int)(threadIdx.x / 3) - 1;
            nx += (nx < 0) ? tiles_x : 0; nx -= (nx >= tiles_x) ? tiles_x : 0;
            ny += (ny < 0) ? tiles_y : 0; ny -= (ny >= tiles_y) ? tiles_y : 0;
            const int dep = (ci - 1) * ntiles + ny * tiles_x + nx;
            unsigned ns = 128u;
            while (vdone[dep] != stamp) {   // exponential back-off: every poll is an L2 access competing with working CTAs
                __nanosleep(ns);
                ns = ns < 2048u ? 2u * ns : ns;
            }
            __threadfence();
        }
        __syncthreads();                                   // dependencies met; every thread has read its ticket
        tile2d_body<KIND, NV, WARPS, R, true>(g, mv, S, SD, ctrl, ctrl->hdr.perm[ci], tile, cap_limit, pose, tag, cell_start, k0, k1,
                                              trace, smem_raw);
        __threadfence();                                   // this thread's pose write-backs are visible device-wide ...
        __syncthreads();                                   // ... and the tile's shared memory is no longer in use
        if (threadIdx.x == 0) {
            vdone[ticket] = s_stamp;                       // ... before the tile is announced (ticket = ci * ntiles + tile)
            s_ticket = (int)atomicAdd(&ctrl->flow_ticket, 1u);
        }
        __syncthreads();
    }
    // the last CTA to leave re-arms the ticket counter for the next launch
    if (threadIdx.x == 0 && atomicAdd(&ctrl->flow_exited, 1u) == gridDim.x - 1) {
        ctrl->flow_exited = 0u;
        ctrl->flow_ticket = 0u;
    }
}

}  // namespace hpmc
