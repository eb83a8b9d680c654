// 2-D colour pass, tile version (S:8(a) rows a4-a11).
//
// One CTA = a tile of 32 x TY active cells of the current colour (one warp per row of 32 active cells, one lane
// per cell).  The CTA first stages every particle of the (2*32+1) x (2*TY+1) cell region around its tile into
// shared memory as compact float4 (x, y, qw, qz) with coalesced loads (a7: "neighbour gather staged in shared
// memory").  After that the warps are independent: active cells of one colour never share a neighbour cell's
// *writes* (their 3x3 blocks only overlap in inactive cells), so everything below the staging
// barrier is warp-synchronous:
//
//   A  every lane generates trial k of its cell (Philox -> member, move type, displacement; leave-cell test
//      with the pinned cell function), runs the circumsphere broad phase over the three staged row runs of its
//      3x3 block and turns the hits into a bit mask; centres closer than the inscribed-disk bound are decided
//      on the spot.  The warp packs all (lane, neighbour) hits into a per-warp queue in shared memory.
//   B  the queue is drained densely: lane e takes entry e, e+32, ... and runs the branch-free separating-axis
//      test; an overlap sets the owner's flag.  This is the paper's block queue at warp scope:
//      lanes no longer idle while one neighbour of one trial is in its narrow phase.
//   C  owners read their flag, accepted moves are written to the staged copy (so trial k+1 of the cell sees it)
//      and to global memory.
//
// A tile whose region holds more particles than the staging capacity falls back to the per-thread global
// path (sweep_cell_global); results are identical.
#pragma once
#include "common.cuh"
#include "overlap.cuh"
#include "sweep.cuh"

namespace hpmc {

constexpr int kTileW = 32;                    // active cells per tile row = lanes of a warp
constexpr int kRegionW = 2 * kTileW + 1;      // staged cells per region row
constexpr int kCapPerCell = 2;                // staging capacity in particles per region cell (pentagon fluid: ~1)
constexpr int kWarpQueueCap = 160;            // narrow-phase queue entries per warp and trial round

template <int TY>
struct Tile2D {
    static constexpr int NT = 32 * TY;
    static constexpr int RH = 2 * TY + 1;
    static constexpr int NCELLS = kRegionW * RH;
    static constexpr int CAP = kCapPerCell * NCELLS;
    static constexpr int CPT = (NCELLS + NT - 1) / NT;   // region cells per thread while staging
    // shared-memory carve (bytes)
    static constexpr size_t off_pose = 0;
    static constexpr size_t off_trial = off_pose + sizeof(float4) * CAP;
    static constexpr size_t off_gidx = off_trial + sizeof(float4) * NT;
    static constexpr size_t off_lstart = off_gidx + sizeof(int) * CAP;
    static constexpr size_t off_queue = off_lstart + sizeof(int) * (NCELLS + 1);
    static constexpr size_t off_wsum = off_queue + sizeof(unsigned) * TY * kWarpQueueCap;
    static constexpr size_t off_flag = off_wsum + sizeof(int) * CPT * TY;
    static constexpr size_t bytes = off_flag + sizeof(unsigned) * NT;
};

// narrow phase of trial pose A against staged pose B, both (x, y, qw, qz); true = overlap (R15 guard band)
template <int KIND, int NV>
__device__ __forceinline__ bool pair_overlap_2d(const GridParams& g, const ShapeF& S, const float4& A, const float4& B, float eps)
{
    const float rx = min_image(B.x, A.x, g.hi[0], g.Ld[0]);
    const float ry = min_image(B.y, A.y, g.hi[1], g.Ld[1]);
    if (KIND == kKindDisk) return rx * rx + ry * ry < S.dmax2;
    const float cA = A.z * A.z - A.w * A.w, sA = 2.0f * A.z * A.w;   // cos t = w^2 - z^2, sin t = 2wz (R30)
    const float cB = B.z * B.z - B.w * B.w, sB = 2.0f * B.z * B.w;
    return !(polygon_max_sep<float, NV>(S, rx, ry, cA, sA, cB, sB) >= eps);
}

template <int KIND, int NV, int TY>
__global__ void __launch_bounds__(32 * TY)
k_sweep_tile2d(const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv, const __grid_constant__ ShapeF S,
               const __grid_constant__ ShapeD SD, Control* __restrict__ ctrl, int colour_index, int cap_limit,
               float4* __restrict__ pos, float4* __restrict__ quat, const int* __restrict__ tag,
               const int* __restrict__ cell_start, uint32_t k0, uint32_t k1, uint2* __restrict__ trace)
{
    using TL = Tile2D<TY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* sm_pose = reinterpret_cast<float4*>(smem_raw + TL::off_pose);     // staged (x, y, qw, qz)
    float4* sm_trial = reinterpret_cast<float4*>(smem_raw + TL::off_trial);   // trial pose of every lane
    int* sm_gidx = reinterpret_cast<int*>(smem_raw + TL::off_gidx);           // global (cell-sorted) index
    int* sm_lstart = reinterpret_cast<int*>(smem_raw + TL::off_lstart);       // local CSR over region cells
    unsigned* sm_queue = reinterpret_cast<unsigned*>(smem_raw + TL::off_queue);
    int* sm_wsum = reinterpret_cast<int*>(smem_raw + TL::off_wsum);
    unsigned* sm_flag = reinterpret_cast<unsigned*>(smem_raw + TL::off_flag);

    const SweepHeader& H = ctrl->hdr;
    const int gamma = H.perm[colour_index];
    const uint32_t t_lo = H.t_lo, t_hi16 = H.t_hi16;
    const float shift[3] = {H.shift[0], H.shift[1], 0.0f};
    const int gx = gamma & 1, gy = (gamma >> 1) & 1;
    const int nax = g.n[0] >> 1, nay = g.n[1] >> 1;
    const int tiles_x = (nax + kTileW - 1) / kTileW;
    const int tx = blockIdx.x % tiles_x, ty = blockIdx.x / tiles_x;
    const int ix0 = tx * kTileW, iy0 = ty * TY;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // region = cells [cx0-1, cx0-1+RW) x [cy0-1, cy0-1+RHv), clipped to what the valid active cells of the tile need
    const int cx0 = 2 * ix0 + gx, cy0 = 2 * iy0 + gy;
    const int RW = 2 * min(kTileW, nax - ix0) + 1, RHv = 2 * min(TY, nay - iy0) + 1;
    const int ncells = RW * RHv;

    // ---- staging: region cell counts -> local CSR (prefix sum) -> coalesced copy ------------------------------
    int cs[TL::CPT], cnt[TL::CPT], inc[TL::CPT];
#pragma unroll
    for (int j = 0; j < TL::CPT; ++j) {
        const int lc = j * TL::NT + tid;
        cs[j] = 0; cnt[j] = 0;
        if (lc < ncells) {
            const int ry = lc / RW, rx = lc - ry * RW;
            int cx = cx0 - 1 + rx, cy = cy0 - 1 + ry;
            cx += (cx < 0) ? g.n[0] : 0; cx -= (cx >= g.n[0]) ? g.n[0] : 0;
            cy += (cy < 0) ? g.n[1] : 0; cy -= (cy >= g.n[1]) ? g.n[1] : 0;
            const int c = cx + g.n[0] * cy;
            cs[j] = cell_start[c];
            cnt[j] = cell_start[c + 1] - cs[j];
        }
        int v = cnt[j];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int n = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += n;
        }
        inc[j] = v;
        if (lane == 31) sm_wsum[j * TY + warp] = v;
    }
    __syncthreads();
    int run = 0, mybase[TL::CPT];
#pragma unroll
    for (int j = 0; j < TL::CPT; ++j)
#pragma unroll
        for (int w = 0; w < TY; ++w) {
            if (w == warp) mybase[j] = run;
            run += sm_wsum[j * TY + w];
        }
    const int ntot = run;
    const bool staged = ntot <= min(cap_limit, TL::CAP);   // block-uniform
    const bool valid = (ix0 + lane < nax) && (iy0 + warp < nay);
    const int cx = cx0 + 2 * lane, cy = cy0 + 2 * warp;     // this lane's active cell
    CellCounters cc;

    if (!staged) {
        // overflow: more particles around this tile than the staging buffers hold -> per-thread global path
        if (valid)
            sweep_cell_global<KIND, NV>(g, mv, S, SD, gamma, t_lo, t_hi16, shift, cx, cy, 0, pos, quat, tag, cell_start, k0, k1,
                                        trace, cc);
        flush_counters(ctrl, cc);
        return;
    }

#pragma unroll
    for (int j = 0; j < TL::CPT; ++j) {
        const int lc = j * TL::NT + tid;
        if (lc < ncells) {
            const int l0 = mybase[j] + inc[j] - cnt[j];
            sm_lstart[lc] = l0;
            for (int m = 0; m < cnt[j]; ++m) {
                const int gi = cs[j] + m;
                const float4 P = pos[gi];
                float4 Q = make_float4(1.f, 0.f, 0.f, 0.f);
                if (KIND != kKindDisk) Q = quat[gi];
                sm_pose[l0 + m] = make_float4(P.x, P.y, Q.x, Q.w);
                sm_gidx[l0 + m] = gi;
            }
        }
    }
    if (tid == 0) sm_lstart[ncells] = ntot;
    __syncthreads();

    // ---- per-lane constants: own cell and the three row runs of its 3x3 block (local indices) -----------------
    const int cell = cx + g.n[0] * cy;
    const long long slot0 = (long long)cell * mv.n_select;
    int own_s = 0, nmem = 0, rs[3] = {0, 0, 0}, re[3] = {0, 0, 0};
    if (valid) {
        const int rxl = 2 * lane + 1, ryl = 2 * warp + 1;
        const int lc = ryl * RW + rxl;
        own_s = sm_lstart[lc];
        nmem = sm_lstart[lc + 1] - own_s;
#pragma unroll
        for (int dy = 0; dy < 3; ++dy) {
            const int row = (ryl + dy - 1) * RW + rxl;
            rs[dy] = sm_lstart[row - 1];
            re[dy] = sm_lstart[row + 2];
        }
    }
    const bool act = valid && nmem > 0;
    if (valid && !act && trace)
        for (int k = 0; k < mv.n_select; ++k) trace[slot0 + k] = make_uint2(0u, 0u);
    const int n0 = re[0] - rs[0], n01 = n0 + (re[1] - rs[1]);
    unsigned* my_queue = sm_queue + warp * kWarpQueueCap;
    const uint32_t c3 = (kTagTrial << 24) | ((uint32_t)gamma << 16) | t_hi16;

    for (int k = 0; k < mv.n_select; ++k) {
        // ---- phase A: trial generation (a0, a5, a6) + broad phase (a8) --------------------------------------
        int p = 0, outcome = 0;
        bool rotate = false, own_ov = false;
        float4 T = make_float4(0.f, 0.f, 1.f, 0.f);
        unsigned mask = 0u;
        if (act) {
            const U4 b0 = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)k, c3, k0, k1);
            p = own_s + (int)mulhi32(b0.x, (uint32_t)nmem);                 // R8
            rotate = (KIND != kKindDisk) && (b0.y >> 31);                    // R7
            const float4 P = sm_pose[p];
            T = P;
            outcome = 1;
            ++cc.trials;
            if (!rotate) {
                T.x = __fmaf_rn(mv.d, usym(b0.z), P.x);                      // R5
                T.y = __fmaf_rn(mv.d, usym(b0.w), P.y);
                int tcx, tcy, tcz;
                if (cell_of(g, shift, T.x, T.y, 0.0f, tcx, tcy, tcz) != cell) outcome = 2;   // a6, R13
            } else {                                                         // R6, 2-D
                float sn, cs_;
                sincosf(0.5f * __fmul_rn(mv.a, usym(b0.z)), &sn, &cs_);
                const float w = P.z * cs_ - P.w * sn, z = P.z * sn + P.w * cs_;
                const float inv = rsqrtf(w * w + z * z);
                T.z = w * inv;
                T.w = z * inv;
            }
            if (outcome == 1) {
                int bit = 0;
#pragma unroll
                for (int dy = 0; dy < 3; ++dy) {
                    for (int q = rs[dy]; q < re[dy]; ++q, ++bit) {
                        if (q == p) continue;
                        const float4 B = sm_pose[q];
                        const float rx = min_image(B.x, T.x, g.hi[0], g.Ld[0]);
                        const float ry = min_image(B.y, T.y, g.hi[1], g.Ld[1]);
                        const float d2 = rx * rx + ry * ry;
                        if (d2 >= S.dmax2) continue;                          // a8 circumsphere (R16)
                        if (KIND == kKindDisk || d2 < S.din2) own_ov = true;  // inside the inscribed-disk bound
                        else if (bit < 32) mask |= 1u << bit;
                        else if (!own_ov) own_ov = pair_overlap_2d<KIND, NV>(g, S, T, B, mv.eps_g);   // > 32 candidates
                    }
                }
                if (own_ov) mask = 0u;                                        // early exit
            }
        }
        if (KIND != kKindDisk) {
            // pack the hits of all lanes into the warp queue (a10)
            const int c = __popc(mask);
            int incl = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += n;
            }
            const int total = __shfl_sync(0xffffffffu, incl, 31);
            int slot = incl - c;
            sm_trial[tid] = T;
            sm_flag[tid] = 0u;
            while (mask) {
                const int b = __ffs(mask) - 1;
                mask &= mask - 1u;
                const int q = (b < n0) ? rs[0] + b : (b < n01) ? rs[1] + (b - n0) : rs[2] + (b - n01);
                if (slot < kWarpQueueCap) my_queue[slot] = ((unsigned)lane << 24) | (unsigned)q;
                else if (!own_ov) own_ov = pair_overlap_2d<KIND, NV>(g, S, T, sm_pose[q], mv.eps_g);   // queue full
                ++slot;
            }
            __syncwarp();
            // ---- phase B: dense narrow phase (a9) -----------------------------------------------------------
            const int nq = min(total, kWarpQueueCap);
            for (int e = lane; e < nq; e += 32) {
                const unsigned ent = my_queue[e];
                const int o = (int)(ent >> 24), q = (int)(ent & 0xffffffu);
                if (pair_overlap_2d<KIND, NV>(g, S, sm_trial[(warp << 5) + o], sm_pose[q], mv.eps_g)) sm_flag[(warp << 5) + o] = 1u;
            }
            __syncwarp();
            if (sm_flag[tid]) own_ov = true;
        }
        // ---- phase C: accept / write back (a11) ---------------------------------------------------------------
        if (act) {
            if (outcome == 1 && own_ov) outcome = 3;
            if (outcome == 1) {
                if (!rotate) {
                    float x = T.x, y = T.y;
                    if (x >= g.hi[0]) x = __fsub_rn(x, g.L[0]); else if (x < g.lo[0]) x = __fadd_rn(x, g.L[0]);
                    if (y >= g.hi[1]) y = __fsub_rn(y, g.L[1]); else if (y < g.lo[1]) y = __fadd_rn(y, g.L[1]);
                    T.x = x; T.y = y;
                    pos[sm_gidx[p]] = make_float4(x, y, 0.0f, 0.0f);
                    ++cc.tacc;
                } else {
                    quat[sm_gidx[p]] = make_float4(T.z, 0.0f, 0.0f, T.w);
                    ++cc.racc;
                }
                sm_pose[p] = T;
            } else if (outcome == 2) {
                ++cc.trcell;
            } else {
                if (rotate) ++cc.rrov; else ++cc.trov;
            }
            if (trace) trace[slot0 + k] = make_uint2((uint32_t)tag[sm_gidx[p]], (rotate ? 1u : 0u) | ((uint32_t)outcome << 8));
        }
        __syncwarp();
    }
    flush_counters(ctrl, cc);
}

}  // namespace hpmc
