// Distributed state across several GPUs: the once-per-sweep routing step -- the paper's
// stage 9, "Migrate particles to new domains and communicate ghost particles" -- on the cell-sorted arrays of one rank.
//
// A rank owns the slab of cell rows [r0, r1) of the sweep's shifted grid; its last row r1 - 1 is the inactive region (R-strip),
// so during the sweep it reads one row of another rank -- row r0 - 1, the inactive last row of the slab below -- and that row
// does not change.  The next sweep has another grid shift: a particle's row moves by at most one.  k_route computes,
// with the pinned cell function, the row of every owned particle in the NEXT sweep's grid and
//     keeps   rows r0 - 1 .. r1 - 1   (r0 - 1: it now belongs to the rank below, but is this rank's ghost row)
//     sends up    rows r1 - 1 and r1  (r1 - 1: the ghost row of the rank above; r1: migrates to it)
//     sends down  row  r0 - 1         (migrates to the rank below)
// and drops the old ghost row.  Rows are taken modulo n_y (periodic box).  The order inside the three outputs is arbitrary:
// the next cell-list build puts the members of every cell in ascending (global) tag.
#pragma once
#include "common.cuh"

namespace hpmc {

// route[0..2] = keep / up / down counts, route[3] = particles that fit no class (owned_only: must stay 0)
template <int WHICH>
__device__ __forceinline__ int warp_slot(unsigned int* counter, bool mine, int lane)
{
    const unsigned bal = __ballot_sync(0xffffffffu, mine);
    int base = 0;
    if (bal != 0u) {
        const int leader = __ffs(bal) - 1;
        if (lane == leader) base = (int)atomicAdd(counter + WHICH, (unsigned)__popc(bal));
        base = __shfl_sync(0xffffffffu, base, leader);
    }
    return base + __popc(bal & ((1u << lane) - 1u));
}

__global__ void __launch_bounds__(256)
k_route(const __grid_constant__ GridParams g, Control* __restrict__ ctrl, uint32_t k0, uint32_t k1, int owned_only, int r0, int r1,
        const float4* __restrict__ src_pose, const int* __restrict__ src_tag, const int* __restrict__ cell_start,
        float4* __restrict__ keep_pose, int* __restrict__ keep_tag, float4* __restrict__ up_pose, int* __restrict__ up_tag, int cap_up,
        float4* __restrict__ down_pose, int* __restrict__ down_tag, int cap_down, unsigned int* __restrict__ route)
{
    __shared__ SweepHeader sh;
    if (threadIdx.x == 0) make_header(g, k0, k1, ctrl->t, false, sh);   // the sweep the next build will set up
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int n0 = g.n[0], n1 = g.n[1];
    const int begin = owned_only ? cell_start[r0 * n0] : 0;
    const int end = owned_only ? cell_start[r1 * n0] : g.N;
    const int i = begin + blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = i < end;
    float4 P = make_float4(0.f, 0.f, 1.f, 0.f);
    int tg = 0, row = -1;
    if (live) {
        P = src_pose[i];
        tg = src_tag[i];
        row = cell_axis(P.y, g.lo[1], sh.shift[1], g.L[1], g.inv_w[1], n1);
    }
    const int ghost = (r0 - 1 + n1) % n1, above = r1 % n1, last = r1 - 1;
    const bool inside = live && row >= r0 && row < r1;
    const bool keep = inside || (live && row == ghost);
    const bool up = live && (row == last || row == above);
    const bool down = live && row == ghost;
    const bool lost = live && !keep && !up && !down;
    const int ik = warp_slot<0>(route, keep, lane);
    const int iu = warp_slot<1>(route, up, lane);
    const int id = warp_slot<2>(route, down, lane);
    if (keep) { keep_pose[ik] = P; keep_tag[ik] = tg; }          // at most as many as there were: always fits
    if (up && iu < cap_up) { up_pose[iu] = P; up_tag[iu] = tg; }
    if (down && id < cap_down) { down_pose[id] = P; down_tag[id] = tg; }
    if (lost) atomicAdd(route + 3, 1u);
}

}  // namespace hpmc
