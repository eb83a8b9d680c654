// Shared parameter blocks and the pinned fp32 geometry helpers of the CUDA path.
// P:<n> = PAPER.md line n, R<k> = DESIGN.md section 2.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "philox.cuh"

namespace hpmc {

constexpr int kMaxVerts = 32;
constexpr int kKindDisk = 0, kKindPolygon = 1, kKindPolyhedron = 2;

// grid + box, passed by value to every kernel (lands in the constant bank)
struct GridParams {
    int dim;
    int n[3];         // cells per side (even, >= 4), R11
    int C;            // number of cells
    int N;            // number of particles
    float L[3];       // box edge (fp32-rounded, R-box)
    float lo[3];      // -L/2 (exact)
    float hi[3];      // +L/2 (exact)
    float inv_w[3];   // (float)(n/L), R13
    float w_f[3];     // (float)(L/n), scale of the grid shift, R10
    double Ld[3];     // (double)L for the fp64 seam subtraction, R21
    // P:134-138 inactive region (R-strip): n[dim-1] bytes, one per layer of cells along the last axis; the cells of a flagged
    // layer make no trials this sweep.  nullptr = none.  Static between hpmc_set_inactive_layers calls: any kernel may read
    // it in front of its programmatic-launch wait.
    const unsigned char* inactive;
    // the ten round keys of Philox4x32-10 for this system's seed, (k0 + r W0, k1 + r W1): operands straight from the constant
    // bank in the tile pass instead of 18 vector adds per block (philox4x32_10_rk)
    uint32_t philox_rk[20];
};

__device__ __forceinline__ bool layer_inactive(const GridParams& g, int layer) { return g.inactive != nullptr && g.inactive[layer] != 0; }

struct MoveParams {
    float d, a;       // R5, R6
    int n_select;     // R9
    float eps_g;      // R15 guard band
};

// what every kernel of one sweep needs to know about that sweep (written by k_prepare)
struct SweepHeader {
    float shift[3];   // R10
    int perm[8];      // R12
    uint32_t t_lo, t_hi16;
    uint32_t pad;
};

constexpr int kCounterSets = 128;

// device-resident control block
struct Control {
    unsigned long long t;  // sweep counter (persists across calls)
    unsigned long long sweeps;
    // trans_acc, trans_rej_overlap, trans_rej_cell, rot_acc, rot_rej_overlap, trials (+2 pad): kCounterSets replicas, one
    // 64-byte line each.  Every warp of a colour pass adds its tallies to the replica picked by its CTA index: thousands of
    // same-address atomics per launch would otherwise serialise in one L2 slice (measured: ~40 us per launch on 1M
    // pentagons).  Readers sum the replicas.
    unsigned long long counters[kCounterSets][8];
    unsigned long long overlaps;     // validator result
    unsigned int flow_ticket, flow_exited;   // k_sweep_tile2d_flow: next (colour, tile) ticket; CTAs that have left
    unsigned int bad_coords, pad_bc;         // particles whose coordinates were not finite or not in [-L/2, L/2) when a cell list was built
    unsigned int route[4];                   // k_route: particles kept / sent up / sent down / fitting no class
    SweepHeader hdr;
};

// Programmatic dependent launch (sm_90+): a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may start
// while its predecessor in the stream still runs; it must not touch anything the predecessor writes (or reads and it writes)
// before pdl_wait(), which returns once the predecessor grid has completed and its memory operations are visible.
// pdl_launch_dependents() lets the successor's launch begin: called at the top, it takes the launch latency (~2 us, a third
// of a colour pass of a 4096-particle system) off the critical path.  Both are no-ops in a kernel launched the plain way.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Cell-sorted state.  3-D: pos = (x, y, z, 0) and quat = (w, x, y, z), two arrays.  2-D: ONE array of
// poses (x, y, qw, qz) in `pos` (R30: z = 0 and qx = qy = 0 always), `quat` is not allocated -- half the bytes per particle.
__device__ __forceinline__ void load_state(int dim, const float4* __restrict__ pos, const float4* __restrict__ quat, int i,
                                           float4& x, float4& q)
{
    const float4 P = __ldcg(&pos[i]);   // L2-coherent: the dataflow pass reads poses other CTAs of the same launch wrote
    if (dim == 2) {
        x = make_float4(P.x, P.y, 0.0f, 0.0f);
        q = make_float4(P.z, 0.0f, 0.0f, P.w);
    } else {
        x = P;
        q = __ldcg(&quat[i]);
    }
}

__device__ __forceinline__ void store_state(int dim, float4* __restrict__ pos, float4* __restrict__ quat, int i, const float4& x,
                                            const float4& q, bool rotated)
{
    if (dim == 2) pos[i] = make_float4(x.x, x.y, q.x, q.w);
    else if (!rotated) pos[i] = x;
    else quat[i] = q;
}

// R13: the one cell function, used both to assign cells and to test "left its cell".
// Explicit _rn intrinsics so that no multiply-add is ever contracted.
__device__ __forceinline__ int cell_axis(float x, float lo, float s, float L, float inv_w, int n)
{
    float f = __fsub_rn(__fsub_rn(x, lo), s);
    if (f < 0.0f) f = __fadd_rn(f, L);
    if (f >= L) f = __fsub_rn(f, L);
    int c = (int)floorf(__fmul_rn(f, inv_w));
    if (c >= n) c -= n;
    return c;
}

// The cell-list builders use the same function but may meet caller data that breaks the precondition (coordinates in
// [-L/2, L/2), finite): such a particle is counted in Control::bad_coords and its cell index clamped into the grid, so that no
// histogram or scatter ever indexes out of bounds; hpmc_count_overlaps / hpmc_get_state then report HPMC_E_ARG.
__device__ __forceinline__ int cell_of_checked(const GridParams& g, const float shift[3], float x, float y, float z, bool& bad)
{
    bad = !(x >= g.lo[0] && x < g.hi[0] && y >= g.lo[1] && y < g.hi[1]) || (g.dim == 3 && !(z >= g.lo[2] && z < g.hi[2]));
    int cx = cell_axis(x, g.lo[0], shift[0], g.L[0], g.inv_w[0], g.n[0]);
    int cy = cell_axis(y, g.lo[1], shift[1], g.L[1], g.inv_w[1], g.n[1]);
    int cz = (g.dim == 3) ? cell_axis(z, g.lo[2], shift[2], g.L[2], g.inv_w[2], g.n[2]) : 0;
    if (bad) {
        cx = min(max(cx, 0), g.n[0] - 1);
        cy = min(max(cy, 0), g.n[1] - 1);
        cz = min(max(cz, 0), g.n[2] - 1);
    }
    return cx + g.n[0] * (cy + g.n[1] * cz);
}

__device__ __forceinline__ int cell_of(const GridParams& g, const float shift[3], float x, float y, float z, int& cx,
                                       int& cy, int& cz)
{
    cx = cell_axis(x, g.lo[0], shift[0], g.L[0], g.inv_w[0], g.n[0]);
    cy = cell_axis(y, g.lo[1], shift[1], g.L[1], g.inv_w[1], g.n[1]);
    cz = (g.dim == 3) ? cell_axis(z, g.lo[2], shift[2], g.L[2], g.inv_w[2], g.n[2]) : 0;
    return cx + g.n[0] * (cy + g.n[1] * cz);
}

// O3.1/O3.2 (R10, R12): grid shift and colour order of sweep t
__device__ inline void make_header(const GridParams& g, uint32_t k0, uint32_t k1, unsigned long long t, bool zero_shift,
                                   SweepHeader& h)
{
    const uint32_t t_lo = (uint32_t)t, t_hi16 = (uint32_t)((t >> 32) & 0xFFFFull);
    h.t_lo = t_lo;
    h.t_hi16 = t_hi16;
    const U4 r = philox4x32_10(0u, t_lo, 0u, (kTagShift << 24) | t_hi16, k0, k1);
    const uint32_t rr[3] = {r.x, r.y, r.z};
    for (int k = 0; k < 3; ++k) h.shift[k] = (k < g.dim && !zero_shift) ? __fmul_rn(g.w_f[k], u01(rr[k])) : 0.0f;
    const int ncol = 1 << g.dim;
    for (int c = 0; c < 8; ++c) h.perm[c] = c;
    int word = 0;
    U4 blk{0, 0, 0, 0};
    for (int i = ncol - 1; i >= 1; --i) {
        if ((word & 3) == 0) blk = philox4x32_10(0u, t_lo, (uint32_t)(word >> 2), (kTagPerm << 24) | t_hi16, k0, k1);
        const uint32_t rw = ((word & 3) == 0) ? blk.x : ((word & 3) == 1) ? blk.y : ((word & 3) == 2) ? blk.z : blk.w;
        const uint32_t j = mulhi32(rw, (uint32_t)(i + 1));
        const int tmp = h.perm[i];
        h.perm[i] = h.perm[j];
        h.perm[j] = tmp;
        ++word;
    }
}

}  // namespace hpmc
