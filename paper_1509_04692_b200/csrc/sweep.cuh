// The checkerboard sweep kernel (S:8(a) rows a4-a11) and the overlap-count validator (a12).
//
// One launch = one colour of the 2^d checkerboard.  Every non-empty cell of that colour
// makes n_select sequential trials (R9); cells of one colour are independent because a trial reads only
// the 3^d block around its own cell and may not leave the cell.
#pragma once
#include "common.cuh"
#include "overlap.cuh"

namespace hpmc {

// minimum-image separation of one coordinate (R21): same-image pairs are one exact fp32 subtraction;
// pairs across the periodic seam are subtracted in fp64 with the exact box edge and rounded once.
__device__ __forceinline__ float min_image(float xj, float xt, float hi, double Ld)
{
    float r = xj - xt;
    if (fabsf(r) > hi) {
        double rd = (double)xj - (double)xt;
        rd += (rd < 0.0) ? Ld : -Ld;
        r = (float)rd;
    }
    return r;
}

constexpr float kGjkDeepF = 1e-4f;   // fp32 GJK "certainly overlapping" threshold (see overlap.cuh)

// exact minimum-image separation in fp64 from the fp32 coordinates (fallback narrow phase only)
__device__ __forceinline__ double min_image_d(float xj, float xt, double Ld)
{
    double rd = (double)xj - (double)xt;
    if (rd > 0.5 * Ld) rd -= Ld;
    else if (rd < -0.5 * Ld) rd += Ld;
    return rd;
}

// narrow phase of trial pose A against staged pose B, both (x, y, qw, qz); one definition for every
// 2-D pass variant; true = overlap (R15 guard band)
template <int KIND, int NV>
__device__ __forceinline__ bool pair_overlap_2d(const GridParams& g, const ShapeF& S, const float4& A, const float4& B, float eps, bool seam)
{
    float rx = B.x - A.x, ry = B.y - A.y;
    if (seam) {
        rx = min_image(B.x, A.x, g.hi[0], g.Ld[0]);
        ry = min_image(B.y, A.y, g.hi[1], g.Ld[1]);
    }
    if (KIND == kKindDisk) return rx * rx + ry * ry < S.dmax2;
    const float cA = A.z * A.z - A.w * A.w, sA = 2.0f * A.z * A.w;   // cos t = w^2 - z^2, sin t = 2wz (R30)
    const float cB = B.z * B.z - B.w * B.w, sB = 2.0f * B.z * B.w;
    return !polygon_separated<NV>(S, rx, ry, cA, sA, cB, sB, eps);
}

struct TrialState {
    float x, y, z;        // trial position (unwrapped)
    float qw, qx, qy, qz; // trial orientation
};

// sin and cos of the half rotation angle h, |h| <= a/2.  For a <= 1 rad (every config: a = 0.1) the Taylor series to
// h^9 / h^10 is exact to fp32 rounding (next terms < 1.3e-11) and costs a dozen FMAs instead of sincosf's range reduction.
__device__ __forceinline__ void small_sincos(float h, float a, float& sn, float& cs)
{
    if (a <= 1.0f) {
        const float h2 = __fmul_rn(h, h);
        float ps = __fmaf_rn(h2, 2.7557319e-6f, -1.9841270e-4f);
        ps = __fmaf_rn(h2, ps, 8.3333333e-3f);
        ps = __fmaf_rn(h2, ps, -1.6666667e-1f);
        sn = __fmaf_rn(__fmul_rn(h, h2), ps, h);
        float pc = __fmaf_rn(h2, -2.7557319e-7f, 2.4801587e-5f);
        pc = __fmaf_rn(h2, pc, -1.3888889e-3f);
        pc = __fmaf_rn(h2, pc, 4.1666667e-2f);
        pc = __fmaf_rn(h2, pc, -0.5f);
        cs = __fmaf_rn(h2, pc, 1.0f);
    } else {
        sincosf(h, &sn, &cs);
    }
}

// R6, 2-D: q' = normalise(q (x) dq) for q = (qw, 0, 0, qz), dq = (cs, 0, 0, sn).  Explicit roundings: one definition for
// make_trial and for the speculative pass, which replays accepted rotations (sweep_spec2d.cuh)
__device__ __forceinline__ void rotate_2d(float qw, float qz, float sn, float cs, float& ow, float& oz)
{
    const float w = __fmaf_rn(qw, cs, -__fmul_rn(qz, sn));
    const float z = __fmaf_rn(qw, sn, __fmul_rn(qz, cs));
    const float inv = rsqrtf(__fmaf_rn(w, w, __fmul_rn(z, z)));
    ow = __fmul_rn(w, inv);
    oz = __fmul_rn(z, inv);
}

// a5 + a6: the trial pose of one move (R5-R7) and the leave-cell test (R13).  b0 = (select, type, ua, ub), uc = first
// word of block 1 (3-D only).  Returns false iff a translation left `cell`.  One definition for every colour-pass
// variant, so that they produce bit-identical trials.
template <int KIND>
__device__ __forceinline__ bool make_trial(const GridParams& g, const MoveParams& mv, const float* shift, int cell, int dim,
                                           const U4& b0, uint32_t uc, const float4& xp, const float4& qp, TrialState& A, bool& rotate)
{
    rotate = (KIND != kKindDisk) && (b0.y >> 31);   // R7
    A = TrialState{xp.x, xp.y, xp.z, qp.x, qp.y, qp.z, qp.w};
    if (!rotate) {
        A.x = __fmaf_rn(mv.d, usym(b0.z), xp.x);   // R5: one rounding per axis
        A.y = __fmaf_rn(mv.d, usym(b0.w), xp.y);
        if (dim == 3) A.z = __fmaf_rn(mv.d, usym(uc), xp.z);
        int tx, ty, tz;
        return cell_of(g, shift, A.x, A.y, A.z, tx, ty, tz) == cell;   // a6: same pinned cell function (R13)
    }
    if (dim == 2) {                                   // R6, 2-D: angle about z
        float sn, cs;
        small_sincos(0.5f * __fmul_rn(mv.a, usym(b0.z)), mv.a, sn, cs);
        rotate_2d(qp.x, qp.w, sn, cs, A.qw, A.qz);
        A.qx = 0.0f; A.qy = 0.0f;
    } else {                                          // R6, 3-D: uniform axis, angle in [-a,a)
        const float zz = usym(b0.z);
        float sphi, cphi, sn, cs;
        sincosf(6.283185307179586f * u01(b0.w), &sphi, &cphi);
        const float rho = sqrtf(fmaxf(0.0f, 1.0f - zz * zz));
        sincosf(0.5f * __fmul_rn(mv.a, usym(uc)), &sn, &cs);
        const float dx = sn * rho * cphi, dy = sn * rho * sphi, dz = sn * zz, dw = cs;
        const float w = qp.x * dw - qp.y * dx - qp.z * dy - qp.w * dz;   // q (x) dq
        const float x = qp.x * dx + qp.y * dw + qp.z * dz - qp.w * dy;
        const float y = qp.x * dy - qp.y * dz + qp.z * dw + qp.w * dx;
        const float z = qp.x * dz + qp.y * dy - qp.z * dx + qp.w * dw;
        const float inv = rsqrtf(w * w + x * x + y * y + z * z);
        A.qw = w * inv; A.qx = x * inv; A.qy = y * inv; A.qz = z * inv;
    }
    return true;
}

// narrow phase of the trial particle A against neighbour B; r = r_B - r_A(trial), already minimum image
template <int KIND, int NV>
__device__ __forceinline__ bool narrow_overlap(const ShapeF& S, const ShapeD& SD, const TrialState& A, const float* MA, float rx,
                                               float ry, float rz, const double* rd, const float4& qB, float eps)
{
    if (KIND == kKindDisk) {
        return true;  // the broad phase already decided: |r|^2 < sigma^2
    } else if (KIND == kKindPolygon) {
        // 2-D orientation angle from q = (cos t/2, 0, 0, sin t/2): cos t = w^2 - z^2, sin t = 2wz
        const float cB = qB.x * qB.x - qB.w * qB.w, sB = 2.0f * qB.x * qB.w;
        return !polygon_separated<NV>(S, rx, ry, MA[0], MA[1], cB, sB, eps);
    } else {
        float MB[9];
        quat_to_matrix<float>(qB.x, qB.y, qB.z, qB.w, MB);
        int portal[3];
        const int verdict = polyhedron_classify<float>(S, MA, MB, V3<float>{rx, ry, rz}, eps, kGjkDeepF, portal);
        if (verdict != kGjkUnsure) return verdict == kGjkOverlap;
        // near contact: decide in fp64 from the raw fp32 state (mixed precision)
        return polyhedron_overlap_f64(SD, make_float4(A.qw, A.qx, A.qy, A.qz), qB, rd[0], rd[1], rd[2], (double)eps, portal);
    }
}

// Per-thread slow path: one thread makes the n_select trials of one active cell reading everything from global
// memory.  Used for 3-D systems and as the overflow fallback of the 2-D tile kernel.
struct CellCounters {
    unsigned int tacc = 0, trov = 0, trcell = 0, racc = 0, rrov = 0, trials = 0;
    unsigned int f64 = 0;    // polyhedron pairs decided by the fp64 re-run (diagnostic, counter slot 6)
    unsigned int nrot = 0;   // rotation trials (tile pass only: it derives trov / rrov from the totals when it flushes)
};

__device__ __forceinline__ void flush_counters(Control* ctrl, CellCounters c)
{
    // counters: warp reduce, one atomic per warp and counter
    c.tacc = __reduce_add_sync(0xffffffffu, c.tacc);
    c.trov = __reduce_add_sync(0xffffffffu, c.trov);
    c.trcell = __reduce_add_sync(0xffffffffu, c.trcell);
    c.racc = __reduce_add_sync(0xffffffffu, c.racc);
    c.rrov = __reduce_add_sync(0xffffffffu, c.rrov);
    c.trials = __reduce_add_sync(0xffffffffu, c.trials);
    c.f64 = __reduce_add_sync(0xffffffffu, c.f64);
    if ((threadIdx.x & 31) == 0 && c.trials) {
        unsigned long long* set = ctrl->counters[(blockIdx.x * 7u + (threadIdx.x >> 5)) & (kCounterSets - 1)];
        if (c.tacc) atomicAdd(&set[0], (unsigned long long)c.tacc);
        if (c.trov) atomicAdd(&set[1], (unsigned long long)c.trov);
        if (c.trcell) atomicAdd(&set[2], (unsigned long long)c.trcell);
        if (c.racc) atomicAdd(&set[3], (unsigned long long)c.racc);
        if (c.rrov) atomicAdd(&set[4], (unsigned long long)c.rrov);
        atomicAdd(&set[5], (unsigned long long)c.trials);
        if (c.f64) atomicAdd(&set[6], (unsigned long long)c.f64);
    }
}

template <int KIND, int NV>
__device__ void sweep_cell_global(const GridParams& g, const MoveParams& mv, const ShapeF& S, const ShapeD& SD, int gamma,
                                  uint32_t t_lo, uint32_t t_hi16, const float* shift, int cx, int cy, int cz,
                                  float4* __restrict__ pos, float4* __restrict__ quat, const int* __restrict__ tag,
                                  const int* __restrict__ cell_start, uint32_t k0, uint32_t k1, uint2* __restrict__ trace,
                                  CellCounters& cc)
{
    unsigned int c_tacc = 0, c_trov = 0, c_trcell = 0, c_racc = 0, c_rrov = 0, c_trials = 0;
    {
        const int cell = cx + g.n[0] * (cy + g.n[1] * cz);
        const int start = cell_start[cell], nmem = cell_start[cell + 1] - start;
        const long long slot0 = (long long)cell * mv.n_select;
        if (nmem == 0 || layer_inactive(g, g.dim == 3 ? cz : cy)) {
            if (trace)
                for (int k = 0; k < mv.n_select; ++k) trace[slot0 + k] = make_uint2(0u, 0u);
        } else {
            for (int k = 0; k < mv.n_select; ++k) {
                // a0: one Philox block per 2-D trial, two per 3-D trial (R3)
                const uint32_t c3 = (kTagTrial << 24) | ((uint32_t)gamma << 16) | t_hi16;
                const U4 b0 = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)k, c3, k0, k1);
                uint32_t uc = 0;
                if (g.dim == 3) uc = philox4x32_10((uint32_t)cell, t_lo, (uint32_t)k | (1u << 16), c3, k0, k1).x;
                // a5: uniformly random member (R8), move type (R7)
                const int p = start + (int)mulhi32(b0.x, (uint32_t)nmem);
                float4 xp, qp;
                load_state(g.dim, pos, quat, p, xp, qp);
                TrialState A;
                bool rotate;
                int outcome = make_trial<KIND>(g, mv, shift, cell, g.dim, b0, uc, xp, qp, A, rotate) ? 1 : 2;   // a5, a6
                ++c_trials;
                if (outcome == 1) {
                    // orientation data of the trial particle, computed once per trial
                    float MA[9];
                    if (KIND == kKindPolygon) {
                        MA[0] = A.qw * A.qw - A.qz * A.qz;
                        MA[1] = 2.0f * A.qw * A.qz;
                    } else if (KIND == kKindPolyhedron) {
                        quat_to_matrix<float>(A.qw, A.qx, A.qy, A.qz, MA);
                    }
                    // a7-a10: scan the 3^d cells around the owning cell (R19), early exit at the first overlap
                    const int zlo = (g.dim == 3) ? -1 : 0, zhi = (g.dim == 3) ? 1 : 0;
                    bool overlap = false;
                    for (int dz = zlo; dz <= zhi && !overlap; ++dz) {
                        int nz = cz + dz;
                        nz += (nz < 0) ? g.n[2] : 0;
                        nz -= (nz >= g.n[2]) ? g.n[2] : 0;
                        for (int dy = -1; dy <= 1 && !overlap; ++dy) {
                            int ny = cy + dy;
                            ny += (ny < 0) ? g.n[1] : 0;
                            ny -= (ny >= g.n[1]) ? g.n[1] : 0;
                            const int row = g.n[0] * (ny + g.n[1] * nz);
                            for (int dx = -1; dx <= 1 && !overlap; ++dx) {
                                int nx = cx + dx;
                                nx += (nx < 0) ? g.n[0] : 0;
                                nx -= (nx >= g.n[0]) ? g.n[0] : 0;
                                const int qs = cell_start[row + nx], qe = cell_start[row + nx + 1];
                                for (int q = qs; q < qe; ++q) {
                                    if (q == p) continue;
                                    const float4 xq = __ldcg(&pos[q]);   // 2-D: the pose (x, y, qw, qz)
                                    const float rx = min_image(xq.x, A.x, g.hi[0], g.Ld[0]);
                                    const float ry = min_image(xq.y, A.y, g.hi[1], g.Ld[1]);
                                    const float rz = (g.dim == 3) ? min_image(xq.z, A.z, g.hi[2], g.Ld[2]) : 0.0f;
                                    if (rx * rx + ry * ry + rz * rz >= S.dmax2) continue;   // a8 circumsphere (R16)
                                    float4 qq = make_float4(1.f, 0.f, 0.f, 0.f);
                                    if (KIND != kKindDisk) qq = (g.dim == 2) ? make_float4(xq.z, 0.f, 0.f, xq.w) : __ldcg(&quat[q]);
                                    double rd[3] = {0.0, 0.0, 0.0};
                                    if (KIND == kKindPolyhedron) {
                                        rd[0] = min_image_d(xq.x, A.x, g.Ld[0]);
                                        rd[1] = min_image_d(xq.y, A.y, g.Ld[1]);
                                        rd[2] = min_image_d(xq.z, A.z, g.Ld[2]);
                                    }
                                    if (narrow_overlap<KIND, NV>(S, SD, A, MA, rx, ry, rz, rd, qq, mv.eps_g)) {
                                        overlap = true;
                                        break;
                                    }
                                }
                            }
                        }
                    }
                    if (overlap) outcome = 3;
                }
                if (outcome == 1) {   // a11: wrap with one fp32 add if needed, write back in place
                    float x = A.x, y = A.y, z = A.z;
                    if (x >= g.hi[0]) x = __fsub_rn(x, g.L[0]); else if (x < g.lo[0]) x = __fadd_rn(x, g.L[0]);
                    if (y >= g.hi[1]) y = __fsub_rn(y, g.L[1]); else if (y < g.lo[1]) y = __fadd_rn(y, g.L[1]);
                    if (g.dim == 3) { if (z >= g.hi[2]) z = __fsub_rn(z, g.L[2]); else if (z < g.lo[2]) z = __fadd_rn(z, g.L[2]); }
                    store_state(g.dim, pos, quat, p, make_float4(x, y, z, xp.w), make_float4(A.qw, A.qx, A.qy, A.qz), rotate);
                    if (rotate) ++c_racc; else ++c_tacc;
                } else if (outcome == 2) {
                    ++c_trcell;
                } else {
                    if (rotate) ++c_rrov; else ++c_trov;
                }
                if (trace) trace[slot0 + k] = make_uint2((uint32_t)tag[p], (rotate ? 1u : 0u) | ((uint32_t)outcome << 8));
            }
        }
    }
    cc.tacc += c_tacc; cc.trov += c_trov; cc.trcell += c_trcell; cc.racc += c_racc; cc.rrov += c_rrov; cc.trials += c_trials;
}

// v1 mapping: one thread per active cell (any dimension).
template <int KIND, int NV>
__global__ void __launch_bounds__(128)
k_sweep_colour(const __grid_constant__ GridParams g, const __grid_constant__ MoveParams mv,
               const __grid_constant__ ShapeF S, const __grid_constant__ ShapeD SD, Control* __restrict__ ctrl, int colour_index,
               float4* __restrict__ pos, float4* __restrict__ quat, const int* __restrict__ tag,
               const int* __restrict__ cell_start, uint32_t k0, uint32_t k1, uint2* __restrict__ trace)
{
    const SweepHeader& H = ctrl->hdr;
    const int gamma = H.perm[colour_index];
    const float shift[3] = {H.shift[0], H.shift[1], H.shift[2]};
    const int nax = g.n[0] >> 1, nay = g.n[1] >> 1, naz = (g.dim == 3) ? (g.n[2] >> 1) : 1;
    const int nactive = nax * nay * naz;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    CellCounters cc;
    if (idx < nactive) {
        const int ix = idx % nax, iy = (idx / nax) % nay, iz = idx / (nax * nay);
        const int cx = 2 * ix + (gamma & 1), cy = 2 * iy + ((gamma >> 1) & 1), cz = (g.dim == 3) ? 2 * iz + ((gamma >> 2) & 1) : 0;
        sweep_cell_global<KIND, NV>(g, mv, S, SD, gamma, H.t_lo, H.t_hi16, shift, cx, cy, cz, pos, quat, tag, cell_start, k0, k1,
                                    trace, cc);
    }
    flush_counters(ctrl, cc);
}

// a12: count pairs (tag_p < tag_q) in 3^d neighbourhoods whose interiors intersect (strict, fp64).
// Runs on a cell list built with zero shift (k_prepare mode 2).
template <int KIND>
__global__ void __launch_bounds__(128)
k_count_overlaps(const __grid_constant__ GridParams g, const __grid_constant__ ShapeD S, Control* __restrict__ ctrl,
                 const float4* __restrict__ pos, const float4* __restrict__ quat, const int* __restrict__ tag,
                 const int* __restrict__ cell_start)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int found = 0;
    if (p < g.N) {
        const float shift[3] = {ctrl->hdr.shift[0], ctrl->hdr.shift[1], ctrl->hdr.shift[2]};
        float4 xp, qp;
        load_state(g.dim, pos, quat, p, xp, qp);
        const int tp = tag[p];
        int cx, cy, cz;
        cell_of(g, shift, xp.x, xp.y, xp.z, cx, cy, cz);
        double MA[9];
        double cA = 1.0, sA = 0.0;
        {
            const double nq = sqrt((double)qp.x * qp.x + (double)qp.y * qp.y + (double)qp.z * qp.z + (double)qp.w * qp.w);
            const double w = qp.x / nq, x = qp.y / nq, y = qp.z / nq, z = qp.w / nq;
            if (KIND == kKindPolygon) { cA = w * w - z * z; sA = 2.0 * w * z; }
            if (KIND == kKindPolyhedron) quat_to_matrix<double>(w, x, y, z, MA);
        }
        const int zlo = (g.dim == 3) ? -1 : 0, zhi = (g.dim == 3) ? 1 : 0;
        for (int dz = zlo; dz <= zhi; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    const int nx = (cx + dx + g.n[0]) % g.n[0], ny = (cy + dy + g.n[1]) % g.n[1], nz = (cz + dz + g.n[2]) % g.n[2];
                    const int c2 = nx + g.n[0] * (ny + g.n[1] * nz);
                    for (int q = cell_start[c2]; q < cell_start[c2 + 1]; ++q) {
                        if (tag[q] <= tp) continue;
                        float4 xq, qq;
                        load_state(g.dim, pos, quat, q, xq, qq);
                        double r[3] = {(double)xq.x - (double)xp.x, (double)xq.y - (double)xp.y, (double)xq.z - (double)xp.z};
                        for (int k = 0; k < g.dim; ++k) {
                            if (r[k] > 0.5 * g.Ld[k]) r[k] -= g.Ld[k];
                            else if (r[k] < -0.5 * g.Ld[k]) r[k] += g.Ld[k];
                        }
                        if (g.dim == 2) r[2] = 0.0;
                        const double d2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
                        if (d2 >= S.dmax2) continue;
                        bool ov = true;
                        if (KIND != kKindDisk) {
                            const double nq = sqrt((double)qq.x * qq.x + (double)qq.y * qq.y + (double)qq.z * qq.z + (double)qq.w * qq.w);
                            const double w = qq.x / nq, x = qq.y / nq, y = qq.z / nq, z = qq.w / nq;
                            if (KIND == kKindPolygon) {
                                ov = polygon_overlap<double, 0>(S, r[0], r[1], cA, sA, w * w - z * z, 2.0 * w * z, 0.0);
                            } else {
                                double MB[9];
                                quat_to_matrix<double>(w, x, y, z, MB);
                                int unused[3];
                                ov = polyhedron_classify<double>(S, MA, MB, V3<double>{r[0], r[1], r[2]}, 0.0, 0.0, unused) != kGjkSeparated;
                            }
                        }
                        if (ov) ++found;
                    }
                }
    }
    found = __reduce_add_sync(0xffffffffu, found);
    if ((threadIdx.x & 31) == 0 && found) atomicAdd(&ctrl->overlaps, (unsigned long long)found);
}

}  // namespace hpmc
