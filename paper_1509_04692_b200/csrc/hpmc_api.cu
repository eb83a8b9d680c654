// C-ABI of libhpmc.so (include/hpmc.h): host-side context, validation, workspace carving and the launch
// sequence of one sweep.  Every step of the hot path runs in the kernels of cell_list.cuh / sweep.cuh.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/hpmc.h"
#include "cell_list.cuh"
#include "common.cuh"
#include "dist.cuh"
#include "overlap.cuh"
#include "sweep.cuh"
#include "ctx.hpp"

using namespace hpmc;

// Pure-FMA microkernel for the measured FP32 roofline denominator (S:8(d): "time a pure-FMA microkernel in the same run"):
// kFmaChains independent dependent-FMA chains per thread, no memory traffic but one store that keeps the result alive.
constexpr int kFmaChains = 16;
__global__ void __launch_bounds__(256) k_fma_peak(float* sink, int iters, float a)
{
    float x[kFmaChains];
#pragma unroll
    for (int j = 0; j < kFmaChains; ++j) x[j] = 1.0f + 1e-3f * (float)(threadIdx.x + j);
    const float b = 1e-6f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < kFmaChains; ++j) x[j] = fmaf(x[j], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kFmaChains; ++j) s += x[j];
    if (s == 123.456f) *sink = s;   // never true: keeps the chains alive without a store per thread
}

namespace {

thread_local std::string g_err_noctx;

int fail(hpmc_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg;
    else g_err_noctx = msg;
    return code;
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes)
    {
        const size_t o = off;
        off = align_up(off + bytes, 256);
        return o;
    }
};

int scan_tiles(const hpmc_ctx* c) { return (c->g.C + 1 + kScanTile - 1) / kScanTile; }

// `done` stamps of the 2-D dataflow pass: 4 colours x tiles of the smallest tile shape (2 rows of 32 active cells)
size_t flow_words(const hpmc_ctx* c)
{
    if (c->g.dim != 2) return 1;
    const size_t nax = c->g.n[0] / 2, nay = c->g.n[1] / 2;
    return 4 * ((nax + kTileWHost - 1) / kTileWHost) * ((nay + 1) / 2) + 4;
}

struct Layout {
    size_t pos[2], quat[2], tag[2], key_rank, cell_start, counts, arrived, tile_sums, flow_done, ctrl, inactive, total;
};

Layout layout_of(const hpmc_ctx* c)
{
    Layout L{};
    Carve cv;
    const size_t N = (size_t)(c->n_cap > 0 ? c->n_cap : 1);
    for (int b = 0; b < 2; ++b) {
        L.pos[b] = cv.take(N * sizeof(float4));
        L.quat[b] = cv.take(c->g.dim == 3 ? N * sizeof(float4) : 0);   // 2-D keeps one pose array
        L.tag[b] = cv.take(N * sizeof(int));
    }
    L.key_rank = cv.take(N * sizeof(int2));
    L.cell_start = cv.take(((size_t)c->g.C + 2) * sizeof(int));
    L.counts = cv.take(((size_t)c->g.C + 2) * sizeof(int));
    L.arrived = cv.take(((size_t)c->g.C + 2) * sizeof(int));
    L.tile_sums = cv.take((size_t)(scan_tiles(c) + 1) * sizeof(int));
    L.flow_done = cv.take(flow_words(c) * sizeof(unsigned int));
    L.ctrl = cv.take(sizeof(Control));
    L.inactive = cv.take((size_t)c->g.n[c->g.dim - 1]);   // inactive-region mask, one byte per layer of cells along the last axis
    L.total = cv.off;
    return L;
}

// host-side shape validation and derived data (convexity, CCW, edge normals); fp64 then rounded for ShapeF
int build_shape(hpmc_ctx* c, const hpmc_shape* s, int dim)
{
    ShapeD& D = c->sd;
    std::memset(&D, 0, sizeof D);
    D.kind = s->kind;
    if (s->kind == HPMC_KIND_DISK) {
        if (!(s->diameter > 0.0)) return fail(c, HPMC_E_SHAPE, "disk diameter must be > 0");
        D.diameter = s->diameter;
        c->d_max = s->diameter;
    } else if (s->kind == HPMC_KIND_POLYGON || s->kind == HPMC_KIND_POLYHEDRON) {
        const bool poly2 = s->kind == HPMC_KIND_POLYGON;
        if ((poly2 && dim != 2) || (!poly2 && dim != 3)) return fail(c, HPMC_E_SHAPE, "polygon needs dim 2, polyhedron dim 3");
        if (!s->verts || s->nverts < (poly2 ? 3 : 4) || s->nverts > HPMC_MAX_VERTS)
            return fail(c, HPMC_E_SHAPE, "vertex count out of range");
        const int nv = s->nverts, vd = poly2 ? 2 : 3;
        D.nverts = nv;
        double rmax = 0.0;
        for (int i = 0; i < nv; ++i) {
            D.vx[i] = s->verts[i * vd];
            D.vy[i] = s->verts[i * vd + 1];
            D.vz[i] = poly2 ? 0.0 : s->verts[i * vd + 2];
            rmax = std::fmax(rmax, std::sqrt(D.vx[i] * D.vx[i] + D.vy[i] * D.vy[i] + D.vz[i] * D.vz[i]));
        }
        const double rho = s->sweep_radius;   // rounded shapes (spheropolygons / spheropolyhedra)
        if (!(rho >= 0.0) || !std::isfinite(rho)) return fail(c, HPMC_E_SHAPE, "sweep_radius must be finite and >= 0");
        D.sweep = 2.0 * rho;
        c->d_max = 2.0 * (rmax + rho);  // circumsphere centred on the particle position
        double r_in = 1e300;    // inscribed radius about the body origin = smallest face/edge offset
        if (poly2) {
            // regular n-gon centred on the origin: equal radii and equal angular steps (see polygon_separated)
            bool regular = true;
            for (int k = 0; k < nv; ++k) {
                const int k1 = (k + 1) % nv;
                const double rk = std::hypot(D.vx[k], D.vy[k]);
                const double cs = (D.vx[k] * D.vx[k1] + D.vy[k] * D.vy[k1]) / (rmax * rmax);
                if (std::fabs(rk - rmax) > 1e-12 * rmax || std::fabs(cs - std::cos(2.0 * 3.14159265358979323846 / nv)) > 1e-12) regular = false;
            }
            D.regular = regular ? 1 : 0;
            for (int k = 0; k < nv; ++k) {
                const int k1 = (k + 1) % nv, k2 = (k + 2) % nv;
                const double ex = D.vx[k1] - D.vx[k], ey = D.vy[k1] - D.vy[k];
                const double fx = D.vx[k2] - D.vx[k1], fy = D.vy[k2] - D.vy[k1];
                if (!(ex * fy - ey * fx > 0.0)) return fail(c, HPMC_E_SHAPE, "polygon must be strictly convex with CCW vertices");
                const double len = std::sqrt(ex * ex + ey * ey);
                D.nx[k] = ey / len;
                D.ny[k] = -ex / len;
                D.fc[k] = D.nx[k] * D.vx[k] + D.ny[k] * D.vy[k];
                if (!(D.fc[k] > 0.0)) return fail(c, HPMC_E_SHAPE, "the body-frame origin must be inside the polygon");
                r_in = std::fmin(r_in, D.fc[k]);
            }
        } else {
            // every vertex must be an extreme point and the origin must be interior: for each vertex v there
            // must be a direction (here: tested with the vertex direction itself and all pair/triple normals)
            // -- brute force over supporting planes through vertex triples.
            int on_hull[HPMC_MAX_VERTS] = {0};
            int nplanes = 0;
            for (int i = 0; i < nv; ++i)
                for (int j = i + 1; j < nv; ++j)
                    for (int k = j + 1; k < nv; ++k) {
                        const double e1[3] = {D.vx[j] - D.vx[i], D.vy[j] - D.vy[i], D.vz[j] - D.vz[i]};
                        const double e2[3] = {D.vx[k] - D.vx[i], D.vy[k] - D.vy[i], D.vz[k] - D.vz[i]};
                        double n[3] = {e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0]};
                        const double len = std::sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
                        if (len < 1e-12) continue;
                        for (double& x : n) x /= len;
                        const double off = n[0] * D.vx[i] + n[1] * D.vy[i] + n[2] * D.vz[i];
                        int npos = 0, nneg = 0;
                        for (int l = 0; l < nv; ++l) {
                            const double dd = n[0] * D.vx[l] + n[1] * D.vy[l] + n[2] * D.vz[l] - off;
                            npos += dd > 1e-9;
                            nneg += dd < -1e-9;
                        }
                        if (npos && nneg) continue;
                        ++nplanes;
                        r_in = std::fmin(r_in, std::fabs(off));
                        // origin strictly inside: on the same side as the other vertices, off the plane
                        const double o = -off;  // n.0 - off
                        if ((npos && !(o > 1e-12)) || (nneg && !(o < -1e-12)))
                            return fail(c, HPMC_E_SHAPE, "the body-frame origin must be inside the polyhedron");
                        for (int l = 0; l < nv; ++l)
                            if (std::fabs(n[0] * D.vx[l] + n[1] * D.vy[l] + n[2] * D.vz[l] - off) < 1e-9) on_hull[l]++;
                    }
            if (nplanes < 4) return fail(c, HPMC_E_SHAPE, "degenerate polyhedron");
            for (int l = 0; l < nv; ++l)
                if (on_hull[l] < 3) return fail(c, HPMC_E_SHAPE, "every vertex must be a hull vertex (convex polyhedron)");
        }
        const double din = std::fmax(0.0, 2.0 * (r_in + rho) - 1e-5);   // the rounded shape holds the ball of radius r_in + rho
        D.din2 = din * din;
        D.rin = r_in;
    } else
        return fail(c, HPMC_E_SHAPE, "unknown shape kind");
    D.dmax2 = c->d_max * c->d_max;  // the validator is strict: no guard band
    ShapeF& F = c->sf;
    std::memset(&F, 0, sizeof F);
    F.kind = D.kind;
    F.nverts = D.nverts;
    F.diameter = (float)D.diameter;
    F.din2 = (float)D.din2;
    F.rin = (float)(D.rin * (1.0 - 1e-6));   // rounded DOWN: the candidate-axis test of polygon_separated must never exclude an axis that separates
    F.regular = D.regular;
    F.sweep = (float)D.sweep;
    for (int i = 0; i < kMaxVerts; ++i) {
        F.vx[i] = (float)D.vx[i]; F.vy[i] = (float)D.vy[i]; F.vz[i] = (float)D.vz[i];
        F.nx[i] = (float)D.nx[i]; F.ny[i] = (float)D.ny[i]; F.fc[i] = (float)D.fc[i];
    }
    return HPMC_OK;
}

void refresh_sweep_range(hpmc_ctx* c)
{
    // broad-phase range of the sweep includes the guard band (R16'): skip iff |r|^2 >= (d_max + eps_g)^2
    const double rr = c->d_max + (double)c->mv.eps_g;
    c->sf.dmax2 = (float)(rr * rr);
}

// fold the recorded event pairs into the per-class sums (synchronises the stream)
bool profile_fold(hpmc_ctx* c)
{
    if (c->ev_class.empty()) return true;
    if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "profile/sync")) return false;
    for (size_t i = 0; i < c->ev_class.size(); ++i) {
        float ms = 0.f;
        if (!cuda_ok(c, cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]), "profile/elapsed")) return false;
        c->prof_ms[c->ev_class[i] & 15] += (double)ms;
        c->prof_n[c->ev_class[i] & 15] += c->ev_class[i] >> 4;   // a bracket may cover several colour passes (dataflow launch)
    }
    c->ev_class.clear();
    c->ev_used = 0;
    return true;
}

struct ProfileScope {
    hpmc_ctx* c;
    bool on;
    ProfileScope(hpmc_ctx* ctx, int cls, int weight = 1) : c(ctx), on(ctx->profile && !ctx->cuda_failed)
    {
        if (!on) return;
        if (c->ev_class.size() >= 4096) profile_fold(c);
        while (c->ev_pool.size() < c->ev_used + 2) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) { on = false; return; }
            c->ev_pool.push_back(e);
        }
        c->ev_class.push_back(cls | (weight << 4));
        cudaEventRecord(c->ev_pool[c->ev_used], c->stream);
    }
    ~ProfileScope()
    {
        if (!on) return;
        cudaEventRecord(c->ev_pool[c->ev_used + 1], c->stream);
        c->ev_used += 2;
    }
};

#define LAUNCH_CHECK(c, what)                                      \
    do {                                                           \
        ++(c)->launches;                                           \
        if (!cuda_ok((c), cudaGetLastError(), what)) return HPMC_E_CUDA; \
    } while (0)

// build the cell list of the current state into buffer 1-cur and flip.  mode as in k_prepare.
int build_cell_list(hpmc_ctx* c, int mode, unsigned long long t_override)
{
    ProfileScope prof(c, 0);
    c->after_colour = false;
    const GridParams& g = c->g;
    const int TB = 256;
    const float4* src_pos = c->state_in_bound ? c->d_pos_bound : c->pos[c->cur];
    const float4* src_quat = c->state_in_bound ? c->d_quat_bound : c->quat[c->cur];
    const int* src_tag = c->state_in_bound ? nullptr : c->tag[c->cur];
    const int dst = c->state_in_bound ? 0 : 1 - c->cur;
    if (c->opt_small_build && g.C <= kSmallBuildMaxCells && g.N <= kSmallBuildMaxN) {   // one CTA does the whole build
        hpmc_launch(c, k_build_small, 1, kSmallBuildThreads, ((size_t)g.C + 2) * sizeof(int),
            g, c->ctrl, c->k0, c->k1, mode, t_override, src_pos, src_quat, src_tag, c->key_rank, c->cell_start, c->pos[dst], c->quat[dst],
            c->tag[dst]);
        LAUNCH_CHECK(c, "k_build_small");
        c->cur = dst;
        c->state_in_bound = false;
        c->have_sorted = true;
        c->cell_valid = true;
        return HPMC_OK;
    }
    const int nblk_part = (g.N + TB - 1) / TB;
    const int nblk_hist = (g.N + TB * kHistItems - 1) / (TB * kHistItems);
    hpmc_launch(c, k_hist, nblk_hist > 0 ? nblk_hist : 1, TB, 0, g, c->ctrl, src_pos, c->counts, c->key_rank, c->k0, c->k1, mode, t_override);
    LAUNCH_CHECK(c, "k_hist");
    const int tiles = scan_tiles(c);
    const bool fused = tiles > 1 && tiles <= kFusedSpineMax;
    if (tiles > 1) {
        hpmc_launch(c, k_scan_reduce, tiles, kScanThreads, 0, c->counts, g.C, c->tile_sums);
        LAUNCH_CHECK(c, "k_scan_reduce");
        if (!fused) {
            hpmc_launch(c, k_scan_spine, 1, kScanThreads, 0, c->tile_sums, tiles, c->ctrl, mode);
            LAUNCH_CHECK(c, "k_scan_spine");
        }
    }
    hpmc_launch(c, k_scan_final, tiles, kScanThreads, 0, c->counts, g.C, c->cell_start, c->tile_sums, tiles == 1 ? 1 : fused ? 2 : 0, c->ctrl, mode);
    LAUNCH_CHECK(c, "k_scan_final");
    if (g.N > 0) {
        hpmc_launch(c, k_scatter, nblk_part, TB, 0, g.N, g.dim, src_pos, src_quat, src_tag, c->key_rank, c->cell_start, c->pos[dst], c->quat[dst],
                                                  c->tag[dst]);
        LAUNCH_CHECK(c, "k_scatter");
        if (g.dim == 3) hpmc_launch(c, k_sort_cells<3>, (g.C + TB - 1) / TB, TB, 0, g.C, c->cell_start, c->pos[dst], c->quat[dst], c->tag[dst]);
        else hpmc_launch(c, k_sort_cells<2>, (g.C + TB - 1) / TB, TB, 0, g.C, c->cell_start, c->pos[dst], c->quat[dst], c->tag[dst]);
        LAUNCH_CHECK(c, "k_sort_cells");
    }
    c->cur = dst;
    c->state_in_bound = false;
    c->have_sorted = true;
    c->cell_valid = true;
    return HPMC_OK;
}

// tile shapes (warps per CTA, rows of 32 active cells per warp); "tile_shape" option, 0 = by grid size
int pick_tile_shape(const hpmc_ctx* c)
{
    if (c->opt_tile_shape) return c->opt_tile_shape;
    const int nax = c->g.n[0] / 2, nay = c->g.n[1] / 2;
    const long long cols = (nax + kTileWHost - 1) / kTileWHost;
    // 4 warps x 1 row (64 registers, 8 CTAs per SM) once its tiles of one colour nearly fill the machine; below that the 2-warp
    // tile spreads a colour over twice as many CTAs (measured on B200, pentagons, n x n lattice: 448 / 512 / 640 -> 2 warps
    // +11 / +16 / +7 %; 768 and above -> 4 warps +13 % and more)
    if (cols * ((nay + 3) / 4) * 32 >= (long long)c->num_sms * 8 * 27) return 2;
    return 3;                                            // 2 warps x 1 row
}

// active rows of cells per tile of each shape (Tile2D<WARPS, R>::TH)
int tile_rows(int shape) { return shape == 1 ? 16 : shape == 2 ? 4 : 2; }

// 2-D systems with fewer active cells per colour than this run one warp per cell instead of one lane per cell: the tile
// kernel would leave most SMs idle (config 1: 961 active cells = 31 warps) and each warp round would be a long serial chain
constexpr int kWarpCellMax2d = 148 * 48;

// 2-D systems: the speculative warp-per-cell pass (sweep_spec2d.cuh), on request only.  Measured on B200 (4096 pentagons): a
// batch of four trials takes 4.4 us against 4 x 1.05 us for the sequential warp-per-cell pass -- every phase of the decision
// tree (replay, 15 x candidates broad phase, queue, tree walk) is itself a few hundred dependent instructions on a lone warp
bool use_spec(const hpmc_ctx* c)
{
    const GridParams& g = c->g;
    if (g.dim != 2 || c->sf.kind == kKindPolyhedron || c->part_n > 1) return false;
    return c->opt_path == 5;
}

// does the 2-D tile pass apply (not the warp-per-cell pass, not the per-thread path), and as a dataflow launch?
bool use_flow(const hpmc_ctx* c)
{
    const GridParams& g = c->g;
    if (g.dim != 2 || c->sf.kind == kKindPolyhedron || c->opt_path == 1 || c->opt_path == 3 || c->opt_path == 5 || c->opt_flow == 0) return false;
    if (c->part_n > 1) return false;   // the ranks exchange boundary rows between the colours: one launch per colour
    const int nactive = (g.n[0] / 2) * (g.n[1] / 2);
    if (c->opt_path == 0 && c->opt_tile_shape == 0 && nactive <= kWarpCellMax2d) return false;
    if (c->opt_flow == 1) return true;
    // auto: the dataflow launch pays when a colour is one to a few waves of tiles (measured on B200: +9 % at 1M pentagons,
    // 1.7 waves; slower below one wave, where the stamps only add latency; no difference from 4M up)
    const long long slots = (long long)c->num_sms * 8;
    const int rows = tile_rows(pick_tile_shape(c));
    const long long tiles = (long long)((g.n[0] / 2 + kTileWHost - 1) / kTileWHost) * ((g.n[1] / 2 + rows - 1) / rows);
    return c->opt_tile_shape == 0 && tiles > slots && tiles <= 4 * slots;
}

// Whole-sweep cluster pass (sweep_cluster2d.cuh): 2-D disks / polygons small enough for one cluster of 16 x 1024 threads
// (one thread per particle in its build) and for a cell_start copy in every CTA's shared memory.
constexpr int kClusterMaxCtas = 16, kClusterThreads = 1024, kClusterMaxCells = 11500;
bool cluster_eligible(const hpmc_ctx* c)
{
    const GridParams& g = c->g;
    if (g.dim != 2 || c->sf.kind == kKindPolyhedron || c->cluster_ctas == 0 || c->part_n > 1 || g.inactive) return false;
    if (g.N < 1 || g.N > kClusterMaxCtas * kClusterThreads || g.C + 2 > kClusterMaxCells) return false;
    // measured on B200 (profiles/r2_cluster.md): 58 us per sweep of 4096 pentagons against 39 us for the graph of five launches --
    // a trial is a ~2 us dependent chain either way and seven cluster barriers do not beat four launch gaps -- so the pass is
    // chosen only on request
    return c->opt_path == 4;
}

// n sweeps through the cluster pass; returns the sweeps done (0: not available here, the caller uses the other passes)
int64_t sweep_cluster(hpmc_ctx* c, int64_t n)
{
    const int kind = c->sf.kind;
    const int nv = (kind == kKindPolygon && c->sf.nverts == 5 && c->sf.regular && c->sd.sweep == 0.0) ? 5 : 0;
    int64_t done = 0;
    while (done < n) {
        const int64_t want = std::min<int64_t>(n - done, 1 << 20);   // sweeps per launch
        int got = 0;
        {
            ProfileScope prof(c, 1, (int)(4 * want));   // timed as 4 colour passes per sweep (the build is inside the launch)
            if (c->cluster_ctas < 0) {   // first use: the largest cluster this device schedules that covers the particles
                for (int ncta = kClusterMaxCtas; ncta >= 1 && c->cluster_ctas < 0; ncta >>= 1) {
                    if (ncta * kClusterThreads < c->g.N) break;
                    got = hpmc_launch_cluster2d(c, want, ncta, kind, nv);
                    if (got < 0) return -1;
                    if (got > 0) c->cluster_ctas = ncta;
                }
                if (c->cluster_ctas < 0) { c->cluster_ctas = 0; prof.on = false; return done; }
            } else {
                got = hpmc_launch_cluster2d(c, want, c->cluster_ctas, kind, nv);
                if (got <= 0) return -1;
            }
        }
        ++c->launches;
        c->cur ^= (got & 1);
        c->t_host += (uint64_t)got;
        done += got;
    }
    return done;
}

int launch_colour_dispatch(hpmc_ctx* c, int ci)
{
    c->flow_now = use_flow(c);
    if (c->flow_now && ci > 0) return HPMC_OK;   // colour 0's dataflow launch covers all four colours
    ProfileScope prof(c, 1, c->flow_now ? 4 : 1);
    // the (kind, unrolled vertex count) variants of each pass are compiled in separate translation units (pass_*.cu)
    const int kind = c->sf.kind;
    const bool sharp = c->sd.sweep == 0.0;   // rounded shapes take the runtime-vertex-count kernels (overlap.cuh)
    const int nvp = c->sf.nverts;             // polyhedra with 8, 20 or 24 vertices have unrolled support functions
    const int nv = (kind == kKindPolygon && nvp == 5 && c->sf.regular && sharp) ? 5
                   : (kind == kKindPolyhedron && sharp && (nvp == 8 || nvp == 20 || nvp == 24)) ? nvp : 0;
    const GridParams& g = c->g;
    const int nactive = (g.n[0] / 2) * (g.n[1] / 2) * (g.dim == 3 ? g.n[2] / 2 : 1);
    bool ok = true;
    if (c->part_n > 1) ok = hpmc_launch_tile2d(c, ci, kind, nv, pick_tile_shape(c));
    else if (c->opt_path == 1 || (g.dim == 2 && kind == kKindPolyhedron)) ok = hpmc_launch_colour(c, ci, kind, nv, nactive);
    else if (use_spec(c)) ok = hpmc_launch_spec2d(c, ci, kind, nv, nactive);
    else if (g.dim == 3 || c->opt_path == 3 || (c->opt_path == 0 && c->opt_tile_shape == 0 && nactive <= kWarpCellMax2d))
        ok = hpmc_launch_warpcell(c, ci, kind, nv, nactive);
    else ok = hpmc_launch_tile2d(c, ci, kind, nv, pick_tile_shape(c));
    if (!ok) return HPMC_E_CUDA;
    LAUNCH_CHECK(c, "colour pass");
    c->after_colour = !c->profile;   // an event record between the launches makes the next one an ordinary successor anyway
    return HPMC_OK;
}

// one sweep: shift + cell list + the colours in the sweep's random order (S:8(a) rows a0-a11)
int sweep_once(hpmc_ctx* c)
{
    int rc = build_cell_list(c, 0, 0ull);
    if (rc != HPMC_OK) return rc;
    const int ncol = 1 << c->g.dim;
    for (int ci = 0; ci < ncol; ++ci) {
        rc = launch_colour_dispatch(c, ci);
        if (rc != HPMC_OK) return rc;
    }
    ++c->t_host;
    return HPMC_OK;
}

// anything the captured launches depend on changed: pointers, move sizes, options, trace
void graph_reset(hpmc_ctx* c)
{
    for (int b = 0; b < 2; ++b)
        if (c->graph_exec[b]) { cudaGraphExecDestroy(c->graph_exec[b]); c->graph_exec[b] = nullptr; }
}

int check_ready(hpmc_ctx* c)
{
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (!c->d_ws || (!c->have_sorted && !c->state_in_bound)) return fail(c, HPMC_E_UNBOUND, "state/workspace not bound");
    return HPMC_OK;
}

}  // namespace

extern "C" {

int hpmc_create(const hpmc_box* box, const hpmc_shape* shape, int64_t N, uint64_t seed, void* cuda_stream, hpmc_ctx** out)
{
    if (!out) return fail(nullptr, HPMC_E_ARG, "out is NULL");
    *out = nullptr;
    if (!box || !shape) return fail(nullptr, HPMC_E_ARG, "box/shape is NULL");
    if (box->dim != 2 && box->dim != 3) return fail(nullptr, HPMC_E_ARG, "dim must be 2 or 3");
    if (N < 0 || N > 2147483000LL) return fail(nullptr, HPMC_E_ARG, "N out of range");
    hpmc_ctx* c = new (std::nothrow) hpmc_ctx();
    if (!c) return fail(nullptr, HPMC_E_ARG, "out of host memory");
    int rc = build_shape(c, shape, box->dim);
    if (rc != HPMC_OK) { g_err_noctx = c->err; delete c; return rc; }
    GridParams& g = c->g;
    g.dim = box->dim;
    g.N = (int)N;
    c->n_cap = (int)N;
    double cells = 1.0;
    for (int k = 0; k < 3; ++k) {
        if (k < g.dim) {
            if (!(box->L[k] > 0.0)) { delete c; return fail(nullptr, HPMC_E_ARG, "box edge must be > 0"); }
            g.L[k] = (float)box->L[k];            // R-box: the box edge is L rounded to fp32
            g.Ld[k] = (double)g.L[k];
            {   // R11: even count, cell width >= d_max + slack.  The slack is d_max 2^-10, or -- in boxes so large that this is
                // not enough -- 3 ulp_fp32(L): fl(fl(x - lo) - s) * inv_w misplaces a cell boundary by up to ~1.5 ulp of a
                // coordinate difference just below L, and two boundaries lie between particles of cells c and c + 2, which
                // must stay >= d_max apart (R22).  Identical to the plain 2^-10 rule up to L ~ 5000 d_max.
                int e = 0;
                std::frexp(std::nextafter(g.Ld[k], 0.0), &e);     // the largest coordinate difference below L = m 2^e, m in [0.5, 1)
                const double ulp = std::ldexp(1.0, e - 24);      // fp32 ulp of values in [L/2, L)
                const double slack = std::fmax(c->d_max / 1024.0, 3.0 * ulp);
                g.n[k] = 2 * (int)std::floor(g.Ld[k] / (2.0 * (c->d_max + slack)));
            }
            if (g.n[k] < 4) { delete c; return fail(nullptr, HPMC_E_GRID, "fewer than 4 cells per side (R11)"); }
            c->w[k] = g.Ld[k] / g.n[k];
            g.w_f[k] = (float)c->w[k];
            g.inv_w[k] = (float)((double)g.n[k] / g.Ld[k]);
        } else {
            g.L[k] = 1.0f; g.Ld[k] = 1.0; g.n[k] = 1; g.w_f[k] = 1.0f; g.inv_w[k] = 1.0f; c->w[k] = 1.0;
        }
        g.hi[k] = 0.5f * g.L[k];
        g.lo[k] = -g.hi[k];
        cells *= g.n[k];
    }
    if (cells > 2147483000.0) { delete c; return fail(nullptr, HPMC_E_GRID, "too many cells for 32-bit ids"); }
    g.C = (int)cells;
    c->seed = seed;
    c->k0 = (uint32_t)seed;
    c->k1 = (uint32_t)(seed >> 32);
    for (uint32_t r = 0; r < 10; ++r) {   // Philox round keys (philox4x32_10_rk)
        g.philox_rk[2 * r] = c->k0 + r * kPhiloxW0;
        g.philox_rk[2 * r + 1] = c->k1 + r * kPhiloxW1;
    }
    c->stream = (cudaStream_t)cuda_stream;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess) c->num_sms = sms;
        c->device = dev;
        if (c->num_sms <= 0) c->num_sms = 148;   // no device visible (CPU-side ABI checks): B200
    }
    c->mv.d = 0.1f; c->mv.a = 0.1f; c->mv.n_select = 4; c->mv.eps_g = 2e-6f;  // R15
    refresh_sweep_range(c);
    *out = c;
    return HPMC_OK;
}

int hpmc_destroy(hpmc_ctx* c)
{
    if (c) {
        graph_reset(c);
        for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    }
    delete c;
    return HPMC_OK;
}

const char* hpmc_last_error(const hpmc_ctx* c) { return c ? c->err.c_str() : g_err_noctx.c_str(); }

int hpmc_get_grid(const hpmc_ctx* c, hpmc_grid_info* o)
{
    if (!c || !o) return HPMC_E_ARG;
    o->dim = c->g.dim;
    for (int k = 0; k < 3; ++k) { o->n[k] = c->g.n[k]; o->w[k] = c->w[k]; o->L_f[k] = c->g.L[k]; o->inv_w[k] = c->g.inv_w[k]; }
    o->d_max = c->d_max;
    o->num_cells = c->g.C;
    o->N = c->g.N;
    return HPMC_OK;
}

// the host copy of the inactive-region mask -> its slot in the workspace; g.inactive stays NULL while no layer is flagged
static int upload_inactive(hpmc_ctx* c)
{
    bool any = false;
    for (unsigned char b : c->inactive_h) any = any || b != 0;
    c->g.inactive = nullptr;
    if (!any || !c->d_inactive) return HPMC_OK;
    if (!cuda_ok(c, cudaMemcpyAsync(c->d_inactive, c->inactive_h.data(), c->inactive_h.size(), cudaMemcpyHostToDevice, c->stream), "inactive/memcpy"))
        return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "inactive/sync")) return HPMC_E_CUDA;
    c->g.inactive = c->d_inactive;
    return HPMC_OK;
}

size_t hpmc_workspace_bytes(const hpmc_ctx* c) { return c ? layout_of(c).total : 0; }

int hpmc_bind(hpmc_ctx* c, float* d_pos4, float* d_quat4, void* d_workspace, size_t bytes)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (((!d_pos4 || !d_quat4) && c->g.N > 0) || !d_workspace) return fail(c, HPMC_E_ARG, "NULL device pointer");
    const Layout L = layout_of(c);
    if (bytes < L.total) return fail(c, HPMC_E_UNBOUND, "workspace smaller than hpmc_workspace_bytes()");
    if (((uintptr_t)d_workspace & 255u) || ((uintptr_t)d_pos4 & 15u) || ((uintptr_t)d_quat4 & 15u))
        return fail(c, HPMC_E_ARG, "workspace must be 256-byte aligned, state arrays 16-byte aligned");
    graph_reset(c);
    const bool first = (c->d_ws == nullptr) || (c->d_ws != (char*)d_workspace);
    c->d_pos_bound = (float4*)d_pos4;
    c->d_quat_bound = (float4*)d_quat4;
    c->d_ws = (char*)d_workspace;
    c->ws_bytes = bytes;
    for (int b = 0; b < 2; ++b) {
        c->pos[b] = (float4*)(c->d_ws + L.pos[b]);
        c->quat[b] = (float4*)(c->d_ws + L.quat[b]);
        c->tag[b] = (int*)(c->d_ws + L.tag[b]);
    }
    c->key_rank = (int2*)(c->d_ws + L.key_rank);
    c->cell_start = (int*)(c->d_ws + L.cell_start);
    c->counts = (int*)(c->d_ws + L.counts);
    c->arrived = (int*)(c->d_ws + L.arrived);
    c->tile_sums = (int*)(c->d_ws + L.tile_sums);
    c->flow_done = (unsigned int*)(c->d_ws + L.flow_done);
    c->ctrl = (Control*)(c->d_ws + L.ctrl);
    c->d_inactive = (unsigned char*)(c->d_ws + L.inactive);
    if (upload_inactive(c) != HPMC_OK) return HPMC_E_CUDA;
    if (first) {  // a new workspace: zero the builder's scratch, (re)create the control block, keeping the host-side sweep counter
        if (!cuda_ok(c, cudaMemsetAsync(c->d_ws + L.counts, 0, L.ctrl - L.counts, c->stream), "bind/memset")) return HPMC_E_CUDA;
        Control& init = c->h_ctrl;
        std::memset(&init, 0, sizeof init);
        init.t = c->t_host;
        if (!cuda_ok(c, cudaMemcpyAsync(c->ctrl, &init, sizeof init, cudaMemcpyHostToDevice, c->stream), "bind/memcpy")) return HPMC_E_CUDA;
        if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "bind/sync")) return HPMC_E_CUDA;  // `init` is a stack object
    } else if (!cuda_ok(c, cudaMemsetAsync(&c->ctrl->bad_coords, 0, sizeof(unsigned int), c->stream), "bind/memset")) {
        return HPMC_E_CUDA;   // a new state: its coordinates are checked afresh
    }
    c->state_in_bound = true;
    c->have_sorted = false;
    c->cur = 0;
    c->dist = false;          // a bound state is a whole state in tag order
    c->g.N = c->n_cap;
    return HPMC_OK;
}

int hpmc_set_moves(hpmc_ctx* c, double d, double a, int n_select)
{
    if (!c) return HPMC_E_ARG;
    if (!(d > 0.0) || !(a >= 0.0) || n_select < 1 || n_select > 65535) return fail(c, HPMC_E_ARG, "need d > 0, a >= 0, 1 <= n_select <= 65535");
    graph_reset(c);
    c->mv.d = (float)d;
    c->mv.a = (float)a;
    c->mv.n_select = n_select;
    return HPMC_OK;
}

int hpmc_sweep(hpmc_ctx* c, int64_t n)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (n < 0) return fail(c, HPMC_E_ARG, "n must be >= 0");
    if (c->dist) return fail(c, HPMC_E_ARG, "distributed state: sweeps go through hpmc_sweep_phase and hpmc_dist_route");
    if (c->trace && c->trace_words < 2 * (int64_t)c->g.C * c->mv.n_select) return fail(c, HPMC_E_TRACE, "trace buffer too small");
    int64_t s = 0;
    // Small 2-D systems: whole sweeps inside one thread-block cluster, any number per launch (sweep_cluster2d.cuh)
    if (cluster_eligible(c)) {
        if (c->state_in_bound) {   // the first build reads the caller's tag-order arrays: one plain sweep
            rc = sweep_once(c);
            if (rc != HPMC_OK) return rc;
            ++s;
        }
        if (s < n) {
            const int64_t got = sweep_cluster(c, n - s);
            if (got < 0) return HPMC_E_CUDA;
            s += got;
        }
        if (s == n) return HPMC_OK;
    }
    // Launch-bound systems (config 1: 11 launches of a few microseconds per sweep): replay a captured graph of two
    // sweeps.  The sweep counter, header and counters live on the device, so the replay needs no new arguments.
    if (c->opt_graph && c->stream != nullptr && !c->trace && !c->profile && n >= 3) {   // the legacy default stream cannot be captured
        if (c->state_in_bound || !c->graph_exec[c->cur]) {   // one plain sweep first: sorted copy exists, kernels are loaded
            rc = sweep_once(c);
            if (rc != HPMC_OK) return rc;
            ++s;
        }
        if (!c->graph_exec[c->cur] && n - s >= 2) {
            const int64_t l0 = c->launches;
            cudaGraph_t graph = nullptr;
            if (!cuda_ok(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal), "graph/begin")) return HPMC_E_CUDA;
            rc = sweep_once(c);
            if (rc == HPMC_OK) rc = sweep_once(c);
            const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
            c->t_host -= (rc == HPMC_OK) ? 2 : 0;   // captured, not run
            if (rc != HPMC_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (!cuda_ok(c, e, "graph/end")) return HPMC_E_CUDA;
            c->graph_launches = c->launches - l0;
            c->launches = l0;
            const cudaError_t ei = cudaGraphInstantiate(&c->graph_exec[c->cur], graph, 0);
            cudaGraphDestroy(graph);
            if (!cuda_ok(c, ei, "graph/instantiate")) return HPMC_E_CUDA;
        }
        while (n - s >= 2 && c->graph_exec[c->cur]) {
            if (!cuda_ok(c, cudaGraphLaunch(c->graph_exec[c->cur], c->stream), "graph/launch")) return HPMC_E_CUDA;
            c->launches += c->graph_launches;
            c->t_host += 2;
            s += 2;
        }
    }
    for (; s < n; ++s) {
        rc = sweep_once(c);
        if (rc != HPMC_OK) return rc;
    }
    return HPMC_OK;
}

int hpmc_count_overlaps(hpmc_ctx* c, int64_t* h_count)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!h_count) return fail(c, HPMC_E_ARG, "h_count is NULL");
    rc = build_cell_list(c, 2, 0ull);
    if (rc != HPMC_OK) return rc;
    if (!cuda_ok(c, cudaMemsetAsync(&c->ctrl->overlaps, 0, sizeof(unsigned long long), c->stream), "count/memset")) return HPMC_E_CUDA;
    if (c->g.N > 0) {
        const int TB = 128, nb = (c->g.N + TB - 1) / TB;
        switch (c->sd.kind) {
            case kKindDisk: k_count_overlaps<kKindDisk><<<nb, TB, 0, c->stream>>>(c->g, c->sd, c->ctrl, c->pos[c->cur], c->quat[c->cur], c->tag[c->cur], c->cell_start); break;
            case kKindPolygon: k_count_overlaps<kKindPolygon><<<nb, TB, 0, c->stream>>>(c->g, c->sd, c->ctrl, c->pos[c->cur], c->quat[c->cur], c->tag[c->cur], c->cell_start); break;
            default: k_count_overlaps<kKindPolyhedron><<<nb, TB, 0, c->stream>>>(c->g, c->sd, c->ctrl, c->pos[c->cur], c->quat[c->cur], c->tag[c->cur], c->cell_start); break;
        }
        LAUNCH_CHECK(c, "k_count_overlaps");
    }
    unsigned long long v = 0;
    unsigned int bad = 0;
    if (!cuda_ok(c, cudaMemcpyAsync(&v, &c->ctrl->overlaps, sizeof v, cudaMemcpyDeviceToHost, c->stream), "count/memcpy")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaMemcpyAsync(&bad, &c->ctrl->bad_coords, sizeof bad, cudaMemcpyDeviceToHost, c->stream), "count/memcpy")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "count/sync")) return HPMC_E_CUDA;
    *h_count = (int64_t)v;
    if (bad) return fail(c, HPMC_E_ARG, "the bound state holds coordinates that are not finite or not in [-L/2, L/2)");
    return HPMC_OK;
}

int hpmc_get_state(hpmc_ctx* c, float* d_pos4_out, float* d_quat4_out, hpmc_counters* h_counters, int64_t* h_sweep_counter)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if ((d_pos4_out || d_quat4_out) && c->dist)
        return fail(c, HPMC_E_ARG, "distributed state: tags are global ids; read hpmc_sorted_pose / hpmc_sorted_tags");
    if ((d_pos4_out || d_quat4_out) && c->g.N > 0) {
        if (c->state_in_bound) {  // nothing ran since bind: the bound arrays are the state
            const size_t bytes = (size_t)c->g.N * sizeof(float4);
            if (d_pos4_out && (float4*)d_pos4_out != c->d_pos_bound &&
                !cuda_ok(c, cudaMemcpyAsync(d_pos4_out, c->d_pos_bound, bytes, cudaMemcpyDeviceToDevice, c->stream), "get_state/copy")) return HPMC_E_CUDA;
            if (d_quat4_out && (float4*)d_quat4_out != c->d_quat_bound &&
                !cuda_ok(c, cudaMemcpyAsync(d_quat4_out, c->d_quat_bound, bytes, cudaMemcpyDeviceToDevice, c->stream), "get_state/copy")) return HPMC_E_CUDA;
        } else {
            const int TB = 256;
            k_unsort<<<(c->g.N + TB - 1) / TB, TB, 0, c->stream>>>(c->g.N, c->g.dim, c->pos[c->cur], c->quat[c->cur], c->tag[c->cur],
                                                                  (float4*)d_pos4_out, (float4*)d_quat4_out);
            LAUNCH_CHECK(c, "k_unsort");
        }
    }
    if (h_counters || h_sweep_counter) {
        Control& h = c->h_ctrl;
        if (!cuda_ok(c, cudaMemcpyAsync(&h, c->ctrl, sizeof h, cudaMemcpyDeviceToHost, c->stream), "get_state/memcpy")) return HPMC_E_CUDA;
        if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "get_state/sync")) return HPMC_E_CUDA;
        if (h_counters) {
            unsigned long long sum[6] = {0, 0, 0, 0, 0, 0};
            for (int r = 0; r < kCounterSets; ++r)
                for (int k = 0; k < 6; ++k) sum[k] += h.counters[r][k];
            h_counters->trans_acc = sum[0]; h_counters->trans_rej_overlap = sum[1];
            h_counters->trans_rej_cell = sum[2]; h_counters->rot_acc = sum[3];
            h_counters->rot_rej_overlap = sum[4]; h_counters->trials = sum[5]; h_counters->sweeps = h.sweeps;
        }
        if (h_sweep_counter) *h_sweep_counter = (int64_t)h.t;
        if (h.bad_coords) return fail(c, HPMC_E_ARG, "the bound state holds coordinates that are not finite or not in [-L/2, L/2)");
    }
    return HPMC_OK;
}

int hpmc_set_sweep_counter(hpmc_ctx* c, uint64_t t)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    c->t_host = t;
    if (c->ctrl) {
        // the dataflow pass stamps tiles with the sweep counter: a counter set back must not meet its old stamps
        if (!cuda_ok(c, cudaMemsetAsync(c->flow_done, 0, flow_words(c) * sizeof(unsigned int), c->stream), "set_t/memset")) return HPMC_E_CUDA;
        const unsigned long long v = t;
        if (!cuda_ok(c, cudaMemcpyAsync(&c->ctrl->t, &v, sizeof v, cudaMemcpyHostToDevice, c->stream), "set_t/memcpy")) return HPMC_E_CUDA;
        if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "set_t/sync")) return HPMC_E_CUDA;
    }
    return HPMC_OK;
}

int hpmc_reset_counters(hpmc_ctx* c)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (!c->ctrl) return fail(c, HPMC_E_UNBOUND, "workspace not bound");
    if (!cuda_ok(c, cudaMemsetAsync(&c->ctrl->sweeps, 0, sizeof(unsigned long long) * (1 + 8 * kCounterSets), c->stream), "reset/memset")) return HPMC_E_CUDA;
    return HPMC_OK;
}

int hpmc_set_trace(hpmc_ctx* c, uint32_t* d_trace, int64_t capacity_words)
{
    if (!c) return HPMC_E_ARG;
    if (d_trace && ((uintptr_t)d_trace & 7u)) return fail(c, HPMC_E_ARG, "trace must be 8-byte aligned");
    graph_reset(c);
    c->trace = (uint2*)d_trace;
    c->trace_words = d_trace ? capacity_words : 0;
    return HPMC_OK;
}

int hpmc_get_cell_list(hpmc_ctx* c, uint64_t t, int32_t* d_cell_start, int32_t* d_member_tags, int32_t* d_cell_of_tag,
                       float* h_shift3, int32_t* h_colour_perm8)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    const bool from_bound = c->state_in_bound;
    const int* src_tag = from_bound ? nullptr : c->tag[c->cur];
    rc = build_cell_list(c, 1, (unsigned long long)t);
    if (rc != HPMC_OK) return rc;
    const size_t nb = (size_t)c->g.N * sizeof(int);
    if (d_cell_start && !cuda_ok(c, cudaMemcpyAsync(d_cell_start, c->cell_start, ((size_t)c->g.C + 1) * sizeof(int), cudaMemcpyDeviceToDevice, c->stream), "cell_list/copy")) return HPMC_E_CUDA;
    if (d_member_tags && c->g.N > 0 && !cuda_ok(c, cudaMemcpyAsync(d_member_tags, c->tag[c->cur], nb, cudaMemcpyDeviceToDevice, c->stream), "cell_list/copy")) return HPMC_E_CUDA;
    if (d_cell_of_tag && c->g.N > 0) {
        const int TB = 256;
        k_cell_of_tag<<<(c->g.N + TB - 1) / TB, TB, 0, c->stream>>>(c->g.N, c->key_rank, src_tag, d_cell_of_tag);
        LAUNCH_CHECK(c, "k_cell_of_tag");
    }
    if (h_shift3 || h_colour_perm8) {
        Control& h = c->h_ctrl;
        if (!cuda_ok(c, cudaMemcpyAsync(&h, c->ctrl, sizeof h, cudaMemcpyDeviceToHost, c->stream), "cell_list/memcpy")) return HPMC_E_CUDA;
        if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "cell_list/sync")) return HPMC_E_CUDA;
        if (h_shift3) for (int k = 0; k < 3; ++k) h_shift3[k] = h.hdr.shift[k];
        if (h_colour_perm8) for (int k = 0; k < 8; ++k) h_colour_perm8[k] = h.hdr.perm[k];
    }
    return HPMC_OK;
}

int hpmc_sweep_host(hpmc_ctx* c, const float* h_pos4, const float* h_quat4, int64_t n, float* h_pos4_out, float* h_quat4_out,
                    hpmc_counters* h_counters)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (!c->d_ws || !c->d_pos_bound) return fail(c, HPMC_E_UNBOUND, "state/workspace not bound");
    if (!h_pos4 || !h_quat4) return fail(c, HPMC_E_ARG, "NULL host pointer");
    const size_t bytes = (size_t)c->g.N * sizeof(float4);
    if (!cuda_ok(c, cudaMemsetAsync(&c->ctrl->bad_coords, 0, sizeof(unsigned int), c->stream), "sweep_host/memset")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaMemcpyAsync(c->d_pos_bound, h_pos4, bytes, cudaMemcpyHostToDevice, c->stream), "sweep_host/h2d")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaMemcpyAsync(c->d_quat_bound, h_quat4, bytes, cudaMemcpyHostToDevice, c->stream), "sweep_host/h2d")) return HPMC_E_CUDA;
    c->state_in_bound = true;
    c->have_sorted = false;
    c->dist = false;
    c->g.N = c->n_cap;
    int rc = hpmc_sweep(c, n);
    if (rc != HPMC_OK) return rc;
    rc = hpmc_get_state(c, (float*)c->d_pos_bound, (float*)c->d_quat_bound, nullptr, nullptr);
    if (rc != HPMC_OK) return rc;
    if (h_pos4_out && !cuda_ok(c, cudaMemcpyAsync(h_pos4_out, c->d_pos_bound, bytes, cudaMemcpyDeviceToHost, c->stream), "sweep_host/d2h")) return HPMC_E_CUDA;
    if (h_quat4_out && !cuda_ok(c, cudaMemcpyAsync(h_quat4_out, c->d_quat_bound, bytes, cudaMemcpyDeviceToHost, c->stream), "sweep_host/d2h")) return HPMC_E_CUDA;
    hpmc_counters tmp;
    rc = hpmc_get_state(c, nullptr, nullptr, h_counters ? h_counters : &tmp, nullptr);  // also synchronises
    return rc;
}

namespace {
// tag-order pose (x, y, qw, qz) <-> pos4 (x, y, 0, 0) + quat4 (qw, 0, 0, qz) over the bound arrays, element by element in place
__global__ void k_pose_expand(int N, float4* __restrict__ pos, float4* __restrict__ quat)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 P = pos[i];
    quat[i] = make_float4(P.z, 0.0f, 0.0f, P.w);
    pos[i] = make_float4(P.x, P.y, 0.0f, 0.0f);
}
__global__ void k_pose_pack(int N, float4* __restrict__ pos, const float4* __restrict__ quat)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 P = pos[i], Q = quat[i];
    pos[i] = make_float4(P.x, P.y, Q.x, Q.w);
}
}  // namespace

int hpmc_sweep_host_pose2d(hpmc_ctx* c, const float* h_pose4, int64_t n, float* h_pose4_out, hpmc_counters* h_counters)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (c->g.dim != 2) return fail(c, HPMC_E_ARG, "hpmc_sweep_host_pose2d needs a 2-D system");
    if (!c->d_ws || !c->d_pos_bound) return fail(c, HPMC_E_UNBOUND, "state/workspace not bound");
    if (!h_pose4) return fail(c, HPMC_E_ARG, "NULL host pointer");
    const int N = c->n_cap, TB = 256;
    const size_t bytes = (size_t)N * sizeof(float4);
    if (!cuda_ok(c, cudaMemsetAsync(&c->ctrl->bad_coords, 0, sizeof(unsigned int), c->stream), "sweep_host_pose2d/memset")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaMemcpyAsync(c->d_pos_bound, h_pose4, bytes, cudaMemcpyHostToDevice, c->stream), "sweep_host_pose2d/h2d")) return HPMC_E_CUDA;
    if (N > 0) {
        k_pose_expand<<<(N + TB - 1) / TB, TB, 0, c->stream>>>(N, (float4*)c->d_pos_bound, (float4*)c->d_quat_bound);
        LAUNCH_CHECK(c, "k_pose_expand");
    }
    c->state_in_bound = true;
    c->have_sorted = false;
    c->dist = false;
    c->g.N = c->n_cap;
    int rc = hpmc_sweep(c, n);
    if (rc != HPMC_OK) return rc;
    rc = hpmc_get_state(c, (float*)c->d_pos_bound, (float*)c->d_quat_bound, nullptr, nullptr);
    if (rc != HPMC_OK) return rc;
    if (h_pose4_out && N > 0) {
        k_pose_pack<<<(N + TB - 1) / TB, TB, 0, c->stream>>>(N, (float4*)c->d_pos_bound, (const float4*)c->d_quat_bound);
        LAUNCH_CHECK(c, "k_pose_pack");
        if (!cuda_ok(c, cudaMemcpyAsync(h_pose4_out, c->d_pos_bound, bytes, cudaMemcpyDeviceToHost, c->stream), "sweep_host_pose2d/d2h")) return HPMC_E_CUDA;
        // the bound arrays are the caller's: leave them in the documented pos4 / quat4 layout
        k_pose_expand<<<(N + TB - 1) / TB, TB, 0, c->stream>>>(N, (float4*)c->d_pos_bound, (float4*)c->d_quat_bound);
        LAUNCH_CHECK(c, "k_pose_expand");
    }
    hpmc_counters tmp;
    rc = hpmc_get_state(c, nullptr, nullptr, h_counters ? h_counters : &tmp, nullptr);  // also synchronises
    return rc;
}

int hpmc_set_option(hpmc_ctx* c, const char* name, int64_t value)
{
    DeviceGuard dev_guard(c);
    if (!c || !name) return HPMC_E_ARG;
    const std::string n(name);
    graph_reset(c);
    // another tile shape indexes the dataflow stamps differently: start from the cleared state
    if (c->flow_done && !c->cuda_failed &&
        !cuda_ok(c, cudaMemsetAsync(c->flow_done, 0, flow_words(c) * sizeof(unsigned int), c->stream), "option/memset")) return HPMC_E_CUDA;
    if (n == "graph") {
        c->opt_graph = value != 0;
    } else if (n == "path") {
        if (value < 0 || value > 5) return fail(c, HPMC_E_ARG, "path must be 0 (auto), 1 (per-thread), 2 (tile), 3 (warp per cell), 4 (cluster) or 5 (speculative warp per cell)");
        c->opt_path = (int)value;
    } else if (n == "tile_cap") {
        if (value < 0) return fail(c, HPMC_E_ARG, "tile_cap must be >= 0");
        c->opt_tile_cap = value > (1 << 30) ? (1 << 30) : (int)value;
    } else if (n == "small_build") {
        c->opt_small_build = value != 0;
    } else if (n == "pdl") {
        c->opt_pdl = value != 0;
    } else if (n == "flow") {
        if (value < -1 || value > 1) return fail(c, HPMC_E_ARG, "flow must be -1 (auto), 0 or 1");
        c->opt_flow = (int)value;
    } else if (n == "tile_shape") {
        if (value < 0 || value > 3) return fail(c, HPMC_E_ARG, "tile_shape must be 0 (auto) or 1..3");
        c->opt_tile_shape = (int)value;
    } else
        return fail(c, HPMC_E_ARG, "unknown option");
    return HPMC_OK;
}

int hpmc_set_profile(hpmc_ctx* c, int on)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (!profile_fold(c)) return HPMC_E_CUDA;
    c->profile = on != 0;
    c->prof_ms[0] = c->prof_ms[1] = 0.0;
    c->prof_n[0] = c->prof_n[1] = 0;
    return HPMC_OK;
}

int hpmc_get_profile(hpmc_ctx* c, double* h_ms_build, int64_t* h_n_build, double* h_ms_colour, int64_t* h_n_colour)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (!profile_fold(c)) return HPMC_E_CUDA;
    if (h_ms_build) *h_ms_build = c->prof_ms[0];
    if (h_n_build) *h_n_build = c->prof_n[0];
    if (h_ms_colour) *h_ms_colour = c->prof_ms[1];
    if (h_n_colour) *h_n_colour = c->prof_n[1];
    return HPMC_OK;
}

int hpmc_describe_pass(const hpmc_ctx* c, char* h_buf, size_t n)
{
    if (!c || !h_buf || n == 0) return HPMC_E_ARG;
    const GridParams& g = c->g;
    const int nactive = (g.n[0] / 2) * (g.n[1] / 2) * (g.dim == 3 ? g.n[2] / 2 : 1);
    std::string d;
    if (cluster_eligible(c) && c->cluster_ctas != 0)
        d = "k_sweep_cluster2d: whole sweeps (build + 4 colour passes) in one launch of one thread-block cluster of " +
            std::to_string(c->cluster_ctas > 0 ? c->cluster_ctas : kClusterMaxCtas) + " CTAs";
    else if (c->opt_path == 1) d = "k_sweep_colour: one thread per active cell";
    else if (use_spec(c)) d = "k_sweep_spec2d: one warp per active cell, the decision tree of 4 trials evaluated at once, 1 colour pass per launch";
    else if (g.dim == 3 || c->opt_path == 3 || (c->opt_path == 0 && c->opt_tile_shape == 0 && nactive <= kWarpCellMax2d))
        d = (g.dim == 3 && c->sf.kind == kKindPolyhedron && nactive > kOccMinActive3d)
                ? "k_sweep_warpcell_occ: one warp per active cell at 96 registers (20 warps/SM), two lanes per narrow-phase pair, 1 colour pass per launch"
                : "k_sweep_warpcell: one warp per active cell, 1 colour pass per launch";
    else {
        static const char* shapes[4] = {"", "8 warps x 2 rows, 2 CTAs/SM", "4 warps x 1 row, 8 CTAs/SM", "2 warps x 1 row, 8 CTAs/SM"};
        const bool flow = use_flow(c);
        d = std::string(flow ? "k_sweep_tile2d_flow<" : "k_sweep_tile2d<") + shapes[pick_tile_shape(c)] + ">: " +
            (flow ? "4 colour passes per launch (dataflow)" : "1 colour pass per launch");
    }
    std::snprintf(h_buf, n, "%s", d.c_str());
    return (int)std::min(d.size(), n - 1);
}

// ---- compute partition across contexts / GPUs --------------------------------------------------------
namespace {
void slab_rows(const hpmc_ctx* c, int rank, int nranks, int& r0, int& r1)
{
    const int TH = tile_rows(pick_tile_shape(c));
    const int nay = c->g.n[1] / 2, tiles_y = (nay + TH - 1) / TH;
    const int ty0 = (int)((long long)tiles_y * rank / nranks), ty1 = (int)((long long)tiles_y * (rank + 1) / nranks);
    r0 = std::min(2 * TH * ty0, c->g.n[1]);
    r1 = std::min(2 * TH * ty1, c->g.n[1]);
}
}  // namespace

int hpmc_set_partition(hpmc_ctx* c, int rank, int nranks)
{
    if (!c) return HPMC_E_ARG;
    if (nranks < 1 || rank < 0 || rank >= nranks) return fail(c, HPMC_E_ARG, "need 0 <= rank < nranks");
    if (nranks > 1 && (c->g.dim != 2 || c->sf.kind == kKindPolyhedron)) return fail(c, HPMC_E_ARG, "partitioned sweeps: 2-D tile pass only");
    if (nranks > 1 && c->trace) return fail(c, HPMC_E_ARG, "partitioned sweeps keep no trace");
    graph_reset(c);
    c->part_rank = rank;
    c->part_n = nranks;
    return HPMC_OK;
}

int hpmc_set_inactive_layers(hpmc_ctx* c, const uint8_t* h_mask, int32_t n)
{
    DeviceGuard dev_guard(c);
    if (!c) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    if (h_mask && n != c->g.n[c->g.dim - 1]) return fail(c, HPMC_E_ARG, "mask length must be the grid extent along the last axis");
    graph_reset(c);   // a captured sweep carries the old grid parameters
    if (h_mask) c->inactive_h.assign(h_mask, h_mask + n);
    else c->inactive_h.clear();
    return upload_inactive(c);
}

int hpmc_sweep_phase(hpmc_ctx* c, int phase)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (phase == -1) {
        rc = build_cell_list(c, 0, 0ull);
        if (rc == HPMC_OK) ++c->t_host;
        return rc;
    }
    if (phase < 0 || phase >= (1 << c->g.dim)) return fail(c, HPMC_E_ARG, "phase must be -1 (build) or a colour index");
    if (!c->have_sorted || (c->dist && !c->cell_valid)) return fail(c, HPMC_E_UNBOUND, "no cell list: run phase -1 first");
    return launch_colour_dispatch(c, phase);
}

int hpmc_partition_rows(const hpmc_ctx* c, int rank, int nranks, int32_t* h_row_begin, int32_t* h_row_end)
{
    if (!c || !h_row_begin || !h_row_end || nranks < 1 || rank < 0 || rank >= nranks) return HPMC_E_ARG;
    int r0, r1;
    slab_rows(c, rank, nranks, r0, r1);
    *h_row_begin = r0;
    *h_row_end = r1;
    return HPMC_OK;
}

int hpmc_row_offsets(hpmc_ctx* c, const int32_t* h_rows, int n, int64_t* h_offsets)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!h_rows || !h_offsets || n < 0 || n > 64) return fail(c, HPMC_E_ARG, "need 0 <= n <= 64 rows");
    if (!c->have_sorted) return fail(c, HPMC_E_UNBOUND, "no cell list: run phase -1 first");
    int vals[64];
    for (int i = 0; i < n; ++i) {
        if (h_rows[i] < 0 || h_rows[i] > c->g.n[1]) return fail(c, HPMC_E_ARG, "cell row out of range");
        if (!cuda_ok(c, cudaMemcpyAsync(&vals[i], c->cell_start + (size_t)h_rows[i] * c->g.n[0], sizeof(int), cudaMemcpyDeviceToHost, c->stream), "rows/memcpy")) return HPMC_E_CUDA;
    }
    if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "rows/sync")) return HPMC_E_CUDA;
    for (int i = 0; i < n; ++i) h_offsets[i] = vals[i];
    return HPMC_OK;
}

int hpmc_sorted_tags(hpmc_ctx* c, void** d_tags)
{
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!d_tags) return fail(c, HPMC_E_ARG, "d_tags is NULL");
    if (!c->have_sorted) return fail(c, HPMC_E_UNBOUND, "no cell-sorted state yet");
    *d_tags = c->tag[c->cur];
    return HPMC_OK;
}

int64_t hpmc_local_count(const hpmc_ctx* c) { return c ? c->g.N : 0; }

static int dist_ready(hpmc_ctx* c)
{
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (c->g.dim != 2 || c->part_n < 2) return fail(c, HPMC_E_ARG, "distributed state: 2-D, after hpmc_set_partition with nranks >= 2");
    if (c->trace) return fail(c, HPMC_E_ARG, "distributed state keeps no trace");
    return HPMC_OK;
}

int hpmc_dist_load(hpmc_ctx* c, const float* d_pose4, const int32_t* d_tags, int64_t n)
{
    DeviceGuard dev_guard(c);
    int rc = dist_ready(c);
    if (rc != HPMC_OK) return rc;
    if (n < 0 || n > c->n_cap) return fail(c, HPMC_E_ARG, "more particles than the context was created for");
    if (n > 0 && (!d_pose4 || !d_tags)) return fail(c, HPMC_E_ARG, "NULL device pointer");
    graph_reset(c);
    c->cur = 0;
    if (n > 0) {
        if (!cuda_ok(c, cudaMemcpyAsync(c->pos[0], d_pose4, (size_t)n * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream), "dist_load/copy")) return HPMC_E_CUDA;
        if (!cuda_ok(c, cudaMemcpyAsync(c->tag[0], d_tags, (size_t)n * sizeof(int), cudaMemcpyDeviceToDevice, c->stream), "dist_load/copy")) return HPMC_E_CUDA;
    }
    c->g.N = (int)n;
    c->dist = true;
    c->state_in_bound = false;
    c->have_sorted = true;     // "sorted" arrays hold the state (no cell list yet: cell_valid is false until phase -1)
    c->cell_valid = false;
    c->after_colour = false;
    return HPMC_OK;
}

int hpmc_dist_route(hpmc_ctx* c, int owned_only, float* d_up_pose4, int32_t* d_up_tags, int64_t cap_up, float* d_down_pose4,
                    int32_t* d_down_tags, int64_t cap_down, int64_t* h_counts4)
{
    DeviceGuard dev_guard(c);
    int rc = dist_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!c->dist) return fail(c, HPMC_E_UNBOUND, "no distributed state: hpmc_dist_load first");
    if (!h_counts4 || cap_up < 0 || cap_down < 0 || (cap_up > 0 && (!d_up_pose4 || !d_up_tags)) || (cap_down > 0 && (!d_down_pose4 || !d_down_tags)))
        return fail(c, HPMC_E_ARG, "NULL buffer");
    if (owned_only && !c->cell_valid) return fail(c, HPMC_E_UNBOUND, "owned_only needs the cell list of the sweep just made");
    int r0, r1;
    slab_rows(c, c->part_rank, c->part_n, r0, r1);
    if (r1 - r0 < 2) return fail(c, HPMC_E_ARG, "a slab needs at least two cell rows");
    if (!cuda_ok(c, cudaMemsetAsync(c->ctrl->route, 0, sizeof(unsigned int) * 4, c->stream), "route/memset")) return HPMC_E_CUDA;
    const int dst = c->cur ^ 1;
    if (c->g.N > 0) {
        const int TB = 256;
        k_route<<<(c->g.N + TB - 1) / TB, TB, 0, c->stream>>>(c->g, c->ctrl, c->k0, c->k1, owned_only ? 1 : 0, r0, r1, c->pos[c->cur], c->tag[c->cur],
                                                              c->cell_start, c->pos[dst], c->tag[dst], (float4*)d_up_pose4, d_up_tags,
                                                              (int)std::min<int64_t>(cap_up, 2147483647), (float4*)d_down_pose4, d_down_tags,
                                                              (int)std::min<int64_t>(cap_down, 2147483647), c->ctrl->route);
        ++c->launches;
        if (!cuda_ok(c, cudaGetLastError(), "k_route")) return HPMC_E_CUDA;
    }
    unsigned int h[4] = {0, 0, 0, 0};
    if (!cuda_ok(c, cudaMemcpyAsync(h, c->ctrl->route, sizeof h, cudaMemcpyDeviceToHost, c->stream), "route/memcpy")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "route/sync")) return HPMC_E_CUDA;
    for (int k = 0; k < 4; ++k) h_counts4[k] = h[k];
    c->cur = dst;
    c->g.N = (int)h[0];
    c->cell_valid = false;
    c->after_colour = false;
    if ((int64_t)h[1] > cap_up || (int64_t)h[2] > cap_down) return fail(c, HPMC_E_ARG, "send buffer too small (counts returned)");
    if (owned_only && h[3] != 0) return fail(c, HPMC_E_ARG, "a particle moved more than one cell row between two sweeps");
    return HPMC_OK;
}

int hpmc_dist_append(hpmc_ctx* c, const float* d_pose4, const int32_t* d_tags, int64_t n)
{
    DeviceGuard dev_guard(c);
    int rc = dist_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!c->dist) return fail(c, HPMC_E_UNBOUND, "no distributed state: hpmc_dist_load first");
    if (n < 0 || (int64_t)c->g.N + n > c->n_cap) return fail(c, HPMC_E_ARG, "more particles than the context was created for");
    if (n == 0) return HPMC_OK;
    if (!d_pose4 || !d_tags) return fail(c, HPMC_E_ARG, "NULL device pointer");
    if (!cuda_ok(c, cudaMemcpyAsync(c->pos[c->cur] + c->g.N, d_pose4, (size_t)n * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream), "dist_append/copy")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaMemcpyAsync(c->tag[c->cur] + c->g.N, d_tags, (size_t)n * sizeof(int), cudaMemcpyDeviceToDevice, c->stream), "dist_append/copy")) return HPMC_E_CUDA;
    c->g.N += (int)n;
    c->cell_valid = false;
    return HPMC_OK;
}

int hpmc_sorted_pose(hpmc_ctx* c, void** d_pose)
{
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!d_pose) return fail(c, HPMC_E_ARG, "d_pose is NULL");
    if (!c->have_sorted) return fail(c, HPMC_E_UNBOUND, "no cell list: run phase -1 first");
    *d_pose = c->pos[c->cur];
    return HPMC_OK;
}

int hpmc_get_stat(hpmc_ctx* c, const char* name, int64_t* h_value)
{
    DeviceGuard dev_guard(c);
    int rc = check_ready(c);
    if (rc != HPMC_OK) return rc;
    if (!name || !h_value) return fail(c, HPMC_E_ARG, "NULL argument");
    if (std::string(name) != "gjk_f64_reruns") return fail(c, HPMC_E_ARG, "unknown stat");
    Control& h = c->h_ctrl;
    if (!cuda_ok(c, cudaMemcpyAsync(&h, c->ctrl, sizeof h, cudaMemcpyDeviceToHost, c->stream), "stat/memcpy")) return HPMC_E_CUDA;
    if (!cuda_ok(c, cudaStreamSynchronize(c->stream), "stat/sync")) return HPMC_E_CUDA;
    unsigned long long v = 0;
    for (int r = 0; r < kCounterSets; ++r) v += h.counters[r][6];
    *h_value = (int64_t)v;
    return HPMC_OK;
}

int hpmc_measure_fp32_peak(hpmc_ctx* c, double* h_tflops)
{
    DeviceGuard dev_guard(c);
    if (!c || !h_tflops) return HPMC_E_ARG;
    if (c->cuda_failed) return HPMC_E_CUDA;
    float* d_sink = nullptr;
    cudaEvent_t e0, e1;
    if (!cuda_ok(c, cudaMalloc(&d_sink, sizeof(float)), "peak/malloc")) return HPMC_E_CUDA;   // 4 bytes: the only allocation the library ever makes
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int threads = 256, blocks = c->num_sms * 8, iters = 8192;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, c->stream);
        k_fma_peak<<<blocks, threads, 0, c->stream>>>(d_sink, iters, 1.0f + 1e-7f * (float)rep);
        cudaEventRecord(e1, c->stream);
        if (!cuda_ok(c, cudaEventSynchronize(e1), "peak/sync")) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * kFmaChains * (double)iters * threads * blocks;
        if (rep > 0 && ms > 0.f) best = std::max(best, flops / (ms * 1e-3) / 1e12);   // the first launch loads the kernel
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_sink);
    if (c->cuda_failed) return HPMC_E_CUDA;
    *h_tflops = best;
    return HPMC_OK;
}

int64_t hpmc_launch_count(const hpmc_ctx* c) { return c ? c->launches : 0; }

}  // extern "C"
