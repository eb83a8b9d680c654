/*
 * hpmc.h -- C-ABI of libhpmc.so: the checkerboard-parallel Metropolis sweep for hard shapes
 * (arXiv:1509.04692, "HPMC") as hand-written CUDA for sm_100a.
 *
 * Citations: P:<n> = line n of the paper text; R<k> = reading k in DESIGN.md section 2.
 *
 * Conventions
 *   - every function returns 0 on success and a negative HPMC_E_* code on failure; the state is
 *     untouched by a failed call; hpmc_last_error() gives a human-readable reason.  A CUDA error is
 *     sticky: later calls on the same context report HPMC_E_CUDA too.
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.  The library allocates no
 *     particle-sized device memory: the caller (PyTorch in this repo) owns the state buffers and the
 *     workspace and must keep them alive while they are bound.  The library never frees them.
 *   - all work is enqueued on the CUDA stream given to hpmc_create (a cudaStream_t passed as void*;
 *     NULL = the legacy default stream).  Calls are asynchronous unless stated otherwise.
 *   - layout: pos4 = N x (x, y, z, 0) fp32, quat4 = N x (w, x, y, z) fp32 unit quaternions, both in
 *     TAG order (particle i at row i).  2-D systems keep z = 0 and quat = (cos t/2, 0, 0, sin t/2) (R30).
 *   - box: orthorhombic, periodic, centred on the origin, coordinates in [-L/2, L/2) (R14).  The box
 *     edge is L rounded to fp32 (R-box).
 *   - precondition on the state handed to hpmc_bind / hpmc_sweep_host: finite coordinates inside the box.  A violation never
 *     corrupts memory (the cell index is clamped) but is counted on the device, and the next hpmc_count_overlaps or
 *     hpmc_get_state(counters) returns HPMC_E_ARG.  A new hpmc_bind clears the count.
 *   - every entry point makes the device of the context (the one current at hpmc_create) current for its duration.
 *   - there is no CPU implementation behind this interface.
 */
#ifndef HPMC_H
#define HPMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HPMC_MAX_VERTS 32

#define HPMC_KIND_DISK 0       /* disk (dim 2) / sphere (dim 3): centre distance vs diameter   */
#define HPMC_KIND_POLYGON 1    /* convex polygon, body-frame vertices counter-clockwise: SAT */
#define HPMC_KIND_POLYHEDRON 2 /* convex polyhedron given by its vertices: GJK on the Minkowski
                                  difference with the support function of Eq. (1)-(2)   */

#define HPMC_OK 0
#define HPMC_E_ARG (-1)       /* bad argument (dim, N, d, a, n_select, NULL pointer, ...)          */
#define HPMC_E_SHAPE (-2)     /* non-convex / not CCW / too many vertices / vertex not on the hull */
#define HPMC_E_GRID (-3)      /* fewer than 4 cells per side (R11) or more than 2^31-2 cells                             */
#define HPMC_E_UNBOUND (-4)   /* state/workspace not bound, or workspace too small                 */
#define HPMC_E_CUDA (-5)      /* a CUDA call failed (sticky)                                       */
#define HPMC_E_TRACE (-6)     /* trace buffer too small for C * n_select slots                     */

typedef struct hpmc_ctx hpmc_ctx; /* opaque, owned by the library, freed by hpmc_destroy */

typedef struct {
    int dim;     /* 2 or 3 */
    double L[3]; /* box edges; L[2] ignored when dim == 2 */
} hpmc_box;

typedef struct {
    int kind;            /* HPMC_KIND_* */
    double diameter;     /* kind 0 */
    int nverts;          /* kind 1: 3..32 vertices (x,y); kind 2: 4..32 vertices (x,y,z) */
    const double* verts; /* h_: nverts*2 or nverts*3 doubles, body frame; read during the call only */
    double sweep_radius; /* kinds 1, 2: >= 0.  > 0 makes the shape a spheropolygon / convex spheropolyhedron: the polygon /
                            polyhedron swept by a disk / sphere of this radius; two of them overlap iff their cores are
                            closer than 2 sweep_radius, and d_max = 2 (circumradius + sweep_radius).  0 = the sharp shape.
                            Ignored for kind 0.  Negative or non-finite: HPMC_E_SHAPE.                                    */
} hpmc_shape;

/* P:47 "percentage of the trial moves are accepted": accepted / attempted per type (R26) */
typedef struct {
    uint64_t trans_acc, trans_rej_overlap, trans_rej_cell;
    uint64_t rot_acc, rot_rej_overlap;
    uint64_t trials, sweeps;
} hpmc_counters;

typedef struct {
    int dim;
    int n[3];        /* cells per side: n_k = 2*floor(L_k / (2 (d_max + slack))), slack = max(d_max 2^-10,
                        3 ulp_fp32(L_k)) (R11)                                                       */
    double w[3];     /* cell width L_k / n_k                                                        */
    float L_f[3];    /* box edge as used by the fp32 state                                          */
    float inv_w[3];  /* (float)(n_k / L_k), the factor inside cell_of (R13)                         */
    double d_max;    /* circumsphere diameter                                                 */
    int64_t num_cells;
    int64_t N;
} hpmc_grid_info;

/* NVT problem statement of P:38-45: N identical hard particles of one shape in a periodic box.
 * Validates the shape (convexity, CCW) and the grid (>= 4 cells per side).  Does NOT check that the
 * initial state is overlap-free -- call hpmc_count_overlaps (mirrors P:247).                       */
int hpmc_create(const hpmc_box* box, const hpmc_shape* shape, int64_t N, uint64_t seed,
                void* cuda_stream, hpmc_ctx** out);
int hpmc_destroy(hpmc_ctx* ctx);                  /* frees the context only: state and workspace belong to the caller (BASELINE.json
                                                     north_star: "PyTorch is used only for device memory and streams")              */
const char* hpmc_last_error(const hpmc_ctx* ctx); /* valid until the next call on ctx; ctx may be NULL */
int hpmc_get_grid(const hpmc_ctx* ctx, hpmc_grid_info* h_out);

/* Bytes of scratch the CALLER must allocate (256-byte aligned) and pass to hpmc_bind: the two cell-sorted SoA buffers of the
 * cell list of P:59 ("a bucket sort efficiently assigns particles to cells"), its keys, histogram and offsets, the dataflow
 * stamps and the control block.                                                                   */
size_t hpmc_workspace_bytes(const hpmc_ctx* ctx);

/* Bind the state -- positions r_i and orientations q_i of the N particles, tag order, see layout above -- and the
 * workspace.  d_pos4/d_quat4 are read by the
 * next hpmc_sweep / hpmc_count_overlaps (the library then works on its own cell-sorted copy inside
 * the workspace) and are used as device staging by hpmc_sweep_host.  Re-binding restarts from the
 * bound arrays; counters and the sweep counter are kept.                                           */
int hpmc_bind(hpmc_ctx* ctx, float* d_pos4, float* d_quat4, void* d_workspace, size_t workspace_bytes);

/* Trial move sizes: translation uniform in the cube [-d,d)^dim (R5), rotation angle uniform in
 * [-a,a) rad (R6), n_select trials per non-empty cell per colour (R9).  d > 0, a >= 0,
 * 1 <= n_select <= 65535.  Defaults: d = 0.1, a = 0.1, n_select = 4.                               */
int hpmc_set_moves(hpmc_ctx* ctx, double d, double a, int n_select);

/* n checkerboard sweeps (P:155-157 restated per north_star): per sweep a fresh grid shift, the
 * colours in a fresh random order, n_select trials in every non-empty cell of each colour.
 * Asynchronous; advances the sweep counter by n.                                                  */
int hpmc_sweep(hpmc_ctx* ctx, int64_t n);

/* Number of particle pairs whose interiors intersect (strict margin < 0, fp64 narrow phase),
 * P:247.  Synchronises the stream.                                                                */
int hpmc_count_overlaps(hpmc_ctx* ctx, int64_t* h_count);

/* Current state back in tag order into caller buffers (may be the bound ones), counters and sweep
 * counter to host.  Any of the out pointers may be NULL.  Synchronises iff a host pointer is given. */
int hpmc_get_state(hpmc_ctx* ctx, float* d_pos4_out, float* d_quat4_out, hpmc_counters* h_counters,
                   int64_t* h_sweep_counter);
int hpmc_set_sweep_counter(hpmc_ctx* ctx, uint64_t t);
int hpmc_reset_counters(hpmc_ctx* ctx);

/* Parity/debug trace (O8): while set, every sweep writes two uint32 words per trial slot
 * (slot = cell*n_select + k): word0 = particle tag, word1 = type (0 translate, 1 rotate) |
 * outcome<<8 with outcome 0 none (empty cell), 1 accepted, 2 rejected: left its cell,
 * 3 rejected: overlap.  The buffer is overwritten each sweep.  NULL disables.                      */
int hpmc_set_trace(hpmc_ctx* ctx, uint32_t* d_trace, int64_t capacity_words);

/* Parity/debug: build the cell list of sweep t (its grid shift) from the current state, without
 * making moves, and copy it out: CSR offsets (num_cells+1), member tags in stored order (N; ascending
 * inside each cell, R8) and the cell id of every particle in tag order (N).  Any pointer may be NULL. */
int hpmc_get_cell_list(hpmc_ctx* ctx, uint64_t t, int32_t* d_cell_start, int32_t* d_member_tags,
                       int32_t* d_cell_of_tag, float* h_shift3, int32_t* h_colour_perm8);

/* End-to-end convenience with HOST buffers (pinned or pageable): copies the state host->device into
 * the bound arrays, runs n sweeps, copies the state and counters back.  Synchronises.              */
int hpmc_sweep_host(hpmc_ctx* ctx, const float* h_pos4, const float* h_quat4, int64_t n,
                    float* h_pos4_out, float* h_quat4_out, hpmc_counters* h_counters);

/* The same for 2-D systems with the state as ONE host array of poses, N x (x, y, qw, qz) fp32 in tag order: a 2-D particle is
 * its position r_i and one rotation angle (R30: z = 0 and q = (cos t/2, 0, 0, sin t/2)), so half of the pos4 + quat4
 * layout is zeros and this call moves half the bytes over the host link (16 N each way).  Copies the poses host->device into
 * the bound arrays (their device staging), expands them to pos4 / quat4 there, runs n sweeps, packs the result and copies
 * poses and counters back.  h_pose4_out may be NULL.  Synchronises.  dim != 2: HPMC_E_ARG.                                 */
int hpmc_sweep_host_pose2d(hpmc_ctx* ctx, const float* h_pose4, int64_t n, float* h_pose4_out, hpmc_counters* h_counters);

/* Tuning and test knobs; results never depend on them (only speed does).
 *   "path"     0 = automatic, 1 = per-thread global-memory colour pass, 2 = shared-memory tile colour pass (2-D; in 3-D
 *              the warp-per-cell pass), 3 = warp-per-cell colour pass (automatic in 3-D and for small 2-D systems),
 *              4 = whole sweeps (cell list + the four colours) inside ONE launch of one thread-block cluster of up to 16 CTAs,
 *              separated by hardware cluster barriers (2-D, at most 16 384 particles and 11 498 cells; never automatic),
 *              5 = warp-per-cell pass that evaluates the decision tree of four consecutive trials of a cell at once (2-D;
 *              never automatic: measured no faster than 3)
 *   "tile_cap" upper limit on the particles a tile may stage; tiles above it take the per-thread path
 *              (tests set 0 to force that fallback everywhere).
 *   "tile_shape" 2-D tile kernel shape: 0 = chosen by grid size, 1 = 8 warps per CTA x 2 rows of 32 active cells per warp,
 *              2 = 4 warps x 1 row at 64 registers (8 CTAs per SM; large grids), 3 = 2 warps x 1 row (small grids).
 *   "flow"     2-D tile pass: -1 (default) or 1 = the four colours of a sweep go out as ONE persistent launch in which a tile
 *              of colour c+1 starts as soon as the nine tiles of colour c around it are done; 0 = one launch per colour.
 *   "small_build" 1 (default): a system with at most 11 500 cells and 8192 particles builds its cell list in one CTA
 *              (one launch instead of three); 0: always the multi-launch build.
 *   "graph"    1 (default): hpmc_sweep(n >= 3) replays a captured CUDA graph of two sweeps; 0: plain launches.
 *              Needs a real stream: contexts created on the legacy default stream (NULL) always use plain launches.
 *   "pdl"      1 (default): the kernels of a sweep are launched with programmatic stream serialisation: a kernel may start
 *              while its predecessor drains, and every kernel waits (griddepcontrol.wait) before it reads or writes anything
 *              a predecessor touches; 0: plain stream order.  */
int hpmc_set_option(hpmc_ctx* ctx, const char* name, int64_t value);

/* Per-kernel device timing for the roofline report (S:8(d)).  While on, CUDA events on the context's stream
 * bracket every cell-list build (rows a1-a3) and every colour-pass launch (rows a4-a11).  hpmc_set_profile
 * resets the sums; hpmc_get_profile synchronises and returns total milliseconds and number of bracketed
 * regions per class since then.  Any out pointer may be NULL.                                          */
int hpmc_set_profile(hpmc_ctx* ctx, int on);
int hpmc_get_profile(hpmc_ctx* ctx, double* h_ms_build, int64_t* h_n_build, double* h_ms_colour, int64_t* h_n_colour);

/* Which colour-pass kernel the current options select for this system, as text (for reports), e.g.
 * "k_sweep_tile2d_flow<4 warps x 1 row, 8 CTAs/SM>: 4 colour passes per launch".  Returns the length written.   */
int hpmc_describe_pass(const hpmc_ctx* ctx, char* h_buf, size_t buf_bytes);

/* ---- One system on several GPUs: partitioned compute over a replicated state -------------------------
 * The checkerboard makes the cells of one colour independent, so their tiles can be dealt to several contexts --
 * one per GPU -- that all hold the WHOLE state (the paper instead distributes the state; on NVLink the state of
 * these systems is a few MB to 1 GB and cheap to replicate).  Every context builds the same cell list (the build is
 * deterministic: members of a cell in ascending tag), runs the colour-pass tiles of its own slab of cell rows, and the caller
 * copies rows of the cell-sorted pose array between the contexts: after every colour pass the first and last cell row of a
 * slab to the contexts that hold the slabs next to it, after the last colour every slab to everybody.  Rows of cells are
 * contiguous in that array and sit at the same offsets in every context.  The trajectory is bit-identical to the
 * single-context one (same Philox keys per cell).  2-D systems, tile pass, no trace.
 *   hpmc_set_partition   this context owns share `rank` of `nranks` (tile rows dealt evenly); (0, 1) = the whole system
 *   hpmc_sweep_phase     phase -1: grid shift + cell list of the next sweep (advances the sweep counter);
 *                        phase 0 .. 2^d - 1: the colour pass of that index in the sweep's random order, own tiles only
 *   hpmc_partition_rows  cell rows [begin, end) of the slab of share `rank` (host arithmetic; same answer in every context)
 *   hpmc_row_offsets     index in the cell-sorted arrays of the first particle of each of n <= 64 cell rows (row n_y = N);
 *                        reads the current cell list, synchronises
 *   hpmc_sorted_pose     device pointer of the current cell-sorted pose array (N x float4 (x, y, qw, qz)); valid until
 *                        the next phase -1                                                                              */
int hpmc_set_partition(hpmc_ctx* ctx, int rank, int nranks);
int hpmc_sweep_phase(hpmc_ctx* ctx, int phase);
int hpmc_partition_rows(const hpmc_ctx* ctx, int rank, int nranks, int32_t* h_row_begin, int32_t* h_row_end);
int hpmc_row_offsets(hpmc_ctx* ctx, const int32_t* h_rows, int n, int64_t* h_offsets);
int hpmc_sorted_pose(hpmc_ctx* ctx, void** d_pose);

/* ---- One system on several GPUs: distributed state with an inactive region -----------------
 * "Each rank covers a portion of the simulation box and owns all of the particles in that region"; "we modify the
 * checkerboard scheme to have only two regions (active and inactive) ... these particles do not move during substeps.
 * Communication between ranks only occurs at the end of the step".
 *
 *   hpmc_set_inactive_layers  h_mask: n = (grid extent along the LAST axis) bytes, host; layer k of cells (a cell row in 2-D, a
 *                        z-layer in 3-D) makes no trials while h_mask[k] != 0 (reading R-strip: the strip is whole cells of the
 *                        sweep's shifted grid, >= d_max wide, and moves with the grid shift).  NULL clears.  Works for every
 *                        colour-pass kernel but the cluster pass, with or without a partition; results match the oracle's
 *                        orc_set_inactive_layers.  The mask is copied; synchronises.
 *
 * With hpmc_set_partition(rank, nranks >= 2) and a mask that flags the LAST cell row of every slab, a context no longer needs
 * the whole state: during a sweep its tiles read rows [r0 - 1, r1) only, and row r0 - 1 -- the inactive last row of the slab
 * below -- does not change.  Such a context holds its own slab plus that ghost row, under GLOBAL tags (the members of a cell
 * are ordered by tag, so the trajectory equals the single-context one with the same mask), and once per sweep the caller
 * moves particles between the contexts (the paper's stage 9).  2-D, tile pass, no trace; N of hpmc_create is the capacity.
 *   hpmc_dist_load     n <= capacity particles as device arrays: poses (x, y, qw, qz) and int32 global tags, any order; they
 *                      become the context's state (hpmc_get_state no longer applies: read hpmc_sorted_pose / hpmc_sorted_tags)
 *   hpmc_dist_route    classify the particles for the grid of the NEXT sweep (header of the current sweep counter) with the
 *                      pinned cell function: keep rows r0 - 1 .. r1 - 1; copy rows r1 - 1 and r1 to the `up` buffers (for the
 *                      context above) and row r0 - 1 to the `down` buffers (for the one below); drop the rest.
 *                      owned_only = 1: after a sweep -- only the own slab is classified (the old ghost row is dropped) and a
 *                      particle that fits no class is an error; 0: after hpmc_dist_load of a superset -- foreign particles are
 *                      dropped silently.  h_counts4 (host) = kept, up, down, unclassified.  Synchronises.  HPMC_E_ARG when a
 *                      send buffer is too small (counts are still returned; the state is then undefined).
 *   hpmc_dist_append   n received particles behind the kept ones
 *   hpmc_local_count   particles the context holds now
 *   hpmc_sorted_tags   device pointer of the tags that go with hpmc_sorted_pose
 * One sweep of a distributed system: phase -1, phases 0..3 (no exchange in between), hpmc_dist_route, exchange, hpmc_dist_append. */
int hpmc_set_inactive_layers(hpmc_ctx* ctx, const uint8_t* h_mask, int32_t n);
int hpmc_dist_load(hpmc_ctx* ctx, const float* d_pose4, const int32_t* d_tags, int64_t n);
int hpmc_dist_route(hpmc_ctx* ctx, int owned_only, float* d_up_pose4, int32_t* d_up_tags, int64_t cap_up, float* d_down_pose4,
                    int32_t* d_down_tags, int64_t cap_down, int64_t* h_counts4);
int hpmc_dist_append(hpmc_ctx* ctx, const float* d_pose4, const int32_t* d_tags, int64_t n);
int64_t hpmc_local_count(const hpmc_ctx* ctx);
int hpmc_sorted_tags(hpmc_ctx* ctx, void** d_tags);

/* Diagnostic tallies kept on the device (synchronises).  Names:
 *   "gjk_f64_reruns"  polyhedron pairs whose fp32 GJK verdict was "unsure" (near contact, or a degenerate simplex) and that
 *                     were decided by the fp64 re-run from the raw fp32 state -- the mixed-precision path of P:106-108,
 *                     R-poly.  Counted since the last hpmc_reset_counters.
 * Unknown names return HPMC_E_ARG.                                                                   */
int hpmc_get_stat(hpmc_ctx* ctx, const char* name, int64_t* h_value);

/* Measured FP32 roofline denominator (S:8(d)): runs a pure-FMA microkernel (16 independent fused multiply-add chains per
 * thread, 8 CTAs of 256 threads per SM, no memory traffic) on the context's stream and returns the best of three timed
 * launches in TFLOP/s (FMA = 2 flops).  Synchronises.  Nominal on B200: 148 SMs x 128 lanes x 2 x 1.965 GHz = 74.4.   */
int hpmc_measure_fp32_peak(hpmc_ctx* ctx, double* h_tflops);

/* The overlap count of P:247 without any allocation and without a workspace: for callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same result as hpmc_bind + hpmc_count_overlaps --
 * the number of pairs whose interiors intersect, strict margin < 0, fp64 narrow phase -- for the n particles given here in
 * the box and with the shape of `ctx` (n need not be the N of hpmc_create; the context needs no hpmc_bind and its own state
 * is not touched).
 *   d_pos4, d_quat4  DEVICE, n x float4 each, tag order, the layout of hpmc_bind (d_quat4 may be NULL for disks / spheres);
 *                    16-byte aligned; read only
 *   d_count_out      DEVICE, one int64, 8-byte aligned: the pair count, or -1 if a coordinate was not finite or not in
 *                    [-L/2, L/2) (the particle is then binned into a clamped cell; nothing is read out of bounds)
 * The cell list it needs lives in ONE static device array inside the library (1.25 MB on every GPU that loads libhpmc.so,
 * held until the process exits), so:
 *   - limits: n <= HPMC_NOALLOC_MAX_N and at most HPMC_NOALLOC_MAX_CELLS cells in the context's grid; beyond them the call
 *     returns HPMC_E_ARG with a message and launches nothing;
 *   - the call makes no cudaMalloc / cudaFree and calls no allocating routine: six kernel launches on the context's stream;
 *     it is asynchronous and never synchronises (read d_count_out after synchronising the stream).  The first call on a
 *     device also resolves the array's device address (cudaGetSymbolAddress): make that first call outside graph capture;
 *   - all calls on a device share the array, which keeps the previous call's contents; each call clears what it needs at
 *     zero.  Calls whose kernels can overlap on the GPU (contexts on different streams, several host threads) RACE on it:
 *     keep them on one stream or order them with events.                                                          */
#define HPMC_NOALLOC_MAX_N 65536
#define HPMC_NOALLOC_MAX_CELLS 131072
int hpmc_count_overlaps_noalloc(hpmc_ctx* ctx, const float* d_pos4, const float* d_quat4, int64_t n, int64_t* d_count_out);

/* Launch bookkeeping for bench.py: kernels launched by this context so far.                        */
int64_t hpmc_launch_count(const hpmc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
