/*
 * hpmc_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, serial, slow, obviously-correct CPU restatement of the checkerboard
 * Metropolis sweep for hard shapes (arXiv:1509.04692, "HPMC"), written from the
 * paper text (/root/reference/PAPER.md, cited below as P:<line>) and from the
 * readings R1..R30 collected in DESIGN.md.
 *
 * Rules this file lives under:
 *   - only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference legs may load it;
 *   - it shares no code, header, table or constant generator with the CUDA path
 *     under paper_1509_04692_b200/csrc/ and neither includes the other;
 *   - every overlap test is fp64; fp32 appears only where DESIGN.md pins a
 *     bit-exact fp32 operation (cell_of, the translation fmaf, the wrap, the
 *     grid shift) so that those integers/positions can be compared bit for bit;
 *   - no blocking, fusion or reordering beyond what the algorithm states.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known answers,
 * closed-form contact distances, Sutherland-Hodgman clipping and Chebyshev-LP
 * brute force for the SAT margins, GJK vs SAT sign, O(N^2) overlap counts, the
 * all-N twin (O6), the zero-overlap invariant, dilute-limit acceptance closed
 * form, colour independence (P4).  Acceptance/pressure VALUES for the
 * pentagon and cube state points are "parity unpinned" against the paper (it
 * prints none); see DESIGN.md.
 */
#ifndef HPMC_ORACLE_H
#define HPMC_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_VERTS 32
#define ORC_MAX_FACES 64
#define ORC_MAX_EDGES 96

#define ORC_KIND_DISK 0       /* disk (dim 2) or sphere (dim 3), "trivial" */
#define ORC_KIND_POLYGON 1    /* convex polygon, CCW body-frame vertices */
#define ORC_KIND_POLYHEDRON 2 /* convex polyhedron given by its vertices */

typedef struct orc_shape orc_shape;
typedef struct orc_sys orc_sys;

typedef struct {
    uint64_t trans_acc, trans_rej_overlap, trans_rej_cell;
    uint64_t rot_acc, rot_rej_overlap;
    uint64_t trials, sweeps;
} orc_counters;

/* O7 instrumentation, "early-exit serial order": candidates in
 * ascending neighbour-cell order (dz, dy, dx loops) then ascending tag. */
typedef struct {
    uint64_t cand_scanned_full;  /* all candidates in the 3^d block, no early exit */
    uint64_t sphere_pass_full;   /* of those, inside the circumsphere range          */
    uint64_t cand_scanned_early; /* scanned until the first overlapping neighbour    */
    uint64_t narrow_tests_early; /* narrow-phase tests until the first overlap       */
    /* filled only with orc_set_work_detail(1): per narrow test counted in narrow_tests_early, */
    uint64_t polygon_axes_early;      /* polygons: separating axes evaluated up to and including the first
                                         one that separates (A's normals, then B's; all 2n if none) */
    uint64_t gjk_support_calls_early; /* polyhedra: support-function calls (Eq. (1)) of the fp64 GJK */
} orc_work;

typedef struct {
    uint64_t compared;       /* trial slots compared                                 */
    uint64_t marginal;       /* outcome differed, |m_min - eps_g| < tol: GPU adopted */
    uint64_t hard_mismatch;  /* particle/type/leave-cell/non-marginal disagreement   */
    int64_t first_bad_slot;  /* slot of the first hard mismatch, -1 if none          */
    uint32_t first_bad_mine[2], first_bad_theirs[2];
    double first_bad_mmin;
} orc_follow_stats;

/* O8 "any other mismatch => FAIL with a dump": the trial pose of one slot and every candidate inside the circumsphere
 * range with its margin, recorded by the next sweep that reaches the slot (orc_set_probe). */
#define ORC_PROBE_MAX 64
typedef struct {
    int64_t slot, particle;
    int32_t rotate, ncand;
    float xt[3], qt[4];               /* trial pose as tested (fp32) */
    int64_t cand[ORC_PROBE_MAX];      /* neighbour particle index */
    double r[ORC_PROBE_MAX][3];       /* minimum-image separation r_j - x_trial */
    float qb[ORC_PROBE_MAX][4];       /* neighbour orientation */
    double margin[ORC_PROBE_MAX];     /* O4 margin of the pair */
} orc_probe;

/* ---- RNG (R3, R4) ------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
float orc_u01(uint32_t r);  /* (r>>8) * 2^-24 in [0,1)              */
float orc_usym(uint32_t r); /* ((int)(r>>8) - 2^23) * 2^-23 in [-1,1) */

/* ---- shapes and margins (O4) ------------------------------------------- */
orc_shape* orc_shape_create(int dim, int kind, double diameter, int nverts, const double* verts);
/* P:89 spheropolygon (dim 2, ORC_KIND_POLYGON) / convex spheropolyhedron (dim 3, ORC_KIND_POLYHEDRON): the polygon /
 * polyhedron ("core") swept by a disk / sphere of radius sweep_radius >= 0; d_max = 2 (circumradius + sweep_radius).
 * margin = distance between the cores - 2 sweep_radius (brute force over vertex/edge/face pairs). */
orc_shape* orc_shape_create_rounded(int dim, int kind, double sweep_radius, int nverts, const double* verts);
double orc_shape_sweep_radius(const orc_shape*);
void orc_shape_destroy(orc_shape*);
double orc_shape_dmax(const orc_shape*);
int orc_shape_nfaces(const orc_shape*);
int orc_shape_nedgedirs(const orc_shape*);
void orc_shape_faces(const orc_shape*, double* normals3, double* offsets);
/* margin m(A,B): r_ab = r_B - r_A (already minimum image), q = (w,x,y,z). */
double orc_shape_margin(const orc_shape*, const double r_ab[3], const double qa[4], const double qb[4]);
/* O9: scale lambda* of r_ab at which the pair first touches (overlap iff lambda < lambda*), from the O4 axis set */
double orc_shape_touch_scale(const orc_shape*, const double r_ab[3], const double qa[4], const double qb[4]);
/* fp64 GJK boolean: 1 origin in interior of B (-) A, 0 disjoint, -1 undecided */
int orc_shape_gjk(const orc_shape*, const double r_ab[3], const double qa[4], const double qb[4]);

/* ---- system -------------------------------------------------------------- */
orc_sys* orc_create(int dim, const double L[3], int kind, double diameter, int nverts,
                    const double* verts, int64_t N, uint64_t seed);
orc_sys* orc_create_rounded(int dim, const double L[3], int kind, double sweep_radius, int nverts, const double* verts,
                            int64_t N, uint64_t seed);
void orc_destroy(orc_sys*);
const orc_shape* orc_sys_shape(const orc_sys*);
int orc_set_moves(orc_sys*, double d, double a, int n_select);
void orc_set_eps_guard(orc_sys*, double eps_g);
void orc_set_state(orc_sys*, const float* pos4, const float* quat4);
void orc_get_state(const orc_sys*, float* pos4, float* quat4);
void orc_set_sweep_counter(orc_sys*, uint64_t t);
uint64_t orc_get_sweep_counter(const orc_sys*);
void orc_get_counters(const orc_sys*, orc_counters*);
void orc_get_work(const orc_sys*, orc_work*);
void orc_reset_counters(orc_sys*);
/* n[3], w[3] (double), w_f[3], inv_w[3] (fp32 as used by cell_of), L_f[3] */
void orc_get_grid(const orc_sys*, int32_t n[3], double w[3], float w_f[3], float inv_w[3], float L_f[3]);
int64_t orc_num_cells(const orc_sys*);

/* O3.1 / O3.2: grid shift and colour order of sweep t */
void orc_sweep_header(const orc_sys*, uint64_t t, float shift[3], int32_t perm[8]);
/* R13: pinned fp32 cell function, returns the linear cell id */
int32_t orc_cell_of(const orc_sys*, const float x[3], const float shift[3]);
/* O3.3: cell ids, CSR offsets (C+1), members ascending by tag (R8) */
void orc_cell_list(const orc_sys*, const float shift[3], int32_t* cell_id, int32_t* cell_start,
                   int32_t* members);

/* One sweep (O3).  neighbour_mode 0 = 3^d cells, 1 = all N-1 particles (O6 twin).
 * reverse_cells != 0 visits same-colour cells in descending id (P4 check).
 * follow: GPU trace to lock-step against (O8) or NULL.  trace_out: 2 words per
 * slot (cell*n_select+k) or NULL.  mmin_out: per-slot m_min (NaN if none) or NULL. */
int orc_sweep(orc_sys*, int neighbour_mode, int reverse_cells, const uint32_t* follow, double follow_tol,
              uint32_t* trace_out, double* mmin_out, orc_follow_stats* fs);
int orc_sweeps(orc_sys*, int64_t n);

/* mutation switches for O11-style checks (default all 0 = the real scheme) */
void orc_set_mutations(orc_sys*, int no_shift, int fixed_colour_order, int no_leave_cell_reject);

/* O7: count separating axes / GJK support calls too (extra narrow-phase work; default off) */
void orc_set_work_detail(orc_sys*, int on);
/* n > 1: the cells of one colour as an OpenMP parallel-for (same results, P4); default 1 = serial */
void orc_set_threads(orc_sys*, int n);
int orc_get_threads(const orc_sys*);

/* P:134-138 (domain decomposition): "we modify the checkerboard scheme to have only two regions (active and inactive) ...
 * these particles do not move during substeps".  Reading R-strip: the inactive region is a set of whole layers
 * of cells along the LAST axis (rows in 2-D, z-layers in 3-D) of the sweep's shifted grid -- a cell is at least d_max wide,
 * the paper's strip width -- and it moves with the grid shift from sweep to sweep.  mask[k] != 0: the cells of layer k make
 * no trials (and draw no random numbers; every other cell's Philox keys are unchanged).  n must equal the grid's extent
 * along that axis; mask = NULL clears it.  Returns 0, or < 0 on a size mismatch. */
int orc_set_inactive_layers(orc_sys*, const uint8_t* mask, int32_t n);

/* O8 dump: record the trial of `slot` (-1 = off) during the following sweeps; read it back with orc_get_probe */
void orc_set_probe(orc_sys*, int64_t slot);
void orc_get_probe(const orc_sys*, orc_probe* out);

/* O11: textbook Metropolis, n_trials single-particle trials, own RNG tag */
int orc_textbook_trials(orc_sys*, int64_t n_trials);

/* O5: all N(N-1)/2 pairs, strict m < 0 */
int64_t orc_count_overlaps_bruteforce(const orc_sys*);
/* same count through the cell list (shift 0) */
int64_t orc_count_overlaps_cells(const orc_sys*);
/* smallest pair margin in the system through the cell list (diagnostic) */
double orc_min_margin_cells(const orc_sys*);
/* O9: histogram of s = 1 - lambda* in [0, s_max) over all pairs of the current state (5^d cell search) */
int64_t orc_scale_histogram(const orc_sys*, double s_max, int nbins, uint64_t* hist);
/* P4: min centre distance between particles of distinct same-colour cells */
double orc_min_same_colour_distance(const orc_sys*, const float shift[3]);

#ifdef __cplusplus
}
#endif
#endif
