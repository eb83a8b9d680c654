/*
 * hpmc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see hpmc_oracle.h).
 *
 * Serial CPU oracle for the checkerboard Metropolis sweep of hard shapes,
 * arXiv:1509.04692.  P:<n> = /root/reference/PAPER.md line n; R<k>/O<k> = the
 * readings and oracle items listed in DESIGN.md.
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -fPIC -shared  (no fast-math:
 * the fp32 pins need IEEE single operations with no FMA contraction).
 *
 * Threads: serial by default (the definition).  orc_set_threads(n > 1) runs the cells of ONE colour as an
 * OpenMP parallel-for -- the "any order" of O3.4, legal because same-colour cells are independent (P:21,
 * P:59; pinned by the P4 tests); every result is identical to the serial run.  Nothing else is parallel.
 */
#define _DEFAULT_SOURCE 1 /* M_PI under -std=c99 */
#include "hpmc_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define TAG_SHIFT 1u
#define TAG_PERM 2u
#define TAG_TRIAL 3u
#define TAG_TEXTBOOK 5u

/* ------------------------------------------------------------------------ */
/* R3: Philox4x32-10 (counter-based RNG replacing the paper's Saru)  */
/* ------------------------------------------------------------------------ */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R4: both maps are exact in fp32 (24-bit integers times a power of two) */
float orc_u01(uint32_t r) { return (float)(r >> 8) * (1.0f / 16777216.0f); }
float orc_usym(uint32_t r) { return (float)((int32_t)(r >> 8) - 8388608) * (1.0f / 8388608.0f); }

/* ------------------------------------------------------------------------ */
/* small vector helpers (fp64)                                              */
/* ------------------------------------------------------------------------ */
static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static void cross3(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}
static void sub3(const double a[3], const double b[3], double c[3])
{
    c[0] = a[0] - b[0]; c[1] = a[1] - b[1]; c[2] = a[2] - b[2];
}
static double norm3(const double a[3]) { return sqrt(dot3(a, a)); }

/* rotate v by the unit quaternion nearest q = (w,x,y,z):  v' = q v q*   */
static void quat_rotate(const double q_in[4], const double v[3], double out[3])
{
    double nq = sqrt(q_in[0] * q_in[0] + q_in[1] * q_in[1] + q_in[2] * q_in[2] + q_in[3] * q_in[3]);
    double w = q_in[0] / nq, u[3] = {q_in[1] / nq, q_in[2] / nq, q_in[3] / nq};
    double t[3], t2[3];
    cross3(u, v, t);       /* u x v */
    cross3(u, t, t2);      /* u x (u x v) */
    for (int k = 0; k < 3; ++k) out[k] = v[k] + 2.0 * w * t[k] + 2.0 * t2[k];
}

/* Hamilton product a (x) b */
static void quat_mul(const double a[4], const double b[4], double c[4])
{
    c[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    c[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    c[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    c[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}

/* ------------------------------------------------------------------------ */
/* shapes (O1, O4)                                                          */
/* ------------------------------------------------------------------------ */
struct orc_shape {
    int dim, kind;
    double diameter;
    int nverts;
    double verts[ORC_MAX_VERTS][3];
    double dmax;                         /* circumsphere diameter           */
    int nfaces;                          /* polygon edges / distinct polyhedron faces */
    double face_n[ORC_MAX_FACES][3];     /* outward unit normals, body frame      */
    double face_c[ORC_MAX_FACES];        /* n . v on the face                     */
    int nedgedirs;                       /* distinct edge directions (polyhedron) */
    double edge_d[ORC_MAX_EDGES][3];
    int nedges;                          /* all edges of the polyhedron as vertex pairs (core distance of rounded shapes) */
    int edge_v[ORC_MAX_EDGES][2];
    double sweep_r;                      /* P:89 spheropolygon / spheropolyhedron: radius of the disk / sphere swept over
                                            the polygon / polyhedron (the "core"); 0 = the sharp shape */
};

static int derive_polygon(orc_shape* s)
{
    int n = s->nverts;
    if (n < 3) return -1;
    s->nfaces = n;
    for (int k = 0; k < n; ++k) {
        const double* a = s->verts[k];
        const double* b = s->verts[(k + 1) % n];
        const double* c = s->verts[(k + 2) % n];
        double e[3], e2[3], z[3];
        sub3(b, a, e);
        sub3(c, b, e2);
        cross3(e, e2, z);
        if (!(z[2] > 0.0)) return -1; /* not strictly convex / not CCW (R17) */
        double len = norm3(e);
        if (!(len > 0.0)) return -1;
        s->face_n[k][0] = e[1] / len; /* outward normal of a CCW edge */
        s->face_n[k][1] = -e[0] / len;
        s->face_n[k][2] = 0.0;
        s->face_c[k] = dot3(s->face_n[k], a);
    }
    s->nedgedirs = 0;
    return 0;
}

/* brute force: every vertex triple whose plane has all vertices on one side (O4) */
static int derive_polyhedron(orc_shape* s)
{
    const double tol = 1e-9;
    int n = s->nverts;
    if (n < 4) return -1;
    s->nfaces = 0;
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j)
            for (int k = j + 1; k < n; ++k) {
                double e1[3], e2[3], nn[3];
                sub3(s->verts[j], s->verts[i], e1);
                sub3(s->verts[k], s->verts[i], e2);
                cross3(e1, e2, nn);
                double len = norm3(nn);
                if (len < 1e-12) continue;
                for (int c = 0; c < 3; ++c) nn[c] /= len;
                double off = dot3(nn, s->verts[i]);
                int npos = 0, nneg = 0;
                for (int l = 0; l < n; ++l) {
                    double dd = dot3(nn, s->verts[l]) - off;
                    if (dd > tol) ++npos;
                    if (dd < -tol) ++nneg;
                }
                if (npos > 0 && nneg > 0) continue; /* not a supporting plane */
                if (npos > 0) { /* all others on the + side: outward is -nn */
                    for (int c = 0; c < 3; ++c) nn[c] = -nn[c];
                    off = -off;
                }
                int dup = 0;
                for (int f = 0; f < s->nfaces; ++f)
                    if (dot3(nn, s->face_n[f]) > 1.0 - 1e-10) { dup = 1; break; }
                if (dup) continue;
                if (s->nfaces >= ORC_MAX_FACES) return -1;
                memcpy(s->face_n[s->nfaces], nn, sizeof nn);
                s->face_c[s->nfaces] = off;
                ++s->nfaces;
            }
    if (s->nfaces < 4) return -1;
    /* every listed vertex must be a hull vertex (lie on >= 3 faces) */
    for (int l = 0; l < n; ++l) {
        int on = 0;
        for (int f = 0; f < s->nfaces; ++f)
            if (fabs(dot3(s->face_n[f], s->verts[l]) - s->face_c[f]) < tol) ++on;
        if (on < 3) return -1;
    }
    /* edges: vertex pairs sharing >= 2 faces; keep distinct directions (up to sign) */
    s->nedgedirs = 0;
    s->nedges = 0;
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j) {
            int shared = 0;
            for (int f = 0; f < s->nfaces; ++f)
                if (fabs(dot3(s->face_n[f], s->verts[i]) - s->face_c[f]) < tol &&
                    fabs(dot3(s->face_n[f], s->verts[j]) - s->face_c[f]) < tol)
                    ++shared;
            if (shared < 2) continue;
            if (s->nedges >= ORC_MAX_EDGES) return -1;
            s->edge_v[s->nedges][0] = i;
            s->edge_v[s->nedges][1] = j;
            ++s->nedges;
            double e[3];
            sub3(s->verts[j], s->verts[i], e);
            double len = norm3(e);
            for (int c = 0; c < 3; ++c) e[c] /= len;
            int dup = 0;
            for (int q = 0; q < s->nedgedirs; ++q)
                if (fabs(dot3(e, s->edge_d[q])) > 1.0 - 1e-10) { dup = 1; break; }
            if (dup) continue;
            if (s->nedgedirs >= ORC_MAX_EDGES) return -1;
            memcpy(s->edge_d[s->nedgedirs], e, sizeof e);
            ++s->nedgedirs;
        }
    return 0;
}

static orc_shape* shape_create(int dim, int kind, double diameter, int nverts, const double* verts, double sweep_r);
orc_shape* orc_shape_create(int dim, int kind, double diameter, int nverts, const double* verts)
{
    return shape_create(dim, kind, diameter, nverts, verts, 0.0);
}
/* P:89 "spheropolygons ... convex spheropolyhedra": the polygon / polyhedron swept by a disk / sphere of radius sweep_r */
orc_shape* orc_shape_create_rounded(int dim, int kind, double sweep_r, int nverts, const double* verts)
{
    if (kind != ORC_KIND_POLYGON && kind != ORC_KIND_POLYHEDRON) return NULL;
    if (!(sweep_r >= 0.0)) return NULL;
    return shape_create(dim, kind, 0.0, nverts, verts, sweep_r);
}
static orc_shape* shape_create(int dim, int kind, double diameter, int nverts, const double* verts, double sweep_r)
{
    if (dim != 2 && dim != 3) return NULL;
    orc_shape* s = (orc_shape*)calloc(1, sizeof *s);
    s->dim = dim;
    s->kind = kind;
    int rc = 0;
    if (kind == ORC_KIND_DISK) {
        if (!(diameter > 0.0)) rc = -1;
        s->diameter = diameter;
        s->dmax = diameter;
    } else if (kind == ORC_KIND_POLYGON || kind == ORC_KIND_POLYHEDRON) {
        int vd = (kind == ORC_KIND_POLYGON) ? 2 : 3;
        if ((kind == ORC_KIND_POLYGON && dim != 2) || (kind == ORC_KIND_POLYHEDRON && dim != 3) ||
            nverts < 3 || nverts > ORC_MAX_VERTS || !verts)
            rc = -1;
        else {
            s->nverts = nverts;
            double rmax = 0.0;
            for (int i = 0; i < nverts; ++i) {
                for (int c = 0; c < 3; ++c) s->verts[i][c] = (c < vd) ? verts[i * vd + c] : 0.0;
                double r = norm3(s->verts[i]);
                if (r > rmax) rmax = r;
            }
            s->sweep_r = sweep_r;
            s->dmax = 2.0 * (rmax + sweep_r); /* "diameter of the sphere that encloses particle i, centered on r_i" P:59 */
            rc = (kind == ORC_KIND_POLYGON) ? derive_polygon(s) : derive_polyhedron(s);
        }
    } else
        rc = -1;
    if (rc != 0) { free(s); return NULL; }
    return s;
}

void orc_shape_destroy(orc_shape* s) { free(s); }
double orc_shape_dmax(const orc_shape* s) { return s->dmax; }
double orc_shape_sweep_radius(const orc_shape* s) { return s->sweep_r; }
int orc_shape_nfaces(const orc_shape* s) { return s->nfaces; }
int orc_shape_nedgedirs(const orc_shape* s) { return s->nedgedirs; }
void orc_shape_faces(const orc_shape* s, double* normals3, double* offsets)
{
    for (int f = 0; f < s->nfaces; ++f) {
        for (int c = 0; c < 3; ++c) normals3[3 * f + c] = s->face_n[f][c];
        offsets[f] = s->face_c[f];
    }
}

/* support height h_X(u) = max over X's world-oriented vertices of u . v   (O4) */
static double support_height(double (*wv)[3], int n, const double u[3])
{
    double h = -INFINITY;
    for (int i = 0; i < n; ++i) {
        double d = dot3(u, wv[i]);
        if (d > h) h = d;
    }
    return h;
}

/* separation along the unit direction nhat read "from A toward B":
 *   nhat . r_AB - h_A(nhat) - h_B(-nhat)                                  (O4) */
static double axis_separation(const double nhat[3], const double r_ab[3], double (*wa)[3], double (*wb)[3], int nv)
{
    double neg[3] = {-nhat[0], -nhat[1], -nhat[2]};
    return dot3(nhat, r_ab) - support_height(wa, nv, nhat) - support_height(wb, nv, neg);
}

/* ---- Euclidean distance between two DISJOINT convex cores, by brute force over feature pairs (rounded shapes) ----
 * The closest points of two disjoint convex polygons are a vertex of one and a point of an edge of the other; of two
 * disjoint convex polyhedra, a vertex of one and a point of a face of the other, or points of two edges.  A vertex whose
 * foot on a face plane falls outside the face is closer to one of the face's edges, which the edge-edge pairs cover (every
 * vertex is the end of an edge). */
static double point_segment_distance(const double p[3], const double a[3], const double b[3])
{
    double ab[3], ap[3], c[3];
    sub3(b, a, ab);
    sub3(p, a, ap);
    double t = dot3(ap, ab) / dot3(ab, ab);
    if (t < 0.0) t = 0.0;
    if (t > 1.0) t = 1.0;
    for (int k = 0; k < 3; ++k) c[k] = a[k] + t * ab[k] - p[k];
    return norm3(c);
}

/* min over (s, t) in [0,1]^2 of |a0 + s (a1-a0) - b0 - t (b1-b0)|: a convex function on a square has its minimum at an
 * interior stationary point or on one of the four sides, and each side is a point-segment problem */
static double segment_segment_distance(const double a0[3], const double a1[3], const double b0[3], const double b1[3])
{
    double best = point_segment_distance(a0, b0, b1);
    double d = point_segment_distance(a1, b0, b1);
    if (d < best) best = d;
    d = point_segment_distance(b0, a0, a1);
    if (d < best) best = d;
    d = point_segment_distance(b1, a0, a1);
    if (d < best) best = d;
    double u[3], v[3], w[3];
    sub3(a1, a0, u);
    sub3(b1, b0, v);
    sub3(a0, b0, w);
    double uu = dot3(u, u), uv = dot3(u, v), vv = dot3(v, v), uw = dot3(u, w), vw = dot3(v, w);
    double den = uu * vv - uv * uv;
    if (den > 1e-14 * uu * vv) { /* not parallel: the stationary point of the two infinite lines */
        double sc = (uv * vw - vv * uw) / den, tc = (uu * vw - uv * uw) / den;
        if (sc > 0.0 && sc < 1.0 && tc > 0.0 && tc < 1.0) {
            double c[3];
            for (int k = 0; k < 3; ++k) c[k] = w[k] + sc * u[k] - tc * v[k];
            d = norm3(c);
            if (d < best) best = d;
        }
    }
    return best;
}

/* wa, wb: world-oriented vertices about each body origin; B's origin sits at r_ab from A's */
static double core_distance(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4], double (*wa)[3],
                            double (*wb)[3])
{
    int nv = s->nverts;
    double pb[ORC_MAX_VERTS][3]; /* B's vertices seen from A's origin */
    for (int i = 0; i < nv; ++i)
        for (int k = 0; k < 3; ++k) pb[i][k] = wb[i][k] + r_ab[k];
    double best = INFINITY;
    if (s->kind == ORC_KIND_POLYGON) {
        for (int i = 0; i < nv; ++i)
            for (int e = 0; e < nv; ++e) {
                double d1 = point_segment_distance(pb[i], wa[e], wa[(e + 1) % nv]);
                double d2 = point_segment_distance(wa[i], pb[e], pb[(e + 1) % nv]);
                if (d1 < best) best = d1;
                if (d2 < best) best = d2;
            }
        return best;
    }
    for (int e = 0; e < s->nedges; ++e)
        for (int f = 0; f < s->nedges; ++f) {
            double d = segment_segment_distance(wa[s->edge_v[e][0]], wa[s->edge_v[e][1]], pb[s->edge_v[f][0]], pb[s->edge_v[f][1]]);
            if (d < best) best = d;
        }
    /* vertex above the inside of a face: the foot p - (n.p - c) n satisfies every other face inequality of that body */
    for (int side = 0; side < 2; ++side) {
        const double* q = side == 0 ? qa : qb;
        for (int f = 0; f < s->nfaces; ++f) {
            double n[3];
            quat_rotate(q, s->face_n[f], n);
            for (int i = 0; i < nv; ++i) {
                double p[3]; /* the other body's vertex relative to this body's origin */
                for (int k = 0; k < 3; ++k) p[k] = side == 0 ? pb[i][k] : wa[i][k] - r_ab[k];
                double h = dot3(n, p) - s->face_c[f];
                if (h < 0.0) continue;
                double foot[3];
                for (int k = 0; k < 3; ++k) foot[k] = p[k] - h * n[k];
                int inside = 1;
                for (int g = 0; g < s->nfaces && inside; ++g) {
                    if (g == f) continue;
                    double ng[3];
                    quat_rotate(q, s->face_n[g], ng);
                    if (dot3(ng, foot) > s->face_c[g]) inside = 0;
                }
                if (inside && h < best) best = h;
            }
        }
    }
    return best;
}

static double sharp_margin(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4]);

/* margin of the pair: < 0 iff the interiors intersect.  Sharp shapes: the separating-axis margin (O4).  Rounded shapes
 * (sweep_r > 0): A (+) ball(r) and B (+) ball(r) intersect iff the cores are closer than 2 r, so
 * m = D(core A, core B) - 2 r with D the Euclidean distance of disjoint cores and the (non-positive) separating-axis margin
 * of cores that touch or intersect (continuous: both vanish at contact). */
double orc_shape_margin(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4])
{
    double m = sharp_margin(s, r_ab, qa, qb);
    if (s->kind == ORC_KIND_DISK || !(s->sweep_r > 0.0)) return m;
    if (m > 0.0) {
        double wa[ORC_MAX_VERTS][3], wb[ORC_MAX_VERTS][3];
        for (int i = 0; i < s->nverts; ++i) {
            quat_rotate(qa, s->verts[i], wa[i]);
            quat_rotate(qb, s->verts[i], wb[i]);
        }
        m = core_distance(s, r_ab, qa, qb, wa, wb);
    }
    return m - 2.0 * s->sweep_r;
}

static double sharp_margin(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4])
{
    if (s->kind == ORC_KIND_DISK) return norm3(r_ab) - s->diameter;

    double wa[ORC_MAX_VERTS][3], wb[ORC_MAX_VERTS][3];
    int nv = s->nverts;
    for (int i = 0; i < nv; ++i) {
        quat_rotate(qa, s->verts[i], wa[i]);
        quat_rotate(qb, s->verts[i], wb[i]);
    }
    double m = -INFINITY;
    /* outward face (edge) normals of A, and negated outward normals of B */
    for (int f = 0; f < s->nfaces; ++f) {
        double na[3], nb[3];
        quat_rotate(qa, s->face_n[f], na);
        quat_rotate(qb, s->face_n[f], nb);
        for (int c = 0; c < 3; ++c) nb[c] = -nb[c];
        double sa = axis_separation(na, r_ab, wa, wb, nv);
        double sb = axis_separation(nb, r_ab, wa, wb, nv);
        if (sa > m) m = sa;
        if (sb > m) m = sb;
    }
    if (s->kind == ORC_KIND_POLYHEDRON) {
        /* +- normalised edge_A x edge_B for all edge-direction pairs */
        for (int i = 0; i < s->nedgedirs; ++i) {
            double ea[3];
            quat_rotate(qa, s->edge_d[i], ea);
            for (int j = 0; j < s->nedgedirs; ++j) {
                double eb[3], n[3];
                quat_rotate(qb, s->edge_d[j], eb);
                cross3(ea, eb, n);
                double len = norm3(n);
                if (len < 1e-9) continue; /* near-parallel edges give no new axis */
                for (int c = 0; c < 3; ++c) n[c] /= len;
                double sp = axis_separation(n, r_ab, wa, wb, nv);
                for (int c = 0; c < 3; ++c) n[c] = -n[c];
                double sn = axis_separation(n, r_ab, wa, wb, nv);
                if (sp > m) m = sp;
                if (sn > m) m = sn;
            }
        }
    }
    return m;
}

/* O9 ("histogram of scale factors s that cause two neighboring particles to overlap"): the scale
 * lambda* of the separation vector at which the pair first touches.  With the O4 axis set,
 * m(lambda r) = max_n [lambda n.r - H_n], H_n = h_A(n) + h_B(-n) > 0, so the pair overlaps iff
 * lambda < lambda* = min over axes with n.r > 0 of H_n / (n.r).  Disks: lambda* = sigma / |r|.
 * A pair overlaps after a uniform compression of all separations by (1 - s) iff s > 1 - lambda*. */
static void touch_axis(const double nhat[3], const double r_ab[3], double (*wa)[3], double (*wb)[3], int nv, double* best)
{
    double nr = dot3(nhat, r_ab);
    if (nr <= 0.0) return;
    double neg[3] = {-nhat[0], -nhat[1], -nhat[2]};
    double lam = (support_height(wa, nv, nhat) + support_height(wb, nv, neg)) / nr;
    if (lam < *best) *best = lam;
}

double orc_shape_touch_scale(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4])
{
    if (s->kind == ORC_KIND_DISK) return s->diameter / norm3(r_ab);
    if (s->sweep_r > 0.0) {
        /* rounded shapes: m(lambda r) is not piecewise linear in lambda; the pair overlaps iff lambda r lies inside the
         * convex set B (-) A, which contains the origin, so m changes sign once on the ray: bisection on [0, d_max / |r|] */
        double lo = 0.0, hi = s->dmax / norm3(r_ab);
        for (int it = 0; it < 100; ++it) {
            double mid = 0.5 * (lo + hi), rr[3] = {mid * r_ab[0], mid * r_ab[1], mid * r_ab[2]};
            if (orc_shape_margin(s, rr, qa, qb) < 0.0) lo = mid; else hi = mid;
        }
        return 0.5 * (lo + hi);
    }
    double wa[ORC_MAX_VERTS][3], wb[ORC_MAX_VERTS][3];
    int nv = s->nverts;
    for (int i = 0; i < nv; ++i) {
        quat_rotate(qa, s->verts[i], wa[i]);
        quat_rotate(qb, s->verts[i], wb[i]);
    }
    double best = INFINITY;
    for (int f = 0; f < s->nfaces; ++f) {
        double na[3], nb[3];
        quat_rotate(qa, s->face_n[f], na);
        quat_rotate(qb, s->face_n[f], nb);
        for (int c = 0; c < 3; ++c) nb[c] = -nb[c];
        touch_axis(na, r_ab, wa, wb, nv, &best);
        touch_axis(nb, r_ab, wa, wb, nv, &best);
    }
    if (s->kind == ORC_KIND_POLYHEDRON) {
        for (int i = 0; i < s->nedgedirs; ++i) {
            double ea[3];
            quat_rotate(qa, s->edge_d[i], ea);
            for (int j = 0; j < s->nedgedirs; ++j) {
                double eb[3], n[3];
                quat_rotate(qb, s->edge_d[j], eb);
                cross3(ea, eb, n);
                double len = norm3(n);
                if (len < 1e-9) continue;
                for (int c = 0; c < 3; ++c) n[c] /= len;
                touch_axis(n, r_ab, wa, wb, nv, &best);
                for (int c = 0; c < 3; ++c) n[c] = -n[c];
                touch_axis(n, r_ab, wa, wb, nv, &best);
            }
        }
    }
    return best;
}

/* ---- fp64 GJK boolean on the Minkowski difference B (-) A, support by Eq. (1) P:97 ---- */
typedef struct { double (*wa)[3]; double (*wb)[3]; int nv; const double* r; } gjk_ctx;

static void gjk_support(const gjk_ctx* g, const double d[3], double out[3])
{
    /* S_{B-A}(d) = S_B(d) - S_A(-d), world frame, B displaced by r_AB */
    int ib = 0, ia = 0;
    double best_b = -INFINITY, best_a = -INFINITY;
    for (int i = 0; i < g->nv; ++i) {
        double db = dot3(d, g->wb[i]);
        double da = -dot3(d, g->wa[i]);
        if (db > best_b) { best_b = db; ib = i; }
        if (da > best_a) { best_a = da; ia = i; }
    }
    for (int c = 0; c < 3; ++c) out[c] = g->wb[ib][c] + g->r[c] - g->wa[ia][c];
}

static void triple_cross(const double a[3], const double b[3], const double c[3], double out[3])
{
    double t[3];
    cross3(a, b, t);
    cross3(t, c, out); /* (a x b) x c */
}

/* GJK sub-steps.  P[np-1] is always the newest support point "a".  Every
 * perpendicular is oriented explicitly against the opposite simplex vertex, so
 * no winding convention has to be maintained.  Return 1 = origin enclosed. */
static int gjk_line(double P[4][3], int* np, double d[3])
{
    const double* a = P[1];
    double ab[3], ao[3] = {-a[0], -a[1], -a[2]};
    sub3(P[0], a, ab);
    triple_cross(ab, ao, ab, d); /* perpendicular to ab, toward the origin */
    *np = 2;
    return dot3(d, d) < 1e-30;   /* origin on the segment's line */
}

static int gjk_triangle(double P[4][3], int* np, double d[3], int dim)
{
    double a[3], b[3], c[3];
    memcpy(a, P[2], sizeof a); memcpy(b, P[1], sizeof b); memcpy(c, P[0], sizeof c);
    double ab[3], ac[3], ao[3] = {-a[0], -a[1], -a[2]}, n[3], e[3];
    sub3(b, a, ab);
    sub3(c, a, ac);
    cross3(ab, ac, n);
    cross3(ab, n, e);                        /* in-plane perpendicular of ab ...      */
    if (dot3(e, ac) > 0.0) for (int k = 0; k < 3; ++k) e[k] = -e[k]; /* ... away from c */
    if (dot3(e, ao) > 0.0) {                 /* origin beyond edge ab: drop c         */
        memcpy(P[0], b, sizeof b); memcpy(P[1], a, sizeof a);
        return gjk_line(P, np, d);
    }
    cross3(n, ac, e);
    if (dot3(e, ab) > 0.0) for (int k = 0; k < 3; ++k) e[k] = -e[k]; /* away from b   */
    if (dot3(e, ao) > 0.0) {                 /* origin beyond edge ac: drop b         */
        memcpy(P[0], c, sizeof c); memcpy(P[1], a, sizeof a);
        return gjk_line(P, np, d);
    }
    if (dim == 2) return 1;                  /* planar: inside all three edges        */
    double side = dot3(n, ao);
    if (side == 0.0) return 1;               /* origin in the triangle itself         */
    for (int k = 0; k < 3; ++k) d[k] = (side > 0.0) ? n[k] : -n[k];
    *np = 3;
    return 0;
}

static int gjk_tetrahedron(double P[4][3], int* np, double d[3])
{
    double a[3], b[3], c[3], dd[3];
    memcpy(a, P[3], sizeof a); memcpy(b, P[2], sizeof b); memcpy(c, P[1], sizeof c); memcpy(dd, P[0], sizeof dd);
    double ab[3], ac[3], ad[3], ao[3] = {-a[0], -a[1], -a[2]};
    sub3(b, a, ab); sub3(c, a, ac); sub3(dd, a, ad);
    double n[3][3];
    cross3(ab, ac, n[0]); if (dot3(n[0], ad) > 0.0) for (int k = 0; k < 3; ++k) n[0][k] = -n[0][k]; /* face abc, away from d */
    cross3(ac, ad, n[1]); if (dot3(n[1], ab) > 0.0) for (int k = 0; k < 3; ++k) n[1][k] = -n[1][k]; /* face acd, away from b */
    cross3(ad, ab, n[2]); if (dot3(n[2], ac) > 0.0) for (int k = 0; k < 3; ++k) n[2][k] = -n[2][k]; /* face adb, away from c */
    double out[3];
    int best = -1;
    for (int f = 0; f < 3; ++f) {
        double len = norm3(n[f]);
        out[f] = (len > 0.0) ? dot3(n[f], ao) / len : -INFINITY;
        if (out[f] > 0.0 && (best < 0 || out[f] > out[best])) best = f;
    }
    if (best < 0) return 1; /* behind all three new faces; the base face was crossed to get here */
    const double* p = (best == 0) ? b : (best == 1) ? c : dd;
    const double* q = (best == 0) ? c : (best == 1) ? dd : b;
    double pp[3], qq[3];
    memcpy(pp, p, sizeof pp); memcpy(qq, q, sizeof qq);
    memcpy(P[0], qq, sizeof qq); memcpy(P[1], pp, sizeof pp); memcpy(P[2], a, sizeof a);
    return gjk_triangle(P, np, d, 3);
}

/* support_calls (may be NULL): number of support-function evaluations (Eq. (1)), O7 */
static int gjk_run(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4], uint64_t* support_calls)
{
    if (s->kind == ORC_KIND_DISK) return (norm3(r_ab) - s->diameter) < 0.0 ? 1 : 0;
    double wa[ORC_MAX_VERTS][3], wb[ORC_MAX_VERTS][3];
    for (int i = 0; i < s->nverts; ++i) {
        quat_rotate(qa, s->verts[i], wa[i]);
        quat_rotate(qb, s->verts[i], wb[i]);
    }
    gjk_ctx g = {wa, wb, s->nverts, r_ab};
    double P[4][3]; /* simplex, newest point last */
    int np = 0;
    double d[3] = {-r_ab[0], -r_ab[1], -r_ab[2]}; /* from the centre of B (-) A toward the origin */
    if (dot3(d, d) < 1e-24) { d[0] = 1.0; d[1] = 0.0; d[2] = 0.0; }
    for (int iter = 0; iter < 256; ++iter) {
        double a[3];
        gjk_support(&g, d, a);
        if (support_calls) ++*support_calls;
        if (dot3(a, d) <= 0.0) return 0; /* a support plane separates the origin: disjoint (touching counts as disjoint) */
        memcpy(P[np++], a, sizeof a);
        int hit;
        if (np == 1) { for (int k = 0; k < 3; ++k) d[k] = -a[k]; hit = dot3(d, d) < 1e-30; }
        else if (np == 2) hit = gjk_line(P, &np, d);
        else if (np == 3) hit = gjk_triangle(P, &np, d, s->dim);
        else hit = gjk_tetrahedron(P, &np, d);
        if (hit) return 1;
    }
    return -1;
}

int orc_shape_gjk(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4])
{
    if (s->sweep_r > 0.0) return -1; /* the cross-check GJK runs on vertex sets only */
    return gjk_run(s, r_ab, qa, qb, NULL);
}

/* O7: separating axes of a convex polygon pair evaluated in serial order -- the outward edge normals of A
 * (k = 0..n-1), then the negated edge normals of B -- until the first axis whose separation is >= eps
 * ("separating planes method"); all 2n when none separates (the pair overlaps). */
static int polygon_axes_until_separation(const orc_shape* s, const double r_ab[3], const double qa[4], const double qb[4], double eps)
{
    double wa[ORC_MAX_VERTS][3], wb[ORC_MAX_VERTS][3];
    int nv = s->nverts, count = 0;
    for (int i = 0; i < nv; ++i) {
        quat_rotate(qa, s->verts[i], wa[i]);
        quat_rotate(qb, s->verts[i], wb[i]);
    }
    for (int side = 0; side < 2; ++side)
        for (int f = 0; f < s->nfaces; ++f) {
            double n[3];
            quat_rotate(side == 0 ? qa : qb, s->face_n[f], n);
            if (side == 1) for (int c = 0; c < 3; ++c) n[c] = -n[c];
            ++count;
            if (axis_separation(n, r_ab, wa, wb, nv) >= eps) return count;
        }
    return count;
}

/* ------------------------------------------------------------------------ */
/* system (O1, O2)                                                          */
/* ------------------------------------------------------------------------ */
struct orc_sys {
    int dim;
    double L[3];   /* box edge, ALREADY rounded to fp32 (DESIGN.md R-box) */
    float L_f[3], lo_f[3], hi_f[3];
    int64_t N;
    float* pos;    /* N*4: x,y,z,0 */
    float* quat;   /* N*4: w,x,y,z */
    orc_shape* shape;
    int32_t n[3];
    double w[3];
    float w_f[3], inv_w[3];
    int64_t C;
    double d, a;
    float d_f, a_f;
    int n_select;
    double eps_g;
    uint64_t seed, t, tb_count;
    orc_counters cnt;
    orc_work work;
    int mut_no_shift, mut_fixed_order, mut_no_leave;
    int work_detail; /* O7: also count separating axes / GJK support calls (costs extra narrow-phase work) */
    int nthreads;    /* 1 = serial (the definition); > 1 = same-colour cells as an OpenMP parallel-for */
    uint8_t* inactive;   /* P:136-138 inactive region: layers of cells along the last axis that make no trials this sweep; NULL = none */
    int64_t probe_slot;      /* O8 "FAIL with a dump": trial slot whose pose and candidates are recorded, -1 = none */
    orc_probe probe;
    int32_t *cell_id, *cell_start, *members;
};

static orc_sys* sys_create(orc_shape* sh, int dim, const double L[3], int64_t N, uint64_t seed);
orc_sys* orc_create(int dim, const double L[3], int kind, double diameter, int nverts, const double* verts,
                    int64_t N, uint64_t seed)
{
    return sys_create(orc_shape_create(dim, kind, diameter, nverts, verts), dim, L, N, seed);
}
orc_sys* orc_create_rounded(int dim, const double L[3], int kind, double sweep_r, int nverts, const double* verts,
                            int64_t N, uint64_t seed)
{
    return sys_create(orc_shape_create_rounded(dim, kind, sweep_r, nverts, verts), dim, L, N, seed);
}
static orc_sys* sys_create(orc_shape* sh, int dim, const double L[3], int64_t N, uint64_t seed)
{
    if (!sh) return NULL;
    orc_sys* s = (orc_sys*)calloc(1, sizeof *s);
    s->dim = dim;
    s->shape = sh;
    s->N = N;
    s->seed = seed;
    s->eps_g = 2e-6; /* R15 */
    s->C = 1;
    for (int k = 0; k < 3; ++k) {
        if (k < dim) {
            s->L_f[k] = (float)L[k];
            s->L[k] = (double)s->L_f[k];
            /* O2 / R11: even count, cell width >= d_max + slack, at least 4 cells.  slack = d_max 2^-10, or 3 ulp_fp32(L) in
             * boxes so large that the fp32 rounding of cell_of (R13) would eat the former (R11); the two coincide
             * for every config of BASELINE.json. */
            {
                int e = 0;
                frexp(nextafter(s->L[k], 0.0), &e);
                double ulp = ldexp(1.0, e - 24);
                double slack = fmax(sh->dmax / 1024.0, 3.0 * ulp);
                s->n[k] = 2 * (int32_t)floor(s->L[k] / (2.0 * (sh->dmax + slack)));
            }
            if (s->n[k] < 4) { orc_shape_destroy(sh); free(s); return NULL; }
            s->w[k] = s->L[k] / s->n[k];
            s->w_f[k] = (float)s->w[k];
            s->inv_w[k] = (float)((double)s->n[k] / s->L[k]);
        } else {
            s->L_f[k] = 1.0f; s->L[k] = 1.0; s->n[k] = 1; s->w[k] = 1.0; s->w_f[k] = 1.0f; s->inv_w[k] = 1.0f;
        }
        s->hi_f[k] = 0.5f * s->L_f[k]; /* exact */
        s->lo_f[k] = -s->hi_f[k];
        s->C *= s->n[k];
    }
    s->pos = (float*)calloc((size_t)(N > 0 ? N : 1) * 4, sizeof(float));
    s->quat = (float*)calloc((size_t)(N > 0 ? N : 1) * 4, sizeof(float));
    for (int64_t i = 0; i < N; ++i) s->quat[4 * i] = 1.0f;
    s->cell_id = (int32_t*)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    s->members = (int32_t*)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
    s->cell_start = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->C + 1));
    s->d = 0.1; s->a = 0.1; s->d_f = 0.1f; s->a_f = 0.1f; s->n_select = 4;
    s->nthreads = 1;
    s->probe_slot = -1;
    return s;
}

void orc_destroy(orc_sys* s)
{
    if (!s) return;
    free(s->pos); free(s->quat); free(s->cell_id); free(s->members); free(s->cell_start); free(s->inactive);
    orc_shape_destroy(s->shape);
    free(s);
}

const orc_shape* orc_sys_shape(const orc_sys* s) { return s->shape; }

int orc_set_moves(orc_sys* s, double d, double a, int n_select)
{
    if (!(d > 0.0) || a < 0.0 || n_select < 1 || n_select > 65535) return -1;
    s->d = d; s->a = a; s->d_f = (float)d; s->a_f = (float)a; s->n_select = n_select;
    return 0;
}
void orc_set_eps_guard(orc_sys* s, double e) { s->eps_g = e; }
void orc_set_state(orc_sys* s, const float* p, const float* q)
{
    memcpy(s->pos, p, sizeof(float) * 4 * (size_t)s->N);
    memcpy(s->quat, q, sizeof(float) * 4 * (size_t)s->N);
}
void orc_get_state(const orc_sys* s, float* p, float* q)
{
    memcpy(p, s->pos, sizeof(float) * 4 * (size_t)s->N);
    memcpy(q, s->quat, sizeof(float) * 4 * (size_t)s->N);
}
void orc_set_sweep_counter(orc_sys* s, uint64_t t) { s->t = t; }
uint64_t orc_get_sweep_counter(const orc_sys* s) { return s->t; }
void orc_get_counters(const orc_sys* s, orc_counters* c) { *c = s->cnt; }
void orc_get_work(const orc_sys* s, orc_work* w) { *w = s->work; }
void orc_reset_counters(orc_sys* s) { memset(&s->cnt, 0, sizeof s->cnt); memset(&s->work, 0, sizeof s->work); }
void orc_get_grid(const orc_sys* s, int32_t n[3], double w[3], float w_f[3], float inv_w[3], float L_f[3])
{
    for (int k = 0; k < 3; ++k) { n[k] = s->n[k]; w[k] = s->w[k]; w_f[k] = s->w_f[k]; inv_w[k] = s->inv_w[k]; L_f[k] = s->L_f[k]; }
}
int64_t orc_num_cells(const orc_sys* s) { return s->C; }
void orc_set_mutations(orc_sys* s, int a, int b, int c) { s->mut_no_shift = a; s->mut_fixed_order = b; s->mut_no_leave = c; }
void orc_set_work_detail(orc_sys* s, int on) { s->work_detail = on; }
void orc_set_threads(orc_sys* s, int n) { s->nthreads = n > 1 ? n : 1; }
int orc_set_inactive_layers(orc_sys* s, const uint8_t* mask, int32_t n)
{
    free(s->inactive);
    s->inactive = NULL;
    if (!mask) return 0;
    if (n != s->n[s->dim - 1]) return -1;
    s->inactive = (uint8_t*)malloc((size_t)n);
    if (!s->inactive) return -2;
    memcpy(s->inactive, mask, (size_t)n);
    return 0;
}
void orc_set_probe(orc_sys* s, int64_t slot) { s->probe_slot = slot; memset(&s->probe, 0, sizeof s->probe); s->probe.slot = -1; }
void orc_get_probe(const orc_sys* s, orc_probe* out) { *out = s->probe; }
int orc_get_threads(const orc_sys* s) { return s->nthreads; }

/* ------------------------------------------------------------------------ */
/* O3.1, O3.2: sweep header                                                 */
/* ------------------------------------------------------------------------ */
void orc_sweep_header(const orc_sys* s, uint64_t t, float shift[3], int32_t perm[8])
{
    uint32_t key[2] = {(uint32_t)s->seed, (uint32_t)(s->seed >> 32)};
    uint32_t t_lo = (uint32_t)t, t_hi16 = (uint32_t)((t >> 32) & 0xFFFFu);
    uint32_t ctr[4] = {0u, t_lo, 0u, (TAG_SHIFT << 24) | t_hi16};
    uint32_t r[4];
    orc_philox4x32_10(ctr, key, r);
    for (int k = 0; k < 3; ++k) shift[k] = (k < s->dim) ? s->w_f[k] * orc_u01(r[k]) : 0.0f; /* R10: [0,w) */
    int ncol = 1 << s->dim;
    for (int c = 0; c < 8; ++c) perm[c] = c;
    /* R12: Fisher-Yates, i = ncol-1 .. 1, j = mulhi(r, i+1); words taken in order from blocks b = 0,1,.. */
    int word = 0;
    uint32_t blk[4] = {0, 0, 0, 0};
    for (int i = ncol - 1; i >= 1; --i) {
        if ((word & 3) == 0) {
            uint32_t c2[4] = {0u, t_lo, (uint32_t)(word >> 2), (TAG_PERM << 24) | t_hi16};
            orc_philox4x32_10(c2, key, blk);
        }
        uint32_t j = (uint32_t)(((uint64_t)blk[word & 3] * (uint64_t)(i + 1)) >> 32);
        int32_t tmp = perm[i]; perm[i] = perm[j]; perm[j] = tmp;
        ++word;
    }
}

/* R13: pinned fp32 cell function (no FMA: build with -ffp-contract=off) */
static int32_t cell_axis(const orc_sys* s, int k, float x, float shift)
{
    float f = (x - s->lo_f[k]) - shift;
    if (f < 0.0f) f += s->L_f[k];
    if (f >= s->L_f[k]) f -= s->L_f[k];
    int32_t c = (int32_t)floorf(f * s->inv_w[k]);
    if (c >= s->n[k]) c -= s->n[k];
    return c;
}

int32_t orc_cell_of(const orc_sys* s, const float x[3], const float shift[3])
{
    int32_t cx = cell_axis(s, 0, x[0], shift[0]);
    int32_t cy = cell_axis(s, 1, x[1], shift[1]);
    int32_t cz = (s->dim == 3) ? cell_axis(s, 2, x[2], shift[2]) : 0;
    return cx + s->n[0] * (cy + s->n[1] * cz); /* O2 */
}

/* O3.3: members of each cell in ascending particle index (R8) */
void orc_cell_list(const orc_sys* s, const float shift[3], int32_t* cell_id, int32_t* cell_start, int32_t* members)
{
    for (int64_t c = 0; c <= s->C; ++c) cell_start[c] = 0;
    for (int64_t i = 0; i < s->N; ++i) {
        cell_id[i] = orc_cell_of(s, &s->pos[4 * i], shift);
        cell_start[cell_id[i] + 1] += 1;
    }
    for (int64_t c = 0; c < s->C; ++c) cell_start[c + 1] += cell_start[c];
    int32_t* fill = (int32_t*)calloc((size_t)(s->C > 0 ? s->C : 1), sizeof(int32_t));
    for (int64_t i = 0; i < s->N; ++i) { /* ascending i => ascending tag inside each cell */
        int32_t c = cell_id[i];
        members[cell_start[c] + fill[c]++] = (int32_t)i;
    }
    free(fill);
}

/* minimum-image separation x_j - x_trial in fp64 from the fp32 values (O3.4f, R21) */
static void min_image(const orc_sys* s, const float* xj, const float* xt, double r[3])
{
    for (int k = 0; k < 3; ++k) {
        if (k < s->dim) {
            double dx = (double)xj[k] - (double)xt[k];
            dx -= s->L[k] * nearbyint(dx / s->L[k]);
            r[k] = dx;
        } else
            r[k] = 0.0;
    }
}

static void quat_to_double(const float* q, double out[4]) { for (int c = 0; c < 4; ++c) out[c] = (double)q[c]; }

/* scan the candidates of one trial; returns m_min (INFINITY if no candidate in range).  wk: O7 work tallies */
static double scan_candidates(const orc_sys* s, orc_work* wk, orc_probe* probe, int neighbour_mode, int64_t i, const float xt[3],
                              const float qt[4], const int32_t cc[3])
{
    const orc_shape* sh = s->shape;
    double qa[4], m_min = INFINITY;
    quat_to_double(qt, qa);
    int found = 0;
    /* R16': the broad-phase range carries the guard band, so that "reject iff m < eps_g" (R15) also holds for
     * pairs at centre distance d_max (touching disks; polygon vertices pointing at each other) */
    double dmax2 = (sh->dmax + s->eps_g) * (sh->dmax + s->eps_g);
    if (neighbour_mode == 1) { /* O6 twin: all N-1 particles */
        for (int64_t j = 0; j < s->N; ++j) {
            if (j == i) continue;
            double r[3], qb[4];
            min_image(s, &s->pos[4 * j], xt, r);
            if (dot3(r, r) >= dmax2) continue; /* R16 */
            quat_to_double(&s->quat[4 * j], qb);
            double m = orc_shape_margin(sh, r, qa, qb);
            if (m < m_min) m_min = m;
        }
        return m_min;
    }
    int zlo = (s->dim == 3) ? -1 : 0, zhi = (s->dim == 3) ? 1 : 0;
    for (int dz = zlo; dz <= zhi; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) { /* R19: 3^d cells around the owning cell */
                int32_t nx = (cc[0] + dx + s->n[0]) % s->n[0];
                int32_t ny = (cc[1] + dy + s->n[1]) % s->n[1];
                int32_t nz = (cc[2] + dz + s->n[2]) % s->n[2];
                int32_t nc = nx + s->n[0] * (ny + s->n[1] * nz);
                for (int32_t p = s->cell_start[nc]; p < s->cell_start[nc + 1]; ++p) {
                    int64_t j = s->members[p];
                    if (j == i) continue;
                    double r[3], qb[4];
                    wk->cand_scanned_full++;
                    if (!found) wk->cand_scanned_early++;
                    min_image(s, &s->pos[4 * j], xt, r);
                    if (dot3(r, r) >= dmax2) continue; /* R16 circumsphere */
                    wk->sphere_pass_full++;
                    if (!found) wk->narrow_tests_early++;
                    quat_to_double(&s->quat[4 * j], qb);
                    double m = orc_shape_margin(sh, r, qa, qb);
                    if (probe && probe->ncand < ORC_PROBE_MAX) {
                        int c = probe->ncand++;
                        probe->cand[c] = j; probe->margin[c] = m;
                        for (int k = 0; k < 3; ++k) probe->r[c][k] = r[k];
                        for (int k = 0; k < 4; ++k) probe->qb[c][k] = s->quat[4 * j + k];
                    }
                    if (!found && s->work_detail && !(sh->sweep_r > 0.0)) { /* O7: what an early-exit narrow phase would have evaluated */
                        if (sh->kind == ORC_KIND_POLYGON)
                            wk->polygon_axes_early += (uint64_t)polygon_axes_until_separation(sh, r, qa, qb, s->eps_g);
                        else if (sh->kind == ORC_KIND_POLYHEDRON)
                            gjk_run(sh, r, qa, qb, &wk->gjk_support_calls_early);
                    }
                    if (m < m_min) m_min = m;
                    if (m < s->eps_g) found = 1;
                }
            }
    return m_min;
}

/* move generators shared by the checkerboard sweep and the textbook twin (R5, R6) */
static void gen_translate(const orc_sys* s, const float* x, const uint32_t u[3], float xt[3])
{
    for (int k = 0; k < 3; ++k) xt[k] = (k < s->dim) ? fmaf(s->d_f, orc_usym(u[k]), x[k]) : x[k]; /* one rounding */
}

static void gen_rotate(const orc_sys* s, const float* q, uint32_t ua, uint32_t ub, uint32_t uc, float qt[4])
{
    double qd[4], dq[4], qn[4];
    quat_to_double(q, qd);
    if (s->dim == 2) { /* angle uniform in [-a,a) about z */
        float theta = s->a_f * orc_usym(ua);
        double h = 0.5 * (double)theta;
        dq[0] = cos(h); dq[1] = 0.0; dq[2] = 0.0; dq[3] = sin(h);
    } else { /* uniform axis on S^2, angle uniform in [-a,a) */
        double z = (double)orc_usym(ua);
        double phi = 2.0 * M_PI * (double)orc_u01(ub);
        double rho = sqrt(1.0 - z * z);
        float theta = s->a_f * orc_usym(uc);
        double h = 0.5 * (double)theta;
        double sh = sin(h);
        dq[0] = cos(h); dq[1] = sh * rho * cos(phi); dq[2] = sh * rho * sin(phi); dq[3] = sh * z;
    }
    quat_mul(qd, dq, qn); /* q_trial = q_i . dq  (right multiplication, R6) */
    double nn = sqrt(qn[0] * qn[0] + qn[1] * qn[1] + qn[2] * qn[2] + qn[3] * qn[3]);
    for (int c = 0; c < 4; ++c) qt[c] = (float)(qn[c] / nn);
}

static void wrap_store(orc_sys* s, int64_t i, const float xt[3], const float qt[4])
{
    for (int k = 0; k < 3; ++k) { /* O3.4g: one fp32 add if needed */
        float x = xt[k];
        if (k < s->dim) {
            if (x >= s->hi_f[k]) x -= s->L_f[k];
            else if (x < s->lo_f[k]) x += s->L_f[k];
        }
        s->pos[4 * i + k] = x;
    }
    for (int c = 0; c < 4; ++c) s->quat[4 * i + c] = qt[c];
}

/* ------------------------------------------------------------------------ */
/* O3: one checkerboard sweep                                               */
/* ------------------------------------------------------------------------ */
typedef struct { /* everything one cell's trials need to know about the sweep */
    uint32_t key[2], t_lo, t_hi16;
    float shift[3];
    int gamma, neighbour_mode;
    const uint32_t* follow;
    double follow_tol;
    uint32_t* trace_out;
    double* mmin_out;
} sweep_ctx;

static void note_bad(orc_follow_stats* fs, int64_t slot, const uint32_t mine[2], const uint32_t* th, double m_min)
{
    fs->hard_mismatch++;
    if (fs->first_bad_slot < 0) { fs->first_bad_slot = slot; memcpy(fs->first_bad_mine, mine, 8); memcpy(fs->first_bad_theirs, th, 8); fs->first_bad_mmin = m_min; }
}

/* O3.4: the n_select sequential trials of one cell (R9).  Tallies go to the caller's cnt / wk / fs. */
static void sweep_cell(orc_sys* s, const sweep_ctx* x, int64_t cell, const int32_t cc[3], orc_counters* cnt, orc_work* wk,
                       orc_follow_stats* fs)
{
    const int32_t nmem = s->cell_start[cell + 1] - s->cell_start[cell];
    for (int k = 0; k < s->n_select; ++k) {
        const int64_t slot = cell * s->n_select + k;
        uint32_t mine[2] = {0u, 0u};
        double m_min = NAN;
        if (nmem > 0) { /* R9: empty cells make no trials */
            uint32_t ctr[4] = {(uint32_t)cell, x->t_lo, (uint32_t)k, (TAG_TRIAL << 24) | ((uint32_t)x->gamma << 16) | x->t_hi16};
            uint32_t b0[4], b1[4] = {0, 0, 0, 0};
            orc_philox4x32_10(ctr, x->key, b0);
            if (s->dim == 3) { ctr[2] = (uint32_t)k | (1u << 16); orc_philox4x32_10(ctr, x->key, b1); }
            const int64_t i = s->members[s->cell_start[cell] + (int32_t)(((uint64_t)b0[0] * (uint64_t)nmem) >> 32)]; /* R8 */
            const int rotate = (s->shape->kind != ORC_KIND_DISK) && (b0[1] >> 31); /* R7 */
            float xt[3], qt[4];
            int outcome;
            cnt->trials++;
            if (!rotate) {
                uint32_t u[3] = {b0[2], b0[3], b1[0]};
                gen_translate(s, &s->pos[4 * i], u, xt);
                memcpy(qt, &s->quat[4 * i], sizeof qt);
            } else {
                memcpy(xt, &s->pos[4 * i], sizeof xt);
                gen_rotate(s, &s->quat[4 * i], b0[2], b0[3], b1[0], qt);
            }
            if (!rotate && !s->mut_no_leave && orc_cell_of(s, xt, x->shift) != (int32_t)cell) {
                outcome = 2; /* O3.4e: leaves its cell -> reject */
            } else {
                orc_probe* probe = (slot == s->probe_slot) ? &s->probe : NULL;
                if (probe) {
                    probe->slot = slot; probe->particle = i; probe->rotate = rotate; probe->ncand = 0;
                    for (int c = 0; c < 3; ++c) probe->xt[c] = xt[c];
                    for (int c = 0; c < 4; ++c) probe->qt[c] = qt[c];
                }
                m_min = scan_candidates(s, wk, probe, x->neighbour_mode, i, xt, qt, cc);
                outcome = (m_min < s->eps_g) ? 3 : 1; /* R15 guard band */
            }
            mine[0] = (uint32_t)i;
            mine[1] = (uint32_t)rotate | ((uint32_t)outcome << 8);
            if (x->follow) { /* O8 lock-step */
                const uint32_t* th = &x->follow[2 * slot];
                int their_outcome = (int)(th[1] >> 8);
                if (th[0] != mine[0] || (th[1] & 0xFFu) != (mine[1] & 0xFFu)) {
                    note_bad(fs, slot, mine, th, m_min);
                } else if (their_outcome != outcome) {
                    int both_overlap_kind = (outcome == 1 || outcome == 3) && (their_outcome == 1 || their_outcome == 3);
                    if (both_overlap_kind && fabs(m_min - s->eps_g) < x->follow_tol) {
                        fs->marginal++;
                        outcome = their_outcome; /* adopt the GPU's decision and continue */
                    } else
                        note_bad(fs, slot, mine, th, m_min);
                }
                fs->compared++;
            }
            if (outcome == 1) {
                wrap_store(s, i, xt, qt);
                if (rotate) cnt->rot_acc++; else cnt->trans_acc++;
            } else if (outcome == 2) {
                cnt->trans_rej_cell++;
            } else {
                if (rotate) cnt->rot_rej_overlap++; else cnt->trans_rej_overlap++;
            }
        } else if (x->follow) {
            const uint32_t* th = &x->follow[2 * slot];
            if (th[0] != 0u || th[1] != 0u) note_bad(fs, slot, mine, th, NAN);
            fs->compared++;
        }
        if (x->trace_out) { x->trace_out[2 * slot] = mine[0]; x->trace_out[2 * slot + 1] = mine[1]; }
        if (x->mmin_out) x->mmin_out[slot] = m_min;
    }
}

static void add_tallies(orc_sys* s, orc_follow_stats* fs, const orc_counters* c, const orc_work* w, const orc_follow_stats* f)
{
    s->cnt.trans_acc += c->trans_acc; s->cnt.trans_rej_overlap += c->trans_rej_overlap; s->cnt.trans_rej_cell += c->trans_rej_cell;
    s->cnt.rot_acc += c->rot_acc; s->cnt.rot_rej_overlap += c->rot_rej_overlap; s->cnt.trials += c->trials;
    s->work.cand_scanned_full += w->cand_scanned_full; s->work.sphere_pass_full += w->sphere_pass_full;
    s->work.cand_scanned_early += w->cand_scanned_early; s->work.narrow_tests_early += w->narrow_tests_early;
    s->work.polygon_axes_early += w->polygon_axes_early; s->work.gjk_support_calls_early += w->gjk_support_calls_early;
    fs->compared += f->compared; fs->marginal += f->marginal; fs->hard_mismatch += f->hard_mismatch;
    if (f->first_bad_slot >= 0 && (fs->first_bad_slot < 0 || f->first_bad_slot < fs->first_bad_slot)) {
        fs->first_bad_slot = f->first_bad_slot; fs->first_bad_mmin = f->first_bad_mmin;
        memcpy(fs->first_bad_mine, f->first_bad_mine, 8); memcpy(fs->first_bad_theirs, f->first_bad_theirs, 8);
    }
}

int orc_sweep(orc_sys* s, int neighbour_mode, int reverse_cells, const uint32_t* follow, double follow_tol,
              uint32_t* trace_out, double* mmin_out, orc_follow_stats* fs)
{
    const uint64_t t = s->t;
    sweep_ctx x;
    x.key[0] = (uint32_t)s->seed; x.key[1] = (uint32_t)(s->seed >> 32);
    x.t_lo = (uint32_t)t; x.t_hi16 = (uint32_t)((t >> 32) & 0xFFFFu);
    x.neighbour_mode = neighbour_mode; x.follow = follow; x.follow_tol = follow_tol; x.trace_out = trace_out; x.mmin_out = mmin_out;
    int32_t perm[8];
    orc_sweep_header(s, t, x.shift, perm);
    if (s->mut_no_shift) x.shift[0] = x.shift[1] = x.shift[2] = 0.0f;
    if (s->mut_fixed_order) for (int c = 0; c < 8; ++c) perm[c] = c;
    orc_cell_list(s, x.shift, s->cell_id, s->cell_start, s->members);
    const int ncol = 1 << s->dim;
    const int64_t nslots = s->C * s->n_select;
    if (trace_out) memset(trace_out, 0, sizeof(uint32_t) * 2 * (size_t)nslots);
    if (mmin_out) for (int64_t q = 0; q < nslots; ++q) mmin_out[q] = NAN;
    orc_follow_stats fs_local;
    if (!fs) fs = &fs_local;
    memset(fs, 0, sizeof *fs);
    fs->first_bad_slot = -1;

    for (int ci = 0; ci < ncol; ++ci) {
        x.gamma = perm[ci];
        /* every cell of colour gamma, in ascending (or descending) id when serial; "any order" is legal (P4) */
#pragma omp parallel num_threads(s->nthreads) if (s->nthreads > 1)
        {
            orc_counters lc; orc_work lw; orc_follow_stats lf;
            memset(&lc, 0, sizeof lc); memset(&lw, 0, sizeof lw); memset(&lf, 0, sizeof lf);
            lf.first_bad_slot = -1;
#pragma omp for schedule(static)
            for (int64_t cq = 0; cq < s->C; ++cq) {
                const int64_t cell = reverse_cells ? (s->C - 1 - cq) : cq;
                int32_t cc[3];
                cc[0] = (int32_t)(cell % s->n[0]);
                cc[1] = (int32_t)((cell / s->n[0]) % s->n[1]);
                cc[2] = (int32_t)(cell / ((int64_t)s->n[0] * s->n[1]));
                int colour = (cc[0] & 1) | ((cc[1] & 1) << 1) | ((cc[2] & 1) << 2);
                if (colour != x.gamma) continue;
                if (s->inactive && s->inactive[cc[s->dim - 1]]) continue;   /* inactive region: no trials, particles stay */
                sweep_cell(s, &x, cell, cc, &lc, &lw, &lf);
            }
#pragma omp critical
            add_tallies(s, fs, &lc, &lw, &lf);
        }
    }
    s->t = t + 1;
    s->cnt.sweeps++;
    return 0;
}

int orc_sweeps(orc_sys* s, int64_t n)
{
    for (int64_t q = 0; q < n; ++q) {
        int rc = orc_sweep(s, 0, 0, NULL, 0.0, NULL, NULL, NULL);
        if (rc) return rc;
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* O11: textbook Metropolis, P:38-45 -- no cells, no checkerboard, no       */
/* leave-cell rule; particle uniform over all N; neighbour search = all N-1 */
/* ------------------------------------------------------------------------ */
int orc_textbook_trials(orc_sys* s, int64_t n_trials)
{
    const uint32_t key[2] = {(uint32_t)s->seed, (uint32_t)(s->seed >> 32)};
    const int32_t cc[3] = {0, 0, 0};
    for (int64_t q = 0; q < n_trials; ++q) {
        uint64_t id = s->tb_count++;
        uint32_t ctr[4] = {(uint32_t)id, (uint32_t)(id >> 32), 0u, (TAG_TEXTBOOK << 24)};
        uint32_t b0[4], b1[4];
        orc_philox4x32_10(ctr, key, b0);
        ctr[2] = 1u;
        orc_philox4x32_10(ctr, key, b1);
        int64_t i = (int64_t)(((uint64_t)b0[0] * (uint64_t)s->N) >> 32); /* 1. select a particle at random */
        int rotate = (s->shape->kind != ORC_KIND_DISK) && (b0[1] >> 31);
        float xt[3], qt[4];
        s->cnt.trials++;
        if (!rotate) {                                                  /* 2. small random trial move     */
            uint32_t u[3] = {b0[2], b0[3], b1[0]};
            gen_translate(s, &s->pos[4 * i], u, xt);
            memcpy(qt, &s->quat[4 * i], sizeof qt);
        } else {
            memcpy(xt, &s->pos[4 * i], sizeof xt);
            gen_rotate(s, &s->quat[4 * i], b0[2], b0[3], b1[0], qt);
        }
        double m_min = scan_candidates(s, &s->work, NULL, 1, i, xt, qt, cc);            /* 3. check all other particles   */
        if (m_min < s->eps_g) {                                         /* 4. reject on overlap           */
            if (rotate) s->cnt.rot_rej_overlap++; else s->cnt.trans_rej_overlap++;
        } else {
            wrap_store(s, i, xt, qt);
            if (rotate) s->cnt.rot_acc++; else s->cnt.trans_acc++;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* validators                                                               */
/* ------------------------------------------------------------------------ */
int64_t orc_count_overlaps_bruteforce(const orc_sys* s) /* O5 */
{
    int64_t count = 0;
    double dmax2 = s->shape->dmax * s->shape->dmax;
    for (int64_t i = 0; i < s->N; ++i)
        for (int64_t j = i + 1; j < s->N; ++j) {
            double r[3], qa[4], qb[4];
            min_image(s, &s->pos[4 * j], &s->pos[4 * i], r);
            if (dot3(r, r) >= dmax2) continue;
            quat_to_double(&s->quat[4 * i], qa);
            quat_to_double(&s->quat[4 * j], qb);
            if (orc_shape_margin(s->shape, r, qa, qb) < 0.0) ++count; /* strict, no guard (R15) */
        }
    return count;
}

static double cells_pair_scan(const orc_sys* s, int64_t* count_out)
{
    float shift[3] = {0.0f, 0.0f, 0.0f};
    int32_t* cid = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->N > 0 ? s->N : 1));
    int32_t* mem = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->N > 0 ? s->N : 1));
    int32_t* cst = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->C + 1));
    orc_cell_list(s, shift, cid, cst, mem);
    int64_t count = 0;
    double mmin = INFINITY, dmax2 = s->shape->dmax * s->shape->dmax;
    int zlo = (s->dim == 3) ? -1 : 0, zhi = (s->dim == 3) ? 1 : 0;
    for (int64_t i = 0; i < s->N; ++i) {
        int64_t cell = cid[i];
        int32_t cx = (int32_t)(cell % s->n[0]), cy = (int32_t)((cell / s->n[0]) % s->n[1]);
        int32_t cz = (int32_t)(cell / ((int64_t)s->n[0] * s->n[1]));
        double qa[4];
        quat_to_double(&s->quat[4 * i], qa);
        for (int dz = zlo; dz <= zhi; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int32_t nx = (cx + dx + s->n[0]) % s->n[0], ny = (cy + dy + s->n[1]) % s->n[1];
                    int32_t nz = (cz + dz + s->n[2]) % s->n[2];
                    int32_t nc = nx + s->n[0] * (ny + s->n[1] * nz);
                    for (int32_t p = cst[nc]; p < cst[nc + 1]; ++p) {
                        int64_t j = mem[p];
                        if (j <= i) continue;
                        double r[3], qb[4];
                        min_image(s, &s->pos[4 * j], &s->pos[4 * i], r);
                        if (dot3(r, r) >= dmax2) continue;
                        quat_to_double(&s->quat[4 * j], qb);
                        double m = orc_shape_margin(s->shape, r, qa, qb);
                        if (m < 0.0) ++count;
                        if (m < mmin) mmin = m;
                    }
                }
    }
    free(cid); free(mem); free(cst);
    if (count_out) *count_out = count;
    return mmin;
}

int64_t orc_count_overlaps_cells(const orc_sys* s)
{
    int64_t c = 0;
    cells_pair_scan(s, &c);
    return c;
}
double orc_min_margin_cells(const orc_sys* s) { return cells_pair_scan(s, NULL); }

/* O9: histogram of s = 1 - lambda* over all pairs i<j of the current state with 0 <= s < s_max, nbins equal
 * bins.  Pairs are found in the 5^d cells around each particle (|r| < d_max / (1 - s_max) can reach two cells
 * away), which needs >= 5 cells per side; returns -1 otherwise, else the number of pairs binned. */
int64_t orc_scale_histogram(const orc_sys* s, double s_max, int nbins, uint64_t* hist)
{
    for (int k = 0; k < s->dim; ++k)
        if (s->n[k] < 5) return -1;
    if (!(s_max > 0.0 && s_max < 0.1) || nbins < 1) return -1;
    float shift[3] = {0.0f, 0.0f, 0.0f};
    int32_t* cid = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->N > 0 ? s->N : 1));
    int32_t* mem = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->N > 0 ? s->N : 1));
    int32_t* cst = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->C + 1));
    orc_cell_list(s, shift, cid, cst, mem);
    for (int b = 0; b < nbins; ++b) hist[b] = 0;
    int64_t binned = 0;
    double range = s->shape->dmax / (1.0 - s_max), range2 = range * range;
    int zr = (s->dim == 3) ? 2 : 0;
    for (int64_t i = 0; i < s->N; ++i) {
        int64_t cell = cid[i];
        int32_t cx = (int32_t)(cell % s->n[0]), cy = (int32_t)((cell / s->n[0]) % s->n[1]);
        int32_t cz = (int32_t)(cell / ((int64_t)s->n[0] * s->n[1]));
        double qa[4];
        quat_to_double(&s->quat[4 * i], qa);
        for (int dz = -zr; dz <= zr; ++dz)
            for (int dy = -2; dy <= 2; ++dy)
                for (int dx = -2; dx <= 2; ++dx) {
                    int32_t nx = ((cx + dx) % s->n[0] + s->n[0]) % s->n[0];
                    int32_t ny = ((cy + dy) % s->n[1] + s->n[1]) % s->n[1];
                    int32_t nz = ((cz + dz) % s->n[2] + s->n[2]) % s->n[2];
                    int32_t nc = nx + s->n[0] * (ny + s->n[1] * nz);
                    for (int32_t p = cst[nc]; p < cst[nc + 1]; ++p) {
                        int64_t j = mem[p];
                        if (j <= i) continue;
                        double r[3], qb[4];
                        min_image(s, &s->pos[4 * j], &s->pos[4 * i], r);
                        if (dot3(r, r) >= range2) continue;
                        quat_to_double(&s->quat[4 * j], qb);
                        double sc = 1.0 - orc_shape_touch_scale(s->shape, r, qa, qb);
                        if (sc < 0.0 || sc >= s_max) continue;
                        int b = (int)(sc / s_max * nbins);
                        if (b >= nbins) b = nbins - 1;
                        hist[b]++;
                        ++binned;
                    }
                }
    }
    free(cid); free(mem); free(cst);
    return binned;
}

/* P4: smallest centre distance between particles that sit in DIFFERENT cells of the SAME colour */
double orc_min_same_colour_distance(const orc_sys* s, const float shift[3])
{
    int32_t* cid = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->N > 0 ? s->N : 1));
    int32_t* mem = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->N > 0 ? s->N : 1));
    int32_t* cst = (int32_t*)malloc(sizeof(int32_t) * (size_t)(s->C + 1));
    orc_cell_list(s, shift, cid, cst, mem);
    double best = INFINITY;
    int zr = (s->dim == 3) ? 2 : 0;
    for (int64_t i = 0; i < s->N; ++i) {
        int64_t cell = cid[i];
        int32_t cx = (int32_t)(cell % s->n[0]), cy = (int32_t)((cell / s->n[0]) % s->n[1]);
        int32_t cz = (int32_t)(cell / ((int64_t)s->n[0] * s->n[1]));
        for (int dz = -zr; dz <= zr; dz += 2)
            for (int dy = -2; dy <= 2; dy += 2)
                for (int dx = -2; dx <= 2; dx += 2) {
                    int32_t nx = ((cx + dx) % s->n[0] + s->n[0]) % s->n[0];
                    int32_t ny = ((cy + dy) % s->n[1] + s->n[1]) % s->n[1];
                    int32_t nz = ((cz + dz) % s->n[2] + s->n[2]) % s->n[2];
                    int32_t nc = nx + s->n[0] * (ny + s->n[1] * nz);
                    if (nc == cell) continue;
                    for (int32_t p = cst[nc]; p < cst[nc + 1]; ++p) {
                        double r[3];
                        min_image(s, &s->pos[4 * mem[p]], &s->pos[4 * i], r);
                        double dd = norm3(r);
                        if (dd < best) best = dd;
                    }
                }
    }
    free(cid); free(mem); free(cst);
    return best;
}
