// Narrow-phase overlap tests of the CUDA path (S:8(a) row a9), templated on the scalar type:
// float in the sweep kernels, double in the overlap-count validator.
//   disk / sphere      : centre distance vs diameter, "trivial"
//   convex polygon     : separating axes over the edge normals of both, in A's frame
//   convex polyhedron  : GJK separating-axis search on the Minkowski difference B (-) A with the support
//                        function of Eq. (2): S(n) = R S_B(R^-1 n) + r_AB - S_A(-n), in A's frame.
//   rounded shapes     : spheropolygons / convex spheropolyhedra, the polygon / polyhedron ("core") swept by a disk /
//                        sphere of radius rho: two of them overlap iff their cores are closer than 2 rho = S.sweep.  Runtime
//                        vertex count only (NV == 0 instantiations), so the unrolled pentagon / cube paths do not carry it.
// Every test answers "is the pair separated by at least eps?"; "no" means overlap (R15, R-poly).
#pragma once
#include "common.cuh"

namespace hpmc {

template <typename T>
struct ShapeT {
    int kind, nverts;
    T diameter;
    T dmax2;              // d_max^2, broad phase R16
    T din2;               // (2 r_in - 1e-5)^2: centres closer than this certainly overlap (r_in = inscribed radius about
                          // the body origin); 0 for disks (the broad phase is the whole test)
    T rin;                // inscribed radius about the body origin (polygons: min_k fc[k]); every support height h(u) >= rin
    T sweep;              // rounded shapes: 2 x sweep radius, the distance below which two cores mean overlap; 0 = sharp
    int regular;          // polygon: regular n-gon centred on the body origin (all |v| equal, equal angles): see polygon_separated
    T vx[kMaxVerts], vy[kMaxVerts], vz[kMaxVerts];
    T nx[kMaxVerts], ny[kMaxVerts], fc[kMaxVerts];  // polygon: outward unit edge normals and offsets n.v
};
using ShapeF = ShapeT<float>;
using ShapeD = ShapeT<double>;

template <typename T>
struct V3 {
    T x, y, z;
};
template <typename T>
__device__ __forceinline__ T dot(const V3<T>& a, const V3<T>& b)
{
    return a.x * b.x + a.y * b.y + a.z * b.z;
}
template <typename T>
__device__ __forceinline__ V3<T> cross(const V3<T>& a, const V3<T>& b)
{
    return V3<T>{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
template <typename T>
__device__ __forceinline__ V3<T> operator-(const V3<T>& a, const V3<T>& b)
{
    return V3<T>{a.x - b.x, a.y - b.y, a.z - b.z};
}
template <typename T>
__device__ __forceinline__ V3<T> operator+(const V3<T>& a, const V3<T>& b)
{
    return V3<T>{a.x + b.x, a.y + b.y, a.z + b.z};
}
template <typename T>
__device__ __forceinline__ V3<T> operator*(T s, const V3<T>& a)
{
    return V3<T>{s * a.x, s * a.y, s * a.z};
}

// ---------------------------------------------------------------------------------------------
// spheropolygons: is the distance between the two core polygons at least S.sweep + eps?  In A's body frame.
//   1. the largest separation of the cores over the edge normals of both (the separating-axis margin, a lower bound of the
//      distance): at least S.sweep + eps -> separated; negative -> the cores themselves intersect -> overlap;
//   2. otherwise the cores are disjoint and closer than their axis separation can tell (vertex against vertex): the
//      distance of two disjoint convex polygons is attained between a vertex of one and an edge of the other, so take the
//      minimum point-segment distance over all such pairs.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T point_segment_dist2(T px, T py, T ax, T ay, T bx, T by)
{
    const T ex = bx - ax, ey = by - ay, wx = px - ax, wy = py - ay;
    T t = (wx * ex + wy * ey) / (ex * ex + ey * ey);
    t = min(max(t, (T)0), (T)1);
    const T dx = wx - t * ex, dy = wy - t * ey;
    return dx * dx + dy * dy;
}

template <typename T>
__device__ __noinline__ bool spheropolygon_separated(const ShapeT<T>& S, T rx, T ry, T cA, T sA, T cB, T sB, T eps)
{
    const int nv = S.nverts;
    const T need = S.sweep + eps;
    const T lx = cA * rx + sA * ry, ly = -sA * rx + cA * ry;   // R_A^T r_AB
    const T c = cA * cB + sA * sB, s = cA * sB - sA * cB;      // R = R_A^T R_B
    T px[kMaxVerts], py[kMaxVerts];                            // B's vertices in A's frame
    for (int j = 0; j < nv; ++j) {
        px[j] = c * S.vx[j] - s * S.vy[j] + lx;
        py[j] = s * S.vx[j] + c * S.vy[j] + ly;
    }
    T msat = -(T)3.0e38;
    for (int k = 0; k < nv; ++k) {
        // A's edge normal k against B's vertices; B's edge normal k (rotated into A's frame) against A's vertices
        const T nxk = c * S.nx[k] - s * S.ny[k], nyk = s * S.nx[k] + c * S.ny[k];
        T ma = S.nx[k] * px[0] + S.ny[k] * py[0];
        T mb = nxk * (S.vx[0] - lx) + nyk * (S.vy[0] - ly);
        for (int j = 1; j < nv; ++j) {
            ma = min(ma, S.nx[k] * px[j] + S.ny[k] * py[j]);
            mb = min(mb, nxk * (S.vx[j] - lx) + nyk * (S.vy[j] - ly));
        }
        msat = max(msat, max(ma, mb) - S.fc[k]);
    }
    if (msat >= need) return true;
    if (msat < (T)0) return false;
    T d2 = (T)3.0e38;
    for (int i = 0; i < nv; ++i)
        for (int k = 0; k < nv; ++k) {
            const int k1 = (k + 1 == nv) ? 0 : k + 1;
            d2 = min(d2, point_segment_dist2(px[i], py[i], S.vx[k], S.vy[k], S.vx[k1], S.vy[k1]));
            d2 = min(d2, point_segment_dist2(S.vx[i], S.vy[i], px[k], py[k], px[k1], py[k1]));
        }
    return d2 >= need * need;
}

// ---------------------------------------------------------------------------------------------
// convex polygons: in A's body frame A's vertices/normals are the stored constants, so only B has to
// be rotated ("a local coordinate system centered on particle A").
// (rx, ry) = r_AB in the world frame; (cA,sA), (cB,sB) = cos/sin of the orientation angles.
// NV > 0: compile-time vertex count (fully unrolled, registers); NV == 0: runtime count.
// Returns true iff NO axis separates the pair by at least eps.  Used by the fp64 validator (a12) with eps = 0; the
// sweep kernels use polygon_separated below.
// ---------------------------------------------------------------------------------------------
template <typename T, int NV>
__device__ __forceinline__ bool polygon_overlap(const ShapeT<T>& S, T rx, T ry, T cA, T sA, T cB, T sB, T eps)
{
    if (NV == 0 && S.sweep > (T)0) return !spheropolygon_separated<T>(S, rx, ry, cA, sA, cB, sB, eps);
    const int nv = (NV > 0) ? NV : S.nverts;
    const T lx = cA * rx + sA * ry;    // R_A^T r_AB
    const T ly = -sA * rx + cA * ry;
    const T c = cA * cB + sA * sB;     // R = R_A^T R_B
    const T s = cA * sB - sA * cB;
    // axes of A: separation_k = min_j n_k . p_j - c_k with p_j = B's vertices in A's frame
    {
        T px[(NV > 0) ? NV : kMaxVerts], py[(NV > 0) ? NV : kMaxVerts];
#pragma unroll
        for (int j = 0; j < nv; ++j) {
            px[j] = c * S.vx[j] - s * S.vy[j] + lx;
            py[j] = s * S.vx[j] + c * S.vy[j] + ly;
        }
#pragma unroll
        for (int k = 0; k < nv; ++k) {
            T m = S.nx[k] * px[0] + S.ny[k] * py[0];
#pragma unroll
            for (int j = 1; j < nv; ++j) m = min(m, S.nx[k] * px[j] + S.ny[k] * py[j]);
            if (m - S.fc[k] >= eps) return false;
        }
    }
    // axes of B: n'_k = R n_k; separation_k = min_j n'_k . (v_j - r_loc) - c_k  (A's vertices seen from B)
    {
        T qx[(NV > 0) ? NV : kMaxVerts], qy[(NV > 0) ? NV : kMaxVerts];
#pragma unroll
        for (int j = 0; j < nv; ++j) {
            qx[j] = S.vx[j] - lx;
            qy[j] = S.vy[j] - ly;
        }
#pragma unroll
        for (int k = 0; k < nv; ++k) {
            const T nxk = c * S.nx[k] - s * S.ny[k];
            const T nyk = s * S.nx[k] + c * S.ny[k];
            T m = nxk * qx[0] + nyk * qy[0];
#pragma unroll
            for (int j = 1; j < nv; ++j) m = min(m, nxk * qx[j] + nyk * qy[j]);
            if (m - S.fc[k] >= eps) return false;
        }
    }
    return true;
}

// The sweep's polygon test (fp32): is the pair separated by at least eps along one of the 2 nv edge normals?  Same axis set
// and the same definition of the separation as polygon_overlap, organised by support functions so that only axes that CAN
// separate are evaluated:
//
//   axis k of A (unit normal n_k, offset c_k, A's frame):  sep_k = n_k . l_A - c_k - h_B(-R^T n_k)
//   axis k of B (as a direction from A toward B: -n_k):    sep_k = -n_k . l_B - c_k - h_A(-R n_k)
//
// with l_A = R_A^T r, l_B = R_B^T r (r = r_AB, world), R = R_A^T R_B and h_X(u) = max_j u . v_j over the BODY-frame
// vertices -- the axis is rotated into the other particle's frame instead of rotating that particle's vertices.
// Every support height is >= r_in, so axis k can only separate if g_k = n_k . l - c_k >= r_in + eps: a cheap test (one dot
// product with constants) that rules out most axes before their nv-vertex support maximum is taken.
//
// Regular n-gon (S.regular; NV > 0 = compile-time n, unrolled): all c_k = r_in and the normals are 2 pi / n apart, so for
// |r| < d_max + eps_g (the broad phase, R16') only the normal closest to l can pass the test -- the next one has
// n . l <= |l| cos(pi/n) < 2 r_in + eps.  One support maximum per side instead of n: 2 x (n dots + select + n dots).
// Branch-free, no early exit (dense narrow phase: a warp finishes with its slowest lane anyway).
// General convex polygon: every axis that passes the test is evaluated (data-dependent loop).
// All fp32 colour-pass variants call this one function, so their decisions agree bit for bit.
template <int NV>
__device__ __forceinline__ bool polygon_separated(const ShapeT<float>& S, float rx, float ry, float cA, float sA, float cB, float sB, float eps)
{
    if (NV == 0 && S.sweep > 0.0f) return spheropolygon_separated<float>(S, rx, ry, cA, sA, cB, sB, eps);
    const int nv = (NV > 0) ? NV : S.nverts;
    const float lAx = cA * rx + sA * ry, lAy = cA * ry - sA * rx;      // R_A^T r
    const float lBx = cB * rx + sB * ry, lBy = cB * ry - sB * rx;      // R_B^T r
    const float c = cA * cB + sA * sB, s = cA * sB - sA * cB;          // R = R_A^T R_B: (x, y) -> (c x - s y, s x + c y)
    if (NV > 0 || S.regular) {
        // the normal of A closest to l_A and the normal of B closest to -l_B (the first of equal maxima)
        float gA = -3.0e38f, nAx = 0.f, nAy = 0.f, gB = -3.0e38f, nBx = 0.f, nBy = 0.f;
        if constexpr (NV > 0) {
            // compile-time count: the maxima with max instructions, then the normals by equality from the last to the first --
            // 14 operations of the half-rate alu pipe per side instead of a compare and three selects per normal (20)
            float a[NV], b[NV];
#pragma unroll
            for (int k = 0; k < NV; ++k) {
                a[k] = fmaf(S.nx[k], lAx, fmaf(S.ny[k], lAy, -S.fc[k]));
                b[k] = -fmaf(S.nx[k], lBx, fmaf(S.ny[k], lBy, S.fc[k]));
                gA = fmaxf(gA, a[k]);
                gB = fmaxf(gB, b[k]);
            }
            nAx = nBx = S.nx[NV - 1];
            nAy = nBy = S.ny[NV - 1];
#pragma unroll
            for (int k = NV - 2; k >= 0; --k) {
                const bool pa = a[k] == gA, pb = b[k] == gB;
                nAx = pa ? S.nx[k] : nAx; nAy = pa ? S.ny[k] : nAy;
                nBx = pb ? S.nx[k] : nBx; nBy = pb ? S.ny[k] : nBy;
            }
        } else {
#pragma unroll
            for (int k = 0; k < nv; ++k) {
                const float a = fmaf(S.nx[k], lAx, fmaf(S.ny[k], lAy, -S.fc[k]));
                const float b = -fmaf(S.nx[k], lBx, fmaf(S.ny[k], lBy, S.fc[k]));
                const bool pa = a > gA, pb = b > gB;
                gA = pa ? a : gA; nAx = pa ? S.nx[k] : nAx; nAy = pa ? S.ny[k] : nAy;
                gB = pb ? b : gB; nBx = pb ? S.nx[k] : nBx; nBy = pb ? S.ny[k] : nBy;
            }
        }
        const float uAx = -(c * nAx + s * nAy), uAy = s * nAx - c * nAy;     // -R^T n_A, in B's frame
        const float uBx = s * nBy - c * nBx, uBy = -(s * nBx + c * nBy);     // -R n_B, in A's frame
        float hB = uAx * S.vx[0] + uAy * S.vy[0], hA = uBx * S.vx[0] + uBy * S.vy[0];
#pragma unroll
        for (int j = 1; j < nv; ++j) {
            hB = fmaxf(hB, uAx * S.vx[j] + uAy * S.vy[j]);
            hA = fmaxf(hA, uBx * S.vx[j] + uBy * S.vy[j]);
        }
        return fmaxf(gA - hB, gB - hA) >= eps;
    }
    const float need = S.rin + eps;
    for (int k = 0; k < nv; ++k) {
        const float a = fmaf(S.nx[k], lAx, fmaf(S.ny[k], lAy, -S.fc[k]));
        if (a >= need) {
            const float ux = -(c * S.nx[k] + s * S.ny[k]), uy = s * S.nx[k] - c * S.ny[k];
            float h = ux * S.vx[0] + uy * S.vy[0];
            for (int j = 1; j < nv; ++j) h = fmaxf(h, ux * S.vx[j] + uy * S.vy[j]);
            if (a - h >= eps) return true;
        }
        const float b = -fmaf(S.nx[k], lBx, fmaf(S.ny[k], lBy, S.fc[k]));
        if (b >= need) {
            const float ux = s * S.ny[k] - c * S.nx[k], uy = -(s * S.nx[k] + c * S.ny[k]);
            float h = ux * S.vx[0] + uy * S.vy[0];
            for (int j = 1; j < nv; ++j) h = fmaxf(h, ux * S.vx[j] + uy * S.vy[j]);
            if (b - h >= eps) return true;
        }
    }
    return false;
}

// ---------------------------------------------------------------------------------------------
// convex polyhedra: GJK.  Rm = rotation taking B's body frame into A's body frame (row major),
// r = r_AB expressed in A's frame.
// ---------------------------------------------------------------------------------------------
// NVP > 0: compile-time vertex count (the loop unrolls and the vertices become constant-bank operands); 0: runtime count.
template <typename T, int NVP = 0>
__device__ __forceinline__ V3<T> support_minkowski(const ShapeT<T>& S, const T* Rm, const V3<T>& r, const V3<T>& dir, int& pair)
{
    // R^-1 dir = R^T dir
    const V3<T> db{Rm[0] * dir.x + Rm[3] * dir.y + Rm[6] * dir.z, Rm[1] * dir.x + Rm[4] * dir.y + Rm[7] * dir.z,
                   Rm[2] * dir.x + Rm[5] * dir.y + Rm[8] * dir.z};
    T bestA = -(T)3.0e38, bestB = -(T)3.0e38;
    int ia = 0, ib = 0;
    const int nv = (NVP > 0) ? NVP : S.nverts;
#pragma unroll
    for (int i = 0; i < nv; ++i) {
        const T da = -(dir.x * S.vx[i] + dir.y * S.vy[i] + dir.z * S.vz[i]);   // S_A(-dir)
        const T dbv = db.x * S.vx[i] + db.y * S.vy[i] + db.z * S.vz[i];        // S_B(R^-1 dir)
        if (da > bestA) { bestA = da; ia = i; }
        if (dbv > bestB) { bestB = dbv; ib = i; }
    }
    pair = ia | (ib << 8);   // the vertices of A and of B behind this point of B (-) A
    const T bx = S.vx[ib], by = S.vy[ib], bz = S.vz[ib];
    return V3<T>{Rm[0] * bx + Rm[1] * by + Rm[2] * bz + r.x - S.vx[ia], Rm[3] * bx + Rm[4] * by + Rm[5] * bz + r.y - S.vy[ia],
                 Rm[6] * bx + Rm[7] * by + Rm[8] * bz + r.z - S.vz[ia]};
}

// closest point to the origin on triangle (a,b,c); mask bit0/1/2 = a/b/c supports the result
template <typename T>
__device__ __forceinline__ V3<T> closest_on_triangle(const V3<T>& a, const V3<T>& b, const V3<T>& c, int& mask)
{
    const V3<T> ab = b - a, ac = c - a;
    const T d1 = -dot(ab, a), d2 = -dot(ac, a);
    if (d1 <= 0 && d2 <= 0) { mask = 1; return a; }
    const T d3 = -dot(ab, b), d4 = -dot(ac, b);
    if (d3 >= 0 && d4 <= d3) { mask = 2; return b; }
    const T vc = d1 * d4 - d3 * d2;
    if (vc <= 0 && d1 >= 0 && d3 <= 0) { mask = 3; return a + (d1 / (d1 - d3)) * ab; }
    const T d5 = -dot(ab, c), d6 = -dot(ac, c);
    if (d6 >= 0 && d5 <= d6) { mask = 4; return c; }
    const T vb = d5 * d2 - d1 * d6;
    if (vb <= 0 && d2 >= 0 && d6 <= 0) { mask = 5; return a + (d2 / (d2 - d6)) * ac; }
    const T va = d3 * d6 - d5 * d4;
    if (va <= 0 && (d4 - d3) >= 0 && (d5 - d6) >= 0) { mask = 6; return b + ((d4 - d3) / ((d4 - d3) + (d5 - d6))) * (c - b); }
    const T denom = (T)1 / (va + vb + vc);
    mask = 7;
    return a + (vb * denom) * ab + (vc * denom) * ac;
}

// GJK verdicts.  kGjkSeparated: a direction was found along which the support functions separate the pair by
// >= eps (a certificate evaluated directly from the support points).  kGjkOverlap: the origin lies inside a
// tetrahedron of Minkowski-difference points, farther than `deep` from each of its faces, so the interiors
// intersect by at least `deep`.  kGjkUnsure: everything else (origin enclosed but close to a face, converged with
// distance < eps, no numerical progress, repeated support point, iteration cap).  Near contact the GJK direction
// v is the small difference of O(1) vectors, so in fp32 its relative error ~1e-7/|v| makes the certificate
// unreliable for gaps below ~1e-3: the fp32 caller re-runs kGjkUnsure pairs in fp64 (mixed precision);
// the fp64 caller treats kGjkUnsure as overlap (conservative, R-poly).
constexpr int kGjkSeparated = 1, kGjkOverlap = 0, kGjkUnsure = -1;
template <typename T, int NVP = 0>
__device__ int gjk_classify(const ShapeT<T>& S, const T* Rm, const V3<T>& r, T eps, T deep)
{
    const T tiny = (sizeof(T) == 4) ? (T)1e-14 : (T)1e-28;
    const T reltol = (sizeof(T) == 4) ? (T)1e-6 : (T)1e-13;
    V3<T> v = r;  // a point of B (-) A (both body origins are interior points)
    T vv = dot(v, v);
    if (vv < tiny) return kGjkUnsure;
    V3<T> W[4];
    int nW = 0;
    for (int iter = 0; iter < 40; ++iter) {
        int wpair;
        const V3<T> w = support_minkowski<T, NVP>(S, Rm, r, V3<T>{-v.x, -v.y, -v.z}, wpair);
        const T vw = dot(v, w);
        if (vw >= 0 && vw * vw >= eps * eps * vv) return kGjkSeparated;   // certificate: v^.w >= eps
        if (iter > 0 && vv - vw <= reltol * vv) return kGjkUnsure;           // converged: distance |v| < eps
        for (int i = 0; i < nW; ++i)
            if (W[i].x == w.x && W[i].y == w.y && W[i].z == w.z) return kGjkUnsure;  // same support point again
        W[nW++] = w;
        V3<T> vn;
        if (nW == 1) {
            vn = w;
        } else if (nW == 2) {
            const V3<T> a = W[1], b = W[0], ab = b - a;
            const T t = -dot(a, ab);
            if (t <= 0) { vn = a; W[0] = a; nW = 1; }
            else {
                const T den = dot(ab, ab);
                if (t >= den) { vn = b; nW = 1; }
                else vn = a + (t / den) * ab;
            }
        } else if (nW == 3) {
            int mask;
            const V3<T> a = W[2], b = W[1], c = W[0];
            vn = closest_on_triangle(a, b, c, mask);
            int k = 0;
            if (mask & 4) W[k++] = c;
            if (mask & 2) W[k++] = b;
            if (mask & 1) W[k++] = a;
            nW = k;
        } else {
            const V3<T> a = W[3], b = W[2], c = W[1], d = W[0];
            // faces (a,b,c | d), (a,c,d | b), (a,d,b | c), (b,d,c | a): origin outside iff on the other side than the 4th vertex
            T best = (T)3.0e38;
            int bestFace = -1, bestMask = 0;
            V3<T> bestV{0, 0, 0};
            T minIn = (T)3.0e38;   // min distance from the origin to the faces (when enclosed)
            bool fat = true;       // every face has a solid area and the opposite vertex stands well clear of it
            const T area_min2 = (T)1e-3 * S.dmax2 * S.dmax2, height_min = (T)10 * deep;
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                const V3<T> p = (f == 3) ? b : a;
                const V3<T> q = (f == 0) ? b : (f == 1) ? c : d;
                const V3<T> s3 = (f == 0) ? c : (f == 1) ? d : (f == 2) ? b : c;
                const V3<T> o = (f == 0) ? d : (f == 1) ? b : (f == 2) ? c : a;
                const V3<T> nn = cross(q - p, s3 - p);
                const T sp = -dot(nn, p);          // origin side
                const T sd = dot(nn, o - p);       // opposite-vertex side
                const T nn2 = dot(nn, nn);
                const T inv = rsqrt(nn2);
                if (sp * sd > 0) minIn = min(minIn, fabs(sp) * inv);
                fat = fat && nn2 >= area_min2 && fabs(sd) * inv >= height_min;
                if (sp * sd <= 0) {                // outside this face (or degenerate): closest point on it
                    int m;
                    const V3<T> cand = closest_on_triangle(p, q, s3, m);
                    const T cc = dot(cand, cand);
                    if (cc < best) { best = cc; bestFace = f; bestMask = m; bestV = cand; }
                }
            }
            // origin inside the tetrahedron.  "Overlap" needs a margin the arithmetic can vouch for: in a sliver (a face of
            // tiny area, or a vertex almost in the plane of the opposite face -- two cubes with nearly parallel faces) the
            // face normals are differences of nearly equal products and the sign of `sp * sd` is rounding noise, so such a
            // tetrahedron only ever yields "unsure" (fp32: re-run in fp64; fp64 with deep = 0: fat is always true).
            if (bestFace < 0) return (minIn > deep && fat) ? kGjkOverlap : kGjkUnsure;
            const V3<T> p = (bestFace == 3) ? b : a;
            const V3<T> q = (bestFace == 0) ? b : (bestFace == 1) ? c : d;
            const V3<T> s3 = (bestFace == 0) ? c : (bestFace == 1) ? d : (bestFace == 2) ? b : c;
            int k = 0;
            if (bestMask & 4) W[k++] = s3;
            if (bestMask & 2) W[k++] = q;
            if (bestMask & 1) W[k++] = p;
            nW = k;
            vn = bestV;
        }
        const T vvn = dot(vn, vn);
        if (vvn < tiny) return kGjkUnsure;              // origin on the simplex: touching or inside
        if (iter > 0 && vvn >= vv) return kGjkUnsure;   // no numerical progress
        v = vn;
        vv = vvn;
    }
    return kGjkUnsure;
}

// Is the origin inside the tetrahedron (a, b, c, d), farther than `deep` from each of its faces, and is the tetrahedron
// solid enough for fp32 to vouch for that (every face has a real area and the opposite vertex stands well clear of it)?
template <typename T>
__device__ __forceinline__ bool origin_deep_inside(const V3<T>& a, const V3<T>& b, const V3<T>& c, const V3<T>& d, T dmax2, T deep)
{
    const T area_min2 = (T)1e-3 * dmax2 * dmax2, height_min = (T)10 * deep;
    bool ok = true;
#pragma unroll
    for (int f = 0; f < 4; ++f) {
        const V3<T> p = (f == 3) ? b : a;
        const V3<T> q = (f == 0) ? b : (f == 1) ? c : d;
        const V3<T> s3 = (f == 0) ? c : (f == 1) ? d : (f == 2) ? b : c;
        const V3<T> o = (f == 0) ? d : (f == 1) ? b : (f == 2) ? c : a;
        const V3<T> nn = cross(q - p, s3 - p);
        const T sp = -dot(nn, p);          // origin side
        const T sd = dot(nn, o - p);       // opposite-vertex side
        const T nn2 = dot(nn, nn);
        const T inv = rsqrt(nn2);
        ok = ok && sp * sd > 0 && fabs(sp) * inv > deep && nn2 >= area_min2 && fabs(sd) * inv >= height_min;
    }
    return ok;
}

// Minkowski portal refinement -- XenoCollide, the paper's GPU overlap check for convex polyhedra ("XenoCollide [32] is faster
// on the GPU"; "implemented as a single loop") -- on the Minkowski difference B (-) A with the support function
// of Eq. (2), same verdicts as gjk_classify:
//   kGjkSeparated  some direction n was found with max_{x in B(-)A} n^ . x <= -eps: a separating plane, evaluated directly
//                  from a support point (the same kind of certificate as in gjk_classify);
//   kGjkOverlap    the origin lies inside a tetrahedron (v0, v1, v2, v3) of points of B (-) A -- v0 = r, the difference of
//                  the two body origins, an interior point -- deeper than `deep` and the tetrahedron is solid
//                  (origin_deep_inside): the interiors intersect by more than `deep` >> eps;
//   kGjkUnsure     everything else (the origin within `deep` of the boundary, a separating direction with less than eps of
//                  clearance, degenerate portals, iteration cap): the fp32 caller decides such a pair in fp64.
// Why not GJK in fp32: the loop body is the same for every lane whatever the state of its simplex (one support call, a few
// cross products and selects), where GJK's case analysis (line / triangle / four faces of a tetrahedron, each with a
// closest-point-on-triangle) makes the lanes of a warp -- one pair each -- execute the union of all cases; and the
// tetrahedron that certifies an overlap has the deep interior point v0 as a vertex, so it is rarely a sliver (GJK's simplex
// of nearby support points often is, which sent those pairs to fp64).
// G = lanes per pair.  G = 1: the lane evaluates both support maxima.  G = 2 (the warp-per-cell pass): the two lanes of an
// aligned pair hold the SAME pair of particles and run the same instructions; in the support call lane `sub` = 0 scans the
// vertices for S_A(-n), lane 1 for S_B(R^-1 n), they exchange the two vertex indices with one shuffle each and both form the
// same point of B (-) A.  Same arithmetic per vertex and the same first-maximum rule as G = 1, so the verdicts -- and the
// trajectories of the passes that use one or the other -- are bit-identical.  ~10 pairs pass the broad phase of a trial, so the
// second lane is free, and the vertex scans are most of an iteration (more so with 20 or 24 vertices).
template <typename T, int NVP, int G>
__device__ __forceinline__ V3<T> support_mpr(const ShapeT<T>& S, const T* Rm, const V3<T>& r, const V3<T>& dir, int& pair, int sub, unsigned pair_mask)
{
    if (G == 1) return support_minkowski<T, NVP>(S, Rm, r, dir, pair);
    // R^-1 dir = R^T dir
    const V3<T> db{Rm[0] * dir.x + Rm[3] * dir.y + Rm[6] * dir.z, Rm[1] * dir.x + Rm[4] * dir.y + Rm[7] * dir.z,
                   Rm[2] * dir.x + Rm[5] * dir.y + Rm[8] * dir.z};
    // support_minkowski's two scans are da = -(dir . v) and dbv = db . v; this lane runs one of them.  -(a + b + c) with the
    // contraction fma(z, vz, fma(y, vy, x vx)) equals the same expression of the negated direction bit for bit
    const V3<T> d = sub ? db : V3<T>{-dir.x, -dir.y, -dir.z};
    T best = -(T)3.0e38;
    int ibest = 0;
    const int nv = (NVP > 0) ? NVP : S.nverts;
#pragma unroll
    for (int i = 0; i < nv; ++i) {
        const T t = d.x * S.vx[i] + d.y * S.vy[i] + d.z * S.vz[i];
        if (t > best) { best = t; ibest = i; }
    }
    const int lane0 = (threadIdx.x & 31) & ~1;
    const int ia = __shfl_sync(pair_mask, ibest, lane0), ib = __shfl_sync(pair_mask, ibest, lane0 + 1);
    pair = ia | (ib << 8);
    const T bx = S.vx[ib], by = S.vy[ib], bz = S.vz[ib];
    return V3<T>{Rm[0] * bx + Rm[1] * by + Rm[2] * bz + r.x - S.vx[ia], Rm[3] * bx + Rm[4] * by + Rm[5] * bz + r.y - S.vy[ia],
                 Rm[6] * bx + Rm[7] * by + Rm[8] * bz + r.z - S.vz[ia]};
}

template <typename T, int NVP = 0, int G = 1>
__device__ int mpr_classify(const ShapeT<T>& S, const T* Rm, const V3<T>& r, T eps, T deep, int* portal, int sub = 0, unsigned pair_mask = 0u)
{
    // portal[0..2]: on kGjkUnsure from the refinement stage, the vertex pairs (index in A | index in B << 8) behind the last
    // portal (v1, v2, v3) -- exact data from which the fp64 re-run rebuilds the tetrahedron (r, v1, v2, v3); else portal[0] = -1
    //
    // ONE loop with ONE support call for all stages ("implemented as a single loop"): the lanes of a warp, one pair
    // each, are in different stages -- first point, second point, portal discovery, portal refinement -- and the support
    // function is nine tenths of an iteration; what differs per stage is a few cross products behind it.
    const T tiny = (T)1e-14;
    portal[0] = -1;
    const V3<T> v0 = r;
    const T v00 = dot(v0, v0);
    if (v00 < tiny) return kGjkUnsure;
    V3<T> v1{0, 0, 0}, v2{0, 0, 0}, v3{0, 0, 0};
    int p1 = -1, p2 = -1, p3 = -1;
    V3<T> n{-v0.x, -v0.y, -v0.z};
    int stage = 0;   // 0: v1 along -v0; 1: v2 along v1 x v0; 2: discovery of v3; 3: refinement
    int verdict = kGjkUnsure;
    bool have_portal = false;
    for (int it = 0; it < 40; ++it) {
        const T nn = dot(n, n);
        if (nn < tiny * (stage == 1 ? v00 : (T)1)) break;             // degenerate direction (stage 1: v0, v1, origin on one line)
        const T inv_n = rsqrt(nn);
        // refinement: the origin is behind the portal by more than `deep`: inside the tetrahedron (v0, v1, v2, v3) ?
        if (stage == 3 && dot(n, v1) * inv_n > deep) {
            if (origin_deep_inside(v0, v1, v2, v3, S.dmax2, deep)) verdict = kGjkOverlap;
            break;
        }
        int pw;
        V3<T> w = support_mpr<T, NVP, G>(S, Rm, r, n, pw, sub, pair_mask);
        // rounded shapes: B (-) A is the difference of the cores swept by a ball of radius 2 rho = S.sweep, whose support point
        // along n lies S.sweep further out (every certificate below then speaks about the rounded bodies)
        if (NVP == 0 && S.sweep > (T)0) w = w + (S.sweep * inv_n) * n;
        const T h = dot(w, n);
        if (h <= 0) {   // the whole of B (-) A lies at n^ . x <= h / |n|: a separating plane if that is <= -eps
            if (h * h >= eps * eps * nn) verdict = kGjkSeparated;
            else have_portal = false;   // a weak separating plane: the portal is of no use to the re-run
            break;
        }
        if (stage == 0) {
            v1 = w; p1 = pw;
            n = cross(v1, v0);
            stage = 1;
        } else if (stage == 1) {
            v2 = w; p2 = pw;
            n = cross(v1 - v0, v2 - v0);
            if (dot(n, v0) > 0) {   // the origin on the positive side of (v0, v1, v2)
                const V3<T> t = v1; v1 = v2; v2 = t;
                const int tp = p1; p1 = p2; p2 = tp;
                n = V3<T>{-n.x, -n.y, -n.z};
            }
            stage = 2;
        } else {
            // Discovery (stage 2) and refinement (stage 3) are ONE body, so that lanes in either stage -- from the third
            // iteration on a warp holds both kinds -- run the same instructions: with c4 = w x v0 the signs of
            // d_k = v_k . c4 = det(v_k, w, v0) say which of v1, v2, v3 the new point w replaces in either stage, and the next
            // direction is (a - c) x (b - c) for a stage-dependent choice of (a, b, c): selects, not two divergent branches.
            // refinement only: the portal has reached the surface, the origin is within ~deep of it
            if (stage == 3 && dot(w - v3, n) <= (T)1e-6 * (nn * inv_n)) break;
            const V3<T> c4 = cross(w, v0);
            const T d1 = dot(v1, c4), d2 = dot(v2, c4), d3 = dot(v3, c4);
            // discovery (a triangle (v1, v2, v3) that the ray from v0 through the origin crosses): w replaces v2 if the origin
            // is outside the plane (v0, v1, w), else v1 if outside (v0, w, v2), else it closes the portal as v3.
            // refinement (push the portal outward): w replaces the vertex that keeps the ray inside the new triangle.
            int slot;
            if (stage == 2) slot = (d1 < 0) ? 2 : (d2 > 0) ? 1 : 3;
            else slot = (d1 > 0) ? ((d2 > 0) ? 1 : 3) : ((d3 > 0) ? 2 : 1);
            if (slot == 1) { v1 = w; p1 = pw; }
            if (slot == 2) { v2 = w; p2 = pw; }
            if (slot == 3) { v3 = w; p3 = pw; }
            const bool discovering = stage == 2 && slot != 3;
            if (!discovering) { stage = 3; have_portal = true; }
            const V3<T> a = discovering ? v1 : v2, b = discovering ? v2 : v3, c = discovering ? v0 : v1;
            n = cross(a - c, b - c);
        }
    }
    if (verdict == kGjkUnsure && have_portal) { portal[0] = p1; portal[1] = p2; portal[2] = p3; }
    return verdict;
}

// which fp32 classifier the colour passes use (the fp64 decisions are always GJK): one switch for every variant, so that
// they stay bit-identical to each other
constexpr bool kFp32UseMpr = true;

// rotation matrix (row major) of the unit quaternion (w,x,y,z)
template <typename T>
__device__ __forceinline__ void quat_to_matrix(T w, T x, T y, T z, T* M)
{
    const T xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z, wx = w * x, wy = w * y, wz = w * z;
    M[0] = 1 - 2 * (yy + zz); M[1] = 2 * (xy - wz);     M[2] = 2 * (xz + wy);
    M[3] = 2 * (xy + wz);     M[4] = 1 - 2 * (xx + zz); M[5] = 2 * (yz - wx);
    M[6] = 2 * (xz - wy);     M[7] = 2 * (yz + wx);     M[8] = 1 - 2 * (xx + yy);
}

// polyhedron pair in A's frame: MA, MB = world rotation matrices of A and B, rw = r_AB (world).  GJK verdict.
// G, sub, pair_mask: two lanes per pair in the fp32 XenoCollide run (support_mpr); G = 1 everywhere else.
template <typename T, int NVP = 0, int G = 1>
__device__ __forceinline__ int polyhedron_classify(const ShapeT<T>& S, const T* MA, const T* MB, const V3<T>& rw, T eps, T deep, int* portal,
                                                   int sub = 0, unsigned pair_mask = 0u)
{
    T Rm[9];  // R = MA^T MB takes B's frame into A's frame (q = q_A* q_B)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) Rm[3 * i + j] = MA[i] * MB[j] + MA[3 + i] * MB[3 + j] + MA[6 + i] * MB[6 + j];
    const V3<T> r{MA[0] * rw.x + MA[3] * rw.y + MA[6] * rw.z, MA[1] * rw.x + MA[4] * rw.y + MA[7] * rw.z,
                  MA[2] * rw.x + MA[5] * rw.y + MA[8] * rw.z};
    portal[0] = -1;
    if (sizeof(T) == 4 && kFp32UseMpr) return mpr_classify<T, NVP, G>(S, Rm, r, eps, deep, portal, sub, pair_mask);
    // GJK runs on the cores (finite for polytopes): rounded shapes are separated by eps iff the cores are by S.sweep + eps
    return gjk_classify<T, NVP>(S, Rm, r, (NVP == 0) ? eps + S.sweep : eps, deep);
}

// fp64 narrow phase from the raw fp32 state: normalised quaternions, exact separation rd (already minimum image).
// portal: what the fp32 XenoCollide run left (mpr_classify), or portal[0] < 0.  With a portal the vertices v1, v2, v3 of
// B (-) A are rebuilt in fp64 from their vertex indices, and if the origin lies strictly inside the tetrahedron (r, v1, v2, v3)
// -- four points of the convex set B (-) A -- the interiors intersect: overlap, decided with ~300 fp64 operations.  Otherwise (no
// portal, or the origin is not inside that tetrahedron) the fp64 GJK decides as before.  The shortcut only ever answers
// "overlap" and only when that is a fact, so the decision is the same with and without it.
template <int NVP = 0>
static __device__ __noinline__ bool polyhedron_overlap_f64(const ShapeD& S, float4 qA, float4 qB, double rx, double ry, double rz, double eps,
                                                           const int* portal)
{
    double MA[9], MB[9];
    const double na = 1.0 / sqrt((double)qA.x * qA.x + (double)qA.y * qA.y + (double)qA.z * qA.z + (double)qA.w * qA.w);
    const double nb = 1.0 / sqrt((double)qB.x * qB.x + (double)qB.y * qB.y + (double)qB.z * qB.z + (double)qB.w * qB.w);
    quat_to_matrix<double>(qA.x * na, qA.y * na, qA.z * na, qA.w * na, MA);
    quat_to_matrix<double>(qB.x * nb, qB.y * nb, qB.z * nb, qB.w * nb, MB);
    if (portal[0] >= 0) {
        double Rm[9];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) Rm[3 * i + j] = MA[i] * MB[j] + MA[3 + i] * MB[3 + j] + MA[6 + i] * MB[6 + j];
        const V3<double> r{MA[0] * rx + MA[3] * ry + MA[6] * rz, MA[1] * rx + MA[4] * ry + MA[7] * rz, MA[2] * rx + MA[5] * ry + MA[8] * rz};
        V3<double> v[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int ia = portal[k] & 255, ib = portal[k] >> 8;
            const double bx = S.vx[ib], by = S.vy[ib], bz = S.vz[ib];
            v[k] = V3<double>{Rm[0] * bx + Rm[1] * by + Rm[2] * bz + r.x - S.vx[ia], Rm[3] * bx + Rm[4] * by + Rm[5] * bz + r.y - S.vy[ia],
                              Rm[6] * bx + Rm[7] * by + Rm[8] * bz + r.z - S.vz[ia]};
        }
        // strictly inside: on the inner side of all four faces by more than 1e-9 (fp64 rounding here is ~1e-15)
        const V3<double> a = r, b = v[0], c = v[1], d = v[2];
        bool inside = true;
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            const V3<double> p = (f == 3) ? b : a;
            const V3<double> q = (f == 0) ? b : (f == 1) ? c : d;
            const V3<double> s3 = (f == 0) ? c : (f == 1) ? d : (f == 2) ? b : c;
            const V3<double> o = (f == 0) ? d : (f == 1) ? b : (f == 2) ? c : a;
            const V3<double> nn = cross(q - p, s3 - p);
            const double sp = -dot(nn, p), sd = dot(nn, o - p), nn2 = dot(nn, nn);
            // sp, sd of one sign; |sp| / |nn| > 1e-9 and the face not degenerate
            inside = inside && sp * sd > 0.0 && sp * sp > 1e-18 * nn2 && nn2 > 1e-20;
        }
        if (inside) return true;
    }
    int unused[3];
    return polyhedron_classify<double, NVP>(S, MA, MB, V3<double>{rx, ry, rz}, eps, 0.0, unused) != kGjkSeparated;
}

}  // namespace hpmc
