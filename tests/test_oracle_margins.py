"""Pins for the oracle's overlap margins (O4).

Each pin is something other than the oracle itself: closed-form contact distances, the AABB interval
test, polygon clipping (Sutherland-Hodgman), a Chebyshev-centre LP over scipy-ConvexHull faces, and
symmetry / rigid-motion invariance.
"""
import math

import numpy as np
import pytest
from scipy.optimize import linprog
from scipy.spatial import ConvexHull

from oracle import hpmc_oracle as ho
from paper_1509_04692_b200 import workloads as wl

PENT = wl.regular_polygon(5, 0.5)
CUBE = wl.cube_vertices(1.0)


def q2(theta):
    return np.array([math.cos(theta / 2), 0.0, 0.0, math.sin(theta / 2)])


def rand_quat(rng):
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


def qmul(a, b):
    """Hamilton product (w, x, y, z): this file's own algebra, not the input generator's."""
    aw, ax, ay, az = np.asarray(a, dtype=np.float64)
    bw, bx, by, bz = np.asarray(b, dtype=np.float64)
    return np.array([aw * bw - ax * bx - ay * by - az * bz, aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx, aw * bz + ax * by - ay * bx + az * bw])


def cube_group():
    """The 24 proper rotations of the cube as unit quaternions: identity, 90/180/270 about the 3 face axes (9), 120/240 about
    the 4 body diagonals (8), 180 about the 6 edge axes (6) -- written out from the axis-angle form."""
    out = [np.array([1.0, 0, 0, 0])]
    for ax in np.eye(3):
        for ang in (np.pi / 2, np.pi, 3 * np.pi / 2):
            out.append(np.concatenate([[np.cos(ang / 2)], np.sin(ang / 2) * ax]))
    for sx in (1, -1):
        for sy in (1, -1):
            d = np.array([1.0, sx, sy]) / np.sqrt(3.0)
            for ang in (2 * np.pi / 3, 4 * np.pi / 3):
                out.append(np.concatenate([[np.cos(ang / 2)], np.sin(ang / 2) * d]))
    for e in ([1, 1, 0], [1, -1, 0], [1, 0, 1], [1, 0, -1], [0, 1, 1], [0, 1, -1]):
        d = np.array(e, dtype=np.float64) / np.sqrt(2.0)
        out.append(np.concatenate([[0.0], d]))
    assert len(out) == 24
    return np.array(out)


def qrot(q, v):
    w, u = q[0], q[1:]
    return v + 2 * w * np.cross(u, v) + 2 * np.cross(u, np.cross(u, v))


# ---------------------------------------------------------------- disks (P5)
def test_disk_margin_closed_form():
    s = ho.Shape(2, ho.KIND_DISK, diameter=1.0)
    ident = [1, 0, 0, 0]
    assert s.margin([1.0, 0.0], ident, ident) == 0.0          # touching is not overlap (R15)
    assert s.margin([0.6, 0.8], ident, ident) == pytest.approx(0.0, abs=1e-15)
    assert s.margin([0.3, 0.4], ident, ident) == pytest.approx(-0.5)
    assert s.margin([3.0, 4.0], ident, ident) == pytest.approx(4.0)
    s3 = ho.Shape(3, ho.KIND_DISK, diameter=2.0)
    assert s3.margin([1.0, 2.0, 2.0], ident, ident) == pytest.approx(1.0)


# ------------------------------------------------------------- pentagons (P6)
def test_pentagon_contact_distances_closed_form():
    s = ho.Shape(2, ho.KIND_POLYGON, verts=PENT)
    assert s.dmax == pytest.approx(1.0)
    c36 = math.cos(math.pi / 5)
    # vertex-vertex along the line of centres: contact at 2R = 1.0; margin = (r-1) cos 36deg
    for r in (0.9, 0.999, 1.0, 1.001, 1.1):
        assert s.margin([r, 0], q2(0.0), q2(math.pi)) == pytest.approx((r - 1.0) * c36, abs=1e-12)
    # edge-edge: contact at 2 R cos 36deg = 0.809017
    for r in (0.7, 0.809017, 0.9):
        assert s.margin([r, 0], q2(-math.pi / 5), q2(4 * math.pi / 5)) == pytest.approx(r - 2 * 0.5 * c36, abs=1e-12)
    # vertex (A) against edge (B): contact at R + R cos 36deg = 0.904508
    for r in (0.85, 0.904508, 0.95):
        assert s.margin([r, 0], q2(0.0), q2(4 * math.pi / 5)) == pytest.approx(r - 0.5 - 0.5 * c36, abs=1e-12)
    assert 2 * 0.5 * c36 == pytest.approx(0.809017, abs=1e-6)
    assert 0.5 + 0.5 * c36 == pytest.approx(0.904508, abs=1e-6)


def test_unit_squares_reduce_to_aabb():
    sq = np.array([[0.5, 0.5], [-0.5, 0.5], [-0.5, -0.5], [0.5, -0.5]])
    s = ho.Shape(2, ho.KIND_POLYGON, verts=sq)
    rng = np.random.default_rng(3)
    for _ in range(500):
        r = rng.uniform(-1.6, 1.6, size=2)
        expect = max(abs(r[0]), abs(r[1])) - 1.0
        # any multiple of 90 degrees leaves a square unchanged
        m = s.margin(r, q2(rng.integers(0, 4) * math.pi / 2), q2(rng.integers(0, 4) * math.pi / 2))
        assert m == pytest.approx(expect, abs=1e-12)


def test_polygon_rejects_bad_vertex_lists():
    with pytest.raises(ValueError):
        ho.Shape(2, ho.KIND_POLYGON, verts=PENT[::-1].copy())                       # clockwise
    with pytest.raises(ValueError):
        ho.Shape(2, ho.KIND_POLYGON, verts=np.array([[0, 0], [1, 0], [0.2, 0.2], [0, 1.0]]))  # concave


def _clip_area(subject, clip):
    """Sutherland-Hodgman: area of (convex subject) intersected with (convex CCW clip)."""
    out = [tuple(p) for p in subject]
    n = len(clip)
    for k in range(n):
        a, b = clip[k], clip[(k + 1) % n]
        ex, ey = b[0] - a[0], b[1] - a[1]
        inp, out = out, []
        if not inp:
            break
        for i in range(len(inp)):
            p, q = inp[i], inp[(i + 1) % len(inp)]
            sp = ex * (p[1] - a[1]) - ey * (p[0] - a[0])
            sq = ex * (q[1] - a[1]) - ey * (q[0] - a[0])
            if sp >= 0:
                out.append(p)
            if (sp > 0 and sq < 0) or (sp < 0 and sq > 0):
                t = sp / (sp - sq)
                out.append((p[0] + t * (q[0] - p[0]), p[1] + t * (q[1] - p[1])))
    if len(out) < 3:
        return 0.0
    x = np.array([p[0] for p in out]); y = np.array([p[1] for p in out])
    return 0.5 * abs(np.dot(x, np.roll(y, -1)) - np.dot(y, np.roll(x, -1)))


def _world2(verts, theta, r):
    c, s = math.cos(theta), math.sin(theta)
    R = np.array([[c, -s], [s, c]])
    return verts @ R.T + np.asarray(r)


def _random_convex_polygon(rng, nv):
    ang = np.sort(rng.uniform(0, 2 * math.pi, size=nv))
    while np.max(np.diff(np.concatenate([ang, [ang[0] + 2 * math.pi]]))) > 0.9 * math.pi:
        ang = np.sort(rng.uniform(0, 2 * math.pi, size=nv))
    return 0.5 * np.stack([np.cos(ang), np.sin(ang)], axis=1)  # points on a circle are in convex position


@pytest.mark.parametrize("which", ["pentagon", "random"])
def test_polygon_margin_sign_vs_clipping(which):
    rng = np.random.default_rng(11)
    n_pairs, disagreements, near = 6000, 0, 0
    for trial in range(n_pairs):
        verts = PENT if which == "pentagon" else _random_convex_polygon(rng, int(rng.integers(3, 9)))
        s = ho.Shape(2, ho.KIND_POLYGON, verts=verts)
        ta, tb = rng.uniform(0, 2 * math.pi, size=2)
        r = rng.uniform(0.55, 1.05) * np.array([math.cos(ta * 3.1), math.sin(ta * 3.1)])
        m = s.margin(r, q2(ta), q2(tb))
        area = _clip_area(_world2(verts, ta, [0, 0]), _world2(verts, tb, r))
        if abs(m) < 1e-9:
            near += 1
            continue
        if m < 0:
            # penetration depth |m| along the best axis implies an intersection of area >= ~m^2/4
            assert area > 0.0, (trial, m, area)
        else:
            assert area < 1e-18, (trial, m, area)
    assert near < 5 and disagreements == 0


def test_polygon_margin_symmetry_and_rigid_motion():
    rng = np.random.default_rng(5)
    s = ho.Shape(2, ho.KIND_POLYGON, verts=PENT)
    for _ in range(300):
        ta, tb, g = rng.uniform(0, 2 * math.pi, size=3)
        r = rng.uniform(-1, 1, size=2)
        m = s.margin(r, q2(ta), q2(tb))
        assert s.margin(-r, q2(tb), q2(ta)) == pytest.approx(m, abs=1e-12)      # m(A,B) = m(B,A)
        c, sn = math.cos(g), math.sin(g)
        rg = np.array([c * r[0] - sn * r[1], sn * r[0] + c * r[1]])
        assert s.margin(rg, q2(ta + g), q2(tb + g)) == pytest.approx(m, abs=1e-12)  # common rotation


# ---------------------------------------------------------------- cubes (P7)
def test_cube_faces_edges_derived_by_brute_force():
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE)
    assert s.nfaces == 6 and s.nedgedirs == 3          # 6 + 6 + 2*9 axis evaluations per pair
    assert s.dmax == pytest.approx(math.sqrt(3.0))
    nn, cc = s.faces()
    assert np.allclose(cc, 0.5)
    assert sorted(map(tuple, np.round(nn).astype(int).tolist())) == sorted(
        [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)])
    tet = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float)
    st = ho.Shape(3, ho.KIND_POLYHEDRON, verts=tet)
    assert st.nfaces == 4 and st.nedgedirs == 6
    octa = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=float)
    so = ho.Shape(3, ho.KIND_POLYHEDRON, verts=octa)
    assert so.nfaces == 8 and so.nedgedirs == 6
    with pytest.raises(ValueError):  # an interior point is not a hull vertex
        ho.Shape(3, ho.KIND_POLYHEDRON, verts=np.vstack([CUBE, [[0.1, 0.0, 0.0]]]))


def test_axis_aligned_cubes_reduce_to_aabb():
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE)
    rng = np.random.default_rng(9)
    ident = np.array([1.0, 0, 0, 0])
    G = cube_group()
    for _ in range(300):
        r = rng.uniform(-1.7, 1.7, size=3)
        expect = np.max(np.abs(r)) - 1.0
        qa, qb = G[rng.integers(0, 24)], G[rng.integers(0, 24)]   # cube symmetries leave the cube unchanged
        m = s.margin(r, qa, qb)
        if expect < 0 or np.sum(np.abs(r) > 1.0) == 1:
            assert m == pytest.approx(expect, abs=1e-12)
        else:
            # disjoint along several axes: the SAT margin is the best FACE axis (edge-edge axes are parallel here)
            assert m == pytest.approx(expect, abs=1e-12)
        assert s.margin(r, ident, ident) == pytest.approx(expect, abs=1e-12)


def test_cube_contact_distances_closed_form():
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE)
    ident = np.array([1.0, 0, 0, 0])
    # face-face contact at 1.0
    assert s.margin([1.0, 0, 0], ident, ident) == pytest.approx(0.0, abs=1e-15)
    assert s.margin([0.99, 0, 0], ident, ident) < 0 < s.margin([1.01, 0, 0], ident, ident)
    # edge-edge contact along (1,1,0)/sqrt2: A identity; B = A turned 90 deg about its own (1,-1,0)... use the
    # classic crossed-edges pose: B rotated by 90 deg about the line of centres u=(1,1,0)/sqrt2.
    u = np.array([1.0, 1.0, 0.0]) / math.sqrt(2)
    qb = np.concatenate([[math.cos(math.pi / 4)], math.sin(math.pi / 4) * u])
    for dist, sign in ((math.sqrt(2) - 1e-3, -1), (math.sqrt(2) + 1e-3, +1)):
        assert np.sign(s.margin(dist * u, ident, qb)) == sign
    # vertex-vertex along (1,1,1)/sqrt3 at sqrt3 (B = point reflection of A = same cube)
    v = np.ones(3) / math.sqrt(3)
    for dist, sign in ((math.sqrt(3) - 1e-3, -1), (math.sqrt(3) + 1e-3, +1)):
        assert np.sign(s.margin(dist * v, ident, ident)) == sign
    # any centre distance >= circumsphere diameter is disjoint whatever the orientations
    rng = np.random.default_rng(2)
    for _ in range(200):
        d = rand_quat(rng)[:3]; d /= np.linalg.norm(d)
        assert s.margin(1.7321 * d, rand_quat(rng), rand_quat(rng)) >= 0.0


def _chebyshev_radius(faces_a, faces_b):
    """max t s.t. n.x + t <= c over all faces of both bodies; t > 0 <=> interiors intersect."""
    A = np.vstack([np.hstack([f[0], np.ones((f[0].shape[0], 1))]) for f in (faces_a, faces_b)])
    b = np.concatenate([faces_a[1], faces_b[1]])
    res = linprog(c=[0, 0, 0, -1.0], A_ub=A, b_ub=b, bounds=[(None, None)] * 3 + [(None, None)], method="highs")
    assert res.status == 0
    return res.x[3]


def _world_faces(verts, q, r):
    wv = np.array([qrot(q, v) for v in verts]) + np.asarray(r)
    hull = ConvexHull(wv)                      # independent face derivation (Qhull)
    eq = hull.equations                        # n.x + off <= 0 inside
    return eq[:, :3], -eq[:, 3]


@pytest.mark.parametrize("body", ["cube", "tetra", "random12"])
def test_polyhedron_margin_sign_vs_lp_and_gjk(body):
    rng = np.random.default_rng(21)
    if body == "cube":
        verts, lo, hi = CUBE, 0.95, 1.75
    elif body == "tetra":
        verts, lo, hi = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float) * 0.5, 0.3, 1.75
    else:
        p = rng.normal(size=(12, 3)); verts = 0.6 * p / np.linalg.norm(p, axis=1, keepdims=True)
        lo, hi = 0.7, 1.25
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=verts)
    n_overlap = n_disjoint = 0
    for _ in range(700):
        qa, qb = rand_quat(rng), rand_quat(rng)
        d = rand_quat(rng)[:3]; d /= np.linalg.norm(d)
        r = rng.uniform(lo, hi) * d
        m = s.margin(r, qa, qb)
        if abs(m) < 1e-7:
            continue
        t = _chebyshev_radius(_world_faces(verts, qa, [0, 0, 0]), _world_faces(verts, qb, r))
        assert (t > 0) == (m < 0), (m, t)
        g = s.gjk(r, qa, qb)                    # the oracle's own fp64 GJK must agree with sign(m)
        assert g == (1 if m < 0 else 0), (m, g)
        n_overlap += m < 0; n_disjoint += m > 0
    assert n_overlap > 100 and n_disjoint > 100


def test_polyhedron_margin_symmetry_and_rigid_motion():
    rng = np.random.default_rng(8)
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE)
    for _ in range(200):
        qa, qb, g = rand_quat(rng), rand_quat(rng), rand_quat(rng)
        r = rng.uniform(-1.2, 1.2, size=3)
        m = s.margin(r, qa, qb)
        assert s.margin(-r, qb, qa) == pytest.approx(m, abs=1e-12)
        assert s.margin(qrot(g, r), qmul(g, qa), qmul(g, qb)) == pytest.approx(m, abs=1e-12)


def test_random_cube_overlap_probability_at_lattice_spacing():
    """R27: two unit cubes with independent uniform orientations at centre distance 1.25 along an axis
    overlap far too often for BASELINE.json configs[3]'s literal start (0.877; 0.109 at 1.5)."""
    rng = np.random.default_rng(4)
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE)
    for dist, p_expect in ((1.25, 0.877), (1.5, 0.109)):
        n = 4000
        hits = sum(s.margin([dist, 0, 0], rand_quat(rng), rand_quat(rng)) < 0 for _ in range(n))
        se = math.sqrt(p_expect * (1 - p_expect) / n)
        assert abs(hits / n - p_expect) < 5 * se + 0.004


def test_gjk_2d_agrees_with_sat_sign():
    rng = np.random.default_rng(17)
    s = ho.Shape(2, ho.KIND_POLYGON, verts=PENT)
    for _ in range(3000):
        ta, tb, tr = rng.uniform(0, 2 * math.pi, size=3)
        r = rng.uniform(0.6, 1.05) * np.array([math.cos(tr), math.sin(tr)])
        m = s.margin(r, q2(ta), q2(tb))
        if abs(m) > 1e-9:
            assert s.gjk(r, q2(ta), q2(tb)) == (1 if m < 0 else 0)
