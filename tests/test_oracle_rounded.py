"""Pins for the oracle's rounded shapes -- spheropolygons and convex spheropolyhedra ("HPMC uses
XenoCollide for convex polygons, spheropolygons, convex polyhedra, convex spheropolyhedra").

A rounded shape is the Minkowski sum of a convex polygon / polyhedron (the core) with a disk / sphere of radius rho, so two
of them overlap iff their cores are closer than 2 rho.  The oracle's margin is D(core A, core B) - 2 rho with D found by brute
force over feature pairs (hpmc_oracle.c: core_distance).  Pinned here by things other than that code:
  - closed-form contact distances (face-face, edge-edge, vertex-vertex, crossed edges, vertex-face);
  - the distance between the cores as a quadratic programme over convex-combination weights (scipy SLSQP);
  - the already-pinned SHARP polygon margin of a densely sampled rounded outline (the arcs as many short edges);
  - the limit of a vanishing core (a disk of diameter 2 rho) and of a vanishing radius (the sharp shape);
  - symmetry, rigid-motion invariance, touch scale = root of the margin;
  - system level: brute-force O(N^2) zero-overlap invariant after sweeps, all-N twin, d_max and the grid.
"""
import math

import numpy as np
import pytest
from scipy.optimize import minimize
from scipy.spatial import ConvexHull

from oracle import hpmc_oracle as ho

SQUARE = np.array([[0.5, 0.5], [-0.5, 0.5], [-0.5, -0.5], [0.5, -0.5]])
CUBE = np.array([[sx * 0.5, sy * 0.5, sz * 0.5] for sz in (-1, 1) for sy in (-1, 1) for sx in (-1, 1)], dtype=np.float64)
IDENT = np.array([1.0, 0.0, 0.0, 0.0])


def pentagon(R):
    k = np.arange(5) * 2 * np.pi / 5
    return np.stack([R * np.cos(k), R * np.sin(k)], axis=1)


def q2(theta):
    return np.array([math.cos(theta / 2), 0.0, 0.0, math.sin(theta / 2)])


def axis_angle(axis, ang):
    a = np.asarray(axis, dtype=np.float64)
    a = a / np.linalg.norm(a)
    return np.concatenate([[math.cos(ang / 2)], math.sin(ang / 2) * a])


def qmul(a, b):
    aw, ax, ay, az = a
    bw, bx, by, bz = b
    return np.array([aw * bw - ax * bx - ay * by - az * bz, aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx, aw * bz + ax * by - ay * bx + az * bw])


def qrot(q, v):
    w, u = q[0], q[1:]
    v = np.asarray(v, dtype=np.float64)
    return v + 2 * w * np.cross(u, v) + 2 * np.cross(u, np.cross(u, v))


def rand_quat(rng):
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


# ------------------------------------------------------------------------------------------- closed forms
def test_rounded_squares_closed_form():
    rho = 0.1
    s = ho.Shape(2, ho.KIND_POLYGON, verts=SQUARE, sweep_radius=rho)
    assert s.sweep_radius == rho
    assert s.dmax == pytest.approx(2 * (math.sqrt(0.5) + rho), abs=1e-15)       # P:59 circumsphere of the rounded shape
    for g in (0.05, 0.2, 0.2000001, 0.35):
        assert s.margin([1 + g, 0.3], IDENT, IDENT) == pytest.approx(g - 2 * rho, abs=1e-12)            # edge - edge
        assert s.margin([1 + g, 1 + g], IDENT, IDENT) == pytest.approx(math.sqrt(2) * g - 2 * rho, abs=1e-12)   # corner - corner
        assert s.margin([1 + g, 1 + 0.5 * g], IDENT, IDENT) == pytest.approx(math.hypot(g, 0.5 * g) - 2 * rho, abs=1e-12)
    # intersecting cores: the (negative) separating-axis margin of the cores, minus 2 rho
    assert s.margin([0.9, 0.0], IDENT, IDENT) == pytest.approx(-0.1 - 2 * rho, abs=1e-12)


def test_rounded_pentagons_vertex_to_vertex_uses_the_euclidean_distance():
    """Vertices pointing at each other along the line of centres: the cores are |r| - 2R apart, so rounded contact is at
    2R + 2 rho.  (The sharp separating-axis margin of the same pose is (|r| - 2R) cos 36 deg: a rounded margin built from it
    would put the contact at 2R + 2 rho / cos 36 deg.)"""
    R, rho = 0.35, 0.1
    s = ho.Shape(2, ho.KIND_POLYGON, verts=pentagon(R), sweep_radius=rho)
    sharp = ho.Shape(2, ho.KIND_POLYGON, verts=pentagon(R))
    for r in (0.75, 0.9, 0.9000001, 1.0):
        assert s.margin([r, 0], q2(0.0), q2(math.pi)) == pytest.approx(r - 2 * R - 2 * rho, abs=1e-12)
        assert sharp.margin([r, 0], q2(0.0), q2(math.pi)) == pytest.approx((r - 2 * R) * math.cos(math.pi / 5), abs=1e-12)
    # vertex of A against the middle of an edge of B: both definitions agree there
    c36 = math.cos(math.pi / 5)
    for r in (0.8, 0.9):
        assert s.margin([r, 0], q2(0.0), q2(4 * math.pi / 5)) == pytest.approx(r - R - R * c36 - 2 * rho, abs=1e-12)


def test_rounded_cubes_closed_form():
    rho = 0.15
    s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE, sweep_radius=rho)
    assert s.dmax == pytest.approx(2 * (math.sqrt(0.75) + rho), abs=1e-15)
    for g in (0.1, 0.3, 0.3000001, 0.5):
        assert s.margin([1 + g, 0.2, -0.1], IDENT, IDENT) == pytest.approx(g - 2 * rho, abs=1e-12)                 # face - face
        assert s.margin([1 + g, 1 + g, 0.3], IDENT, IDENT) == pytest.approx(math.sqrt(2) * g - 2 * rho, abs=1e-12)  # parallel edges
        assert s.margin([1 + g, 1 + g, 1 + g], IDENT, IDENT) == pytest.approx(math.sqrt(3) * g - 2 * rho, abs=1e-12)  # vertex - vertex
        # crossed edges: A turned 45 deg about x has an edge along x at height sqrt(1/2); B turned 45 deg about y has an edge
        # along y at depth sqrt(1/2); the edges cross at right angles, interior to interior
        qa, qb = axis_angle([1, 0, 0], math.pi / 4), axis_angle([0, 1, 0], math.pi / 4)
        assert s.margin([0.05, -0.1, math.sqrt(2) + g], qa, qb) == pytest.approx(g - 2 * rho, abs=1e-12)
        # vertex of B (body diagonal turned onto -z) above the inside of A's top face
        d = np.array([1.0, 1.0, 1.0]) / math.sqrt(3)
        ax = np.cross(d, [0, 0, -1.0])
        qb = axis_angle(ax, math.acos(-d[2]))
        assert np.allclose(qrot(qb, d), [0, 0, -1])
        assert s.margin([0.1, -0.05, 0.5 + math.sqrt(0.75) + g], IDENT, qb) == pytest.approx(g - 2 * rho, abs=1e-12)
    assert s.margin([0.8, 0.0, 0.0], IDENT, IDENT) == pytest.approx(-0.2 - 2 * rho, abs=1e-12)


# --------------------------------------------------------------------------- distance of the cores as a QP
def qp_distance(VA, VB):
    """min | sum a_i VA_i - sum b_j VB_j | over convex-combination weights."""
    na, nb = len(VA), len(VB)
    M = np.concatenate([VA, -VB], axis=0)          # point difference = w @ M

    def f(w):
        p = w @ M
        return p @ p

    def grad(w):
        return 2 * M @ (w @ M)

    cons = [{"type": "eq", "fun": lambda w: np.sum(w[:na]) - 1, "jac": lambda w: np.concatenate([np.ones(na), np.zeros(nb)])},
            {"type": "eq", "fun": lambda w: np.sum(w[na:]) - 1, "jac": lambda w: np.concatenate([np.zeros(na), np.ones(nb)])}]
    best = np.inf
    for w0 in (np.concatenate([np.full(na, 1 / na), np.full(nb, 1 / nb)]),):
        res = minimize(f, w0, jac=grad, bounds=[(0, 1)] * (na + nb), constraints=cons, method="SLSQP",
                       options={"ftol": 1e-16, "maxiter": 500})
        best = min(best, res.fun)
    return math.sqrt(max(best, 0.0))


def random_convex_polygon(rng, n, scale=0.5):
    while True:
        pts = rng.normal(size=(3 * n, 2)) * scale * 0.6
        hull = ConvexHull(pts)
        v = pts[hull.vertices]                      # CCW for 2-D hulls
        if len(v) >= n:
            ang = np.sort(rng.choice(len(v), size=n, replace=False))
            v = v[ang]
            # strictly convex with the origin inside?
            ok = True
            for k in range(n):
                a, b, c = v[k], v[(k + 1) % n], v[(k + 2) % n]
                e, f = b - a, c - b
                if e[0] * f[1] - e[1] * f[0] <= 1e-3 or e[0] * -a[1] + e[1] * a[0] <= 1e-3:
                    ok = False
            if ok:
                return v


@pytest.mark.parametrize("seed", [1, 2])
def test_rounded_polygon_margin_equals_qp_distance_minus_two_rho(seed):
    rng = np.random.default_rng(seed)
    checked = 0
    for trial in range(60):
        nv = int(rng.integers(3, 9))
        V = pentagon(0.4) if trial % 4 == 0 else random_convex_polygon(rng, nv)
        rho = float(rng.uniform(0.02, 0.3))
        s = ho.Shape(2, ho.KIND_POLYGON, verts=V, sweep_radius=rho)
        sharp = ho.Shape(2, ho.KIND_POLYGON, verts=V)
        ta, tb = rng.uniform(0, 2 * np.pi, size=2)
        r = rng.normal(size=2)
        r *= rng.uniform(0.3, 1.1) * s.dmax / np.linalg.norm(r)
        m = s.margin(r, q2(ta), q2(tb))
        m_sharp = sharp.margin(r, q2(ta), q2(tb))
        if m_sharp <= 0:
            assert m == pytest.approx(m_sharp - 2 * rho, abs=1e-12)
            continue
        Ra = np.array([[math.cos(ta), -math.sin(ta)], [math.sin(ta), math.cos(ta)]])
        Rb = np.array([[math.cos(tb), -math.sin(tb)], [math.sin(tb), math.cos(tb)]])
        D = qp_distance(V @ Ra.T, V @ Rb.T + r)
        assert m == pytest.approx(D - 2 * rho, abs=2e-6), (trial, nv, rho)
        assert D >= m_sharp - 1e-9                        # the separating-axis margin never exceeds the distance
        checked += 1
    assert checked >= 25


def tetrahedron():
    return np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64) * 0.3


def random_hull_3d(rng, n):
    while True:
        pts = rng.normal(size=(n, 3))
        pts = 0.45 * pts / np.linalg.norm(pts, axis=1, keepdims=True) * rng.uniform(0.8, 1.0, size=(n, 1))
        hull = ConvexHull(pts)
        if len(hull.vertices) == n and np.all(hull.equations[:, 3] < -0.05):
            return pts


@pytest.mark.parametrize("seed", [1, 2])
def test_rounded_polyhedron_margin_equals_qp_distance_minus_two_rho(seed):
    rng = np.random.default_rng(100 + seed)
    checked = 0
    for trial in range(45):
        V = (CUBE, tetrahedron(), random_hull_3d(rng, 10))[trial % 3]
        rho = float(rng.uniform(0.02, 0.3))
        s = ho.Shape(3, ho.KIND_POLYHEDRON, verts=V, sweep_radius=rho)
        sharp = ho.Shape(3, ho.KIND_POLYHEDRON, verts=V)
        qa, qb = rand_quat(rng), rand_quat(rng)
        r = rng.normal(size=3)
        r *= rng.uniform(0.35, 1.1) * s.dmax / np.linalg.norm(r)
        m = s.margin(r, qa, qb)
        m_sharp = sharp.margin(r, qa, qb)
        if m_sharp <= 0:
            assert m == pytest.approx(m_sharp - 2 * rho, abs=1e-12)
            continue
        WA = np.array([qrot(qa, v) for v in V])
        WB = np.array([qrot(qb, v) for v in V]) + r
        D = qp_distance(WA, WB)
        assert m == pytest.approx(D - 2 * rho, abs=2e-6), (trial, rho)
        assert D >= m_sharp - 1e-9
        checked += 1
    assert checked >= 20


# -------------------------------------------------- the rounded outline as a sharp polygon with many short edges
def rounded_outline(V, rho, per_corner):
    """Points ON the boundary of polygon (+) disk(rho): at every vertex the arc between the outward normals of the two edges
    that meet there, `per_corner` points per arc, CCW.  Their hull lies inside the rounded shape, within the sagitta
    rho (1 - cos(dtheta / 2)) of its boundary."""
    n = len(V)
    out = []
    sag = 0.0
    for k in range(n):
        a, b, c = V[(k - 1) % n], V[k], V[(k + 1) % n]
        e0, e1 = b - a, c - b
        t0 = math.atan2(-e0[0], e0[1])      # angle of the outward normal (e_y, -e_x) of the incoming edge
        t1 = math.atan2(-e1[0], e1[1])
        while t1 < t0:
            t1 += 2 * math.pi
        for j in range(per_corner):
            t = t0 + (t1 - t0) * j / (per_corner - 1)
            out.append(b + rho * np.array([math.cos(t), math.sin(t)]))
        sag = max(sag, rho * (1 - math.cos(0.5 * (t1 - t0) / (per_corner - 1))))
    return np.array(out), sag


def test_rounded_polygon_margin_against_the_sharp_margin_of_its_sampled_outline():
    rng = np.random.default_rng(7)
    n_sign = 0
    for trial in range(200):
        if trial % 2 == 0:
            V, per = pentagon(0.35), 6            # 30 vertices
        else:
            V, per = SQUARE * 0.7, 8              # 32 vertices
        rho = float(rng.uniform(0.05, 0.2))
        dense, sag = rounded_outline(V, rho, per)
        s = ho.Shape(2, ho.KIND_POLYGON, verts=V, sweep_radius=rho)
        sd = ho.Shape(2, ho.KIND_POLYGON, verts=dense)
        ta, tb = rng.uniform(0, 2 * np.pi, size=2)
        r = rng.normal(size=2)
        r *= rng.uniform(0.5, 1.05) * s.dmax / np.linalg.norm(r)
        m = s.margin(r, q2(ta), q2(tb))
        md = sd.margin(r, q2(ta), q2(tb))
        if m > 0:
            # disjoint: the hulls are inside the rounded shapes, so their distance is >= m and <= m + 2 sag; the separating-axis
            # margin of the hulls is that distance times at least the cosine of half an arc step
            half_step = math.pi / (per - 1) / 2
            assert md <= m + 2 * sag + 1e-12
            assert md >= m * math.cos(half_step) - 1e-12
        elif m < -2 * sag - 1e-9:
            assert md < 0                        # the rounded shapes interpenetrate by more than the sampling error
            n_sign += 1
    assert n_sign > 20


# -------------------------------------------------------------------------------- limits and symmetries
def test_vanishing_core_is_a_disk_and_vanishing_radius_is_the_sharp_shape():
    rho = 0.5
    tiny = ho.Shape(2, ho.KIND_POLYGON, verts=pentagon(1e-4), sweep_radius=rho)
    disk = ho.Shape(2, ho.KIND_DISK, diameter=2 * rho)
    tiny3 = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE * 1e-4, sweep_radius=rho)
    sphere = ho.Shape(3, ho.KIND_DISK, diameter=2 * rho)
    rng = np.random.default_rng(5)
    for _ in range(50):
        r = rng.uniform(-1.2, 1.2, size=3)
        assert tiny.margin(r[:2], q2(rng.uniform(0, 6)), q2(rng.uniform(0, 6))) == pytest.approx(disk.margin(r[:2], IDENT, IDENT), abs=2.1e-4)
        assert tiny3.margin(r, rand_quat(rng), rand_quat(rng)) == pytest.approx(sphere.margin(r, IDENT, IDENT), abs=2.1e-4)
    sharp = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE)
    zero = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE, sweep_radius=0.0)
    for _ in range(20):
        r, qa, qb = rng.uniform(-1.5, 1.5, size=3), rand_quat(rng), rand_quat(rng)
        assert zero.margin(r, qa, qb) == sharp.margin(r, qa, qb)


def test_rounded_margin_symmetry_rigid_motion_and_touch_scale():
    rng = np.random.default_rng(11)
    s2 = ho.Shape(2, ho.KIND_POLYGON, verts=pentagon(0.35), sweep_radius=0.1)
    s3 = ho.Shape(3, ho.KIND_POLYHEDRON, verts=CUBE * 0.7, sweep_radius=0.15)
    for _ in range(40):
        ta, tb, tg = rng.uniform(0, 2 * np.pi, size=3)
        r = rng.uniform(-0.9, 0.9, size=2)
        m = s2.margin(r, q2(ta), q2(tb))
        assert s2.margin(-r, q2(tb), q2(ta)) == pytest.approx(m, abs=1e-12)
        Rg = np.array([[math.cos(tg), -math.sin(tg)], [math.sin(tg), math.cos(tg)]])
        assert s2.margin(Rg @ r, q2(ta + tg), q2(tb + tg)) == pytest.approx(m, abs=1e-12)
        lam = s2.touch_scale(r, q2(ta), q2(tb))
        assert abs(s2.margin(lam * r, q2(ta), q2(tb))) < 1e-9
        qa, qb, qg = rand_quat(rng), rand_quat(rng), rand_quat(rng)
        r3 = rng.uniform(-1.2, 1.2, size=3)
        m3 = s3.margin(r3, qa, qb)
        assert s3.margin(-r3, qb, qa) == pytest.approx(m3, abs=1e-12)
        assert s3.margin(qrot(qg, r3), qmul(qg, qa), qmul(qg, qb)) == pytest.approx(m3, abs=1e-11)
        lam = s3.touch_scale(r3, qa, qb)
        assert abs(s3.margin(lam * r3, qa, qb)) < 1e-9


# ------------------------------------------------------------------------------------------- system level
def rounded_system(dim, n_lat, seed=1):
    rng = np.random.default_rng(seed)
    if dim == 2:
        verts, rho, spacing = pentagon(0.35), 0.1, 1.0          # d_max = 0.9 < spacing: any orientation is overlap-free
        N = n_lat * n_lat
        idx = (np.arange(n_lat) + 0.5) * spacing - 0.5 * n_lat * spacing
        y, x = np.meshgrid(idx, idx, indexing="ij")
        pos = np.zeros((N, 4), np.float32)
        pos[:, 0], pos[:, 1] = x.ravel(), y.ravel()
        th = rng.uniform(0, 2 * np.pi, size=N)
        quat = np.zeros((N, 4), np.float32)
        quat[:, 0], quat[:, 3] = np.cos(th / 2), np.sin(th / 2)
        L = (n_lat * spacing,) * 2
        kind = ho.KIND_POLYGON
    else:
        verts, rho, spacing = CUBE * 0.6, 0.15, 1.4             # d_max = 2 (0.52 + 0.15) = 1.339 < spacing
        N = n_lat ** 3
        idx = (np.arange(n_lat) + 0.5) * spacing - 0.5 * n_lat * spacing
        z, y, x = np.meshgrid(idx, idx, idx, indexing="ij")
        pos = np.zeros((N, 4), np.float32)
        pos[:, 0], pos[:, 1], pos[:, 2] = x.ravel(), y.ravel(), z.ravel()
        q = rng.normal(size=(N, 4))
        quat = (q / np.linalg.norm(q, axis=1, keepdims=True)).astype(np.float32)
        L = (n_lat * spacing,) * 3
        kind = ho.KIND_POLYHEDRON
    o = ho.Oracle(dim, L, kind, N, seed, verts=verts, sweep_radius=rho)
    o.set_moves(0.15, 0.3, 4)
    o.set_state(pos, quat)
    return o, verts, rho


@pytest.mark.parametrize("dim,n_lat", [(2, 12), (3, 6)])
def test_rounded_system_grid_sweeps_and_zero_overlap_invariant(dim, n_lat):
    o, verts, rho = rounded_system(dim, n_lat)
    dmax = 2 * (np.max(np.linalg.norm(verts, axis=1)) + rho)
    assert np.all(o.w[:dim] >= dmax * (1 + 2.0 ** -10))             # R11 with the rounded circumsphere
    assert o.count_overlaps_bruteforce() == 0
    for s in range(12):
        o.sweep()
        assert o.count_overlaps_bruteforce() == 0
        assert o.count_overlaps_cells() == 0
    c = o.counters()
    assert c["trans_acc"] > 0 and c["rot_acc"] > 0 and c["trans_rej_overlap"] > 0 and c["rot_rej_overlap"] > 0
    # O6 twin: scanning all N - 1 particles instead of the 3^d cells makes identical decisions
    a, _, _ = rounded_system(dim, n_lat)
    b, _, _ = rounded_system(dim, n_lat)
    for s in range(3):
        a.sweep()
        b.sweep(neighbour_mode=1)
    pa, qa = a.get_state(); pb, qb = b.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)


def test_planted_rounded_overlap_is_counted():
    o, verts, rho = rounded_system(2, 8)
    pos, quat = o.get_state()
    # cores 0.15 apart at closest (vertex to vertex): rounded shapes overlap (2 rho = 0.2), sharp ones would not
    pos[1, 0] = pos[0, 0] + 0.7 + 0.15
    pos[1, 1] = pos[0, 1]
    quat[0] = q2(0.0); quat[1] = q2(math.pi)
    o.set_state(pos, quat)
    assert o.count_overlaps_bruteforce() == 1 and o.count_overlaps_cells() == 1
    sharp = ho.Oracle(2, (8.0, 8.0), ho.KIND_POLYGON, 64, 1, verts=verts)
    sharp.set_state(pos, quat)
    assert sharp.count_overlaps_bruteforce() == 0
