"""Seeded synthetic inputs I0..I4 for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the test oracle, so it holds none of the method's
arithmetic: no RNG stream of the sweep, no cell function, no overlap test.  It only places
particles on a lattice, draws orientations from a seeded numpy generator and lists shape vertices.
It imports numpy only (no torch, no binding, no oracle).

The paper's own benchmark states (pentagons at phi=0.676, dodecahedra at phi=0.5) are
equilibrated configurations that are not available; BASELINE.json fixes these lattice starts as
stand-ins.  Site (ix,iy[,iz]) -> particle index i = ix + n_lat*(iy + n_lat*iz),
x_k = (i_k + 0.5)*spacing - L/2, generated in fp64 and rounded once to fp32.
"""
from dataclasses import dataclass, field

import numpy as np

KIND_DISK, KIND_POLYGON, KIND_POLYHEDRON = 0, 1, 2


@dataclass
class Workload:
    name: str
    dim: int
    N: int
    L: tuple
    kind: int
    diameter: float
    verts: np.ndarray          # (nverts, dim) fp64 body-frame vertices, or None for disks
    d: float
    a: float
    n_select: int
    sweeps: int                # run length BASELINE.json quotes for this config
    pos4: np.ndarray           # (N,4) fp32: x,y,z,0
    quat4: np.ndarray          # (N,4) fp32: w,x,y,z
    warmup_sweeps: int = 0     # sweeps to melt the lattice before timing
    notes: str = ""
    extra: dict = field(default_factory=dict)
    sweep_radius: float = 0.0  # > 0: spheropolygon / spheropolyhedron, `verts` is the core


def regular_polygon(nv: int, circumradius: float) -> np.ndarray:
    """CCW vertices, vertex k at angle 2*pi*k/nv (R17)."""
    k = np.arange(nv, dtype=np.float64)
    ang = 2.0 * np.pi * k / nv
    return np.stack([circumradius * np.cos(ang), circumradius * np.sin(ang)], axis=1)


def cube_vertices(edge: float) -> np.ndarray:
    h = 0.5 * edge
    return np.array([[sx * h, sy * h, sz * h] for sz in (-1, 1) for sy in (-1, 1) for sx in (-1, 1)], dtype=np.float64)


def _lattice(dim: int, n_lat: int, spacing: float) -> np.ndarray:
    L = n_lat * spacing
    idx = np.arange(n_lat, dtype=np.float64)
    coord = (idx + 0.5) * spacing - 0.5 * L
    if dim == 2:
        y, x = np.meshgrid(coord, coord, indexing="ij")
        p = np.stack([x.ravel(), y.ravel(), np.zeros(n_lat * n_lat)], axis=1)
    else:
        z, y, x = np.meshgrid(coord, coord, coord, indexing="ij")
        p = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    pos4 = np.zeros((p.shape[0], 4), dtype=np.float32)
    pos4[:, :3] = p.astype(np.float32)
    return pos4


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def _identity_quats(N: int) -> np.ndarray:
    q = np.zeros((N, 4), dtype=np.float32)
    q[:, 0] = 1.0
    return q


def _qmul(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    aw, ax, ay, az = a[..., 0], a[..., 1], a[..., 2], a[..., 3]
    bw, bx, by, bz = b[..., 0], b[..., 1], b[..., 2], b[..., 3]
    return np.stack([aw * bw - ax * bx - ay * by - az * bz,
                     aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx,
                     aw * bz + ax * by - ay * bx + az * bw], axis=-1)


def _cube_group() -> np.ndarray:
    """The 24 proper rotations of the cube as unit quaternions (closure of two 90-degree turns)."""
    s = np.sqrt(0.5)
    gens = [np.array([s, 0, 0, s]), np.array([s, s, 0, 0])]
    elems = [np.array([1.0, 0, 0, 0])]
    frontier = list(elems)
    while frontier:
        nxt = []
        for e in frontier:
            for g in gens:
                c = _qmul(e, g)
                if c[np.argmax(np.abs(c) > 1e-9)] < 0:
                    c = -c
                if not any(np.allclose(c, f, atol=1e-9) for f in elems):
                    elems.append(c)
                    nxt.append(c)
        frontier = nxt
    assert len(elems) == 24
    return np.array(elems)


def disks(n_lat: int = 64, seed: int = 1, spacing: float = 1.1, name: str = "k0_disks") -> Workload:
    """I0: BASELINE.json configs[0]; 2-D hard disks, diameter 1, square lattice spacing 1.1 (phi=0.649)."""
    pos4 = _lattice(2, n_lat, spacing)
    N = n_lat * n_lat
    L = n_lat * spacing
    return Workload(name=name, dim=2, N=N, L=(L, L), kind=KIND_DISK, diameter=1.0, verts=None, d=0.15, a=0.0,
                    n_select=4, sweeps=1000, pos4=pos4, quat4=_identity_quats(N), warmup_sweeps=200,
                    extra={"seed": seed, "phi": N * np.pi * 0.25 / (L * L)})


def pentagons(n_lat: int = 64, seed: int = 1, name: str = None, sweeps: int = None) -> Workload:
    """I1/I2/I4: configs[1], [2], [4]; regular pentagons R=0.5 on a square lattice at spacing 1.0.

    Circumcircles of lattice neighbours are exactly tangent, so an orientation whose vertex
    direction lies within 0.01 rad of a lattice axis is redrawn (R29): every pair then starts with
    a positive gap >= 5e-5.
    """
    N = n_lat * n_lat
    pos4 = _lattice(2, n_lat, 1.0)
    rng = _rng(seed, 101)
    theta = 2.0 * np.pi * rng.random(N)
    k = np.arange(5) * (2.0 * np.pi / 5.0)
    for _ in range(64):
        ang = np.mod(theta[:, None] + k[None, :], 0.5 * np.pi)
        bad = np.any((ang < 0.01) | (ang > 0.5 * np.pi - 0.01), axis=1)
        if not bad.any():
            break
        theta[bad] = 2.0 * np.pi * rng.random(int(bad.sum()))
    else:
        raise RuntimeError("orientation redraw did not converge")
    quat4 = np.zeros((N, 4), dtype=np.float32)
    quat4[:, 0] = np.cos(0.5 * theta).astype(np.float32)
    quat4[:, 3] = np.sin(0.5 * theta).astype(np.float32)
    if name is None:
        name = {64: "k1_pentagons_4096", 1024: "k2_pentagons_1M", 4096: "k4_pentagons_16M"}.get(n_lat, f"pentagons_{N}")
    if sweeps is None:
        sweeps = {64: 10000, 1024: 1000, 4096: 100}.get(n_lat, 100)
    warm = {64: 200, 1024: 50, 4096: 10}.get(n_lat, 50)
    L = float(n_lat)
    area = 5.0 / 2.0 * 0.25 * np.sin(2.0 * np.pi / 5.0)
    return Workload(name=name, dim=2, N=N, L=(L, L), kind=KIND_POLYGON, diameter=0.0, verts=regular_polygon(5, 0.5),
                    d=0.1, a=0.1, n_select=4, sweeps=sweeps, pos4=pos4, quat4=quat4, warmup_sweeps=warm,
                    extra={"seed": seed, "phi": N * area / (L * L)})


def rounded_polygons(n_lat: int = 64, seed: int = 1, nv: int = 5, circumradius: float = 0.35, sweep_radius: float = 0.1,
                     spacing: float = 1.0, d: float = 0.1, a: float = 0.3, name: str = None) -> Workload:
    """Spheropolygons: regular nv-gons of the given circumradius swept by a disk of `sweep_radius`, on a square lattice
    with uniform-random orientations.  The caller keeps d_max = 2 (circumradius + sweep_radius) below `spacing`, so that every
    orientation is overlap-free."""
    assert 2.0 * (circumradius + sweep_radius) < spacing
    N = n_lat * n_lat
    pos4 = _lattice(2, n_lat, spacing)
    theta = 2.0 * np.pi * _rng(seed, 404).random(N)
    quat4 = np.zeros((N, 4), dtype=np.float32)
    quat4[:, 0] = np.cos(0.5 * theta).astype(np.float32)
    quat4[:, 3] = np.sin(0.5 * theta).astype(np.float32)
    L = n_lat * spacing
    side = 2.0 * circumradius * np.sin(np.pi / nv)
    area = 0.5 * nv * circumradius ** 2 * np.sin(2.0 * np.pi / nv) + nv * side * sweep_radius + np.pi * sweep_radius ** 2
    return Workload(name=name or f"rounded_{nv}gons_{N}", dim=2, N=N, L=(L, L), kind=KIND_POLYGON, diameter=0.0,
                    verts=regular_polygon(nv, circumradius), sweep_radius=sweep_radius, d=d, a=a, n_select=4, sweeps=100,
                    pos4=pos4, quat4=quat4, warmup_sweeps=50, extra={"seed": seed, "phi": N * area / (L * L)})


def cubes(n_lat: int = 32, seed: int = 1, max_tilt: float = 0.15, name: str = "k3_cubes", spacing: float = 1.25,
          d: float = 0.1, a: float = 0.1, edge: float = 1.0, sweep_radius: float = 0.0) -> Workload:
    """I3: configs[3]; unit cubes as generic 8-vertex polyhedra on a simple-cubic lattice, spacing 1.25.

    DEVIATION (R27): uniform-random orientations at spacing 1.25 overlap with probability 0.877 per
    bond, so the start is q_i = g_i (x) tau_i with g_i uniform over the 24 proper cube rotations and
    tau_i a tilt of angle uniform in [0, 0.15] rad about a uniform random axis; each cube's half
    extent along a lattice axis is then <= 0.61 < 0.625 and the start is overlap-free.

    Other `spacing` / `max_tilt` / move sizes give test cases (the caller keeps 0.5 (1 + sqrt 2 sin(max_tilt)) below
    spacing / 2): e.g. spacing 1.0006 with tilts of 2e-4 rad is a crystal of nearly parallel, nearly touching faces.
    `edge` and `sweep_radius` make rounded cubes (spheropolyhedra): a cube of that edge swept by a sphere of that
    radius; the caller keeps 0.61 edge + sweep_radius below spacing / 2.
    """
    N = n_lat ** 3
    pos4 = _lattice(3, n_lat, spacing)
    rng = _rng(seed, 303)
    G = _cube_group()
    g = G[rng.integers(0, 24, size=N)]
    z = 2.0 * rng.random(N) - 1.0
    phi = 2.0 * np.pi * rng.random(N)
    rho = np.sqrt(1.0 - z * z)
    axis = np.stack([rho * np.cos(phi), rho * np.sin(phi), z], axis=1)
    ang = max_tilt * rng.random(N)
    tau = np.concatenate([np.cos(0.5 * ang)[:, None], np.sin(0.5 * ang)[:, None] * axis], axis=1)
    q = _qmul(g, tau)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    L = n_lat * spacing
    return Workload(name=name, dim=3, N=N, L=(L, L, L), kind=KIND_POLYHEDRON, diameter=0.0, verts=cube_vertices(edge),
                    sweep_radius=sweep_radius,
                    d=d, a=a, n_select=4, sweeps=1000, pos4=pos4, quat4=q.astype(np.float32), warmup_sweeps=200,
                    notes="initial orientations: cube-group element x tilt<=0.15 rad (BASELINE.json's uniform-random "
                          "orientations are infeasible at spacing 1.25)",
                    extra={"seed": seed, "phi": N / L ** 3})


def dodecahedron_vertices(circumradius: float = 0.5) -> np.ndarray:
    """The 20 vertices of a regular dodecahedron: (+-1,+-1,+-1) and the cyclic permutations of (0, +-1/phi, +-phi)."""
    gr = 0.5 * (1.0 + np.sqrt(5.0))
    v = [[sx, sy, sz] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)]
    for a in (-1, 1):
        for b in (-1, 1):
            v += [[0, a / gr, b * gr], [a / gr, b * gr, 0], [a * gr, 0, b / gr]]
    v = np.array(v, dtype=np.float64)
    return v * (circumradius / np.sqrt(3.0))


def truncated_octahedron_vertices(circumradius: float = 0.5) -> np.ndarray:
    """The 24 vertices of a truncated octahedron: all permutations of (0, +-1, +-2)."""
    import itertools
    v = set()
    for perm in itertools.permutations((0, 1, 2)):
        for s1 in (-1, 1):
            for s2 in (-1, 1):
                c = [0.0, 0.0, 0.0]
                c[perm[1]] = s1 * 1.0
                c[perm[2]] = s2 * 2.0
                v.add(tuple(c))
    v = np.array(sorted(v), dtype=np.float64)
    return v * (circumradius / np.sqrt(5.0))


def polyhedra(verts: np.ndarray, n_lat: int = 6, spacing: float = 1.05, seed: int = 1, max_tilt: float = 0.2,
              name: str = "polyhedra") -> Workload:
    """Generic convex polyhedra (the paper's other benchmark shapes) on a simple-cubic lattice: spacing above the
    circumsphere diameter, so any orientation is overlap-free; small random tilts.  Parity cases for the GJK kernel with more
    vertices than a cube; not one of the BASELINE.json configs."""
    N = n_lat ** 3
    dmax = 2.0 * float(np.max(np.linalg.norm(verts, axis=1)))
    assert spacing > dmax
    pos4 = _lattice(3, n_lat, spacing)
    rng = _rng(seed, 404)
    z = 2.0 * rng.random(N) - 1.0
    phi = 2.0 * np.pi * rng.random(N)
    rho = np.sqrt(1.0 - z * z)
    axis = np.stack([rho * np.cos(phi), rho * np.sin(phi), z], axis=1)
    ang = max_tilt * rng.random(N)
    q = np.concatenate([np.cos(0.5 * ang)[:, None], np.sin(0.5 * ang)[:, None] * axis], axis=1)
    L = n_lat * spacing
    return Workload(name=name, dim=3, N=N, L=(L, L, L), kind=KIND_POLYHEDRON, diameter=0.0, verts=verts, d=0.1, a=0.2,
                    n_select=4, sweeps=100, pos4=pos4, quat4=q.astype(np.float32), warmup_sweeps=50,
                    extra={"seed": seed})


def fcc_spheres(m: int = 32, phi: float = 0.60, d: float = 0.06, name: str = "fcc_spheres") -> Workload:
    """4 m^3 hard spheres of diameter 1 on a face-centred cubic lattice at volume fraction `phi`: the paper's sphere validation
    state is 131 072 = 4 x 32^3 spheres at phi = 0.60, started "on the known self-assembled FCC" lattice."""
    A = (4.0 * (np.pi / 6.0) / phi) ** (1.0 / 3.0)
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    idx = np.stack(np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij"), axis=-1).reshape(-1, 3)
    p = (idx[:, None, :] + basis[None, :, :] + 0.25).reshape(-1, 3) * A - 0.5 * m * A
    N = p.shape[0]
    pos4 = np.zeros((N, 4), dtype=np.float32)
    pos4[:, :3] = p.astype(np.float32)
    L = m * A
    return Workload(name=name, dim=3, N=N, L=(L, L, L), kind=KIND_DISK, diameter=1.0, verts=None, d=d, a=0.0, n_select=4,
                    sweeps=100, pos4=pos4, quat4=_identity_quats(N), warmup_sweeps=50, notes=f"FCC crystal start at phi = {phi}",
                    extra={"phi": phi})


def bcc_polyhedra(verts: np.ndarray, m: int = 20, phi: float = 0.7, volume: float = None, name: str = "bcc_polyhedra",
                  d: float = 0.04, a: float = 0.05) -> Workload:
    """2 m^3 identical convex polyhedra on a body-centred cubic lattice at volume fraction `phi`, all in the body orientation:
    the paper's third validation state is 16 000 = 2 x 20^3 truncated octahedra at phi = 0.7 on "the known self-assembled ...
    BCC" lattice; truncated octahedra with the vertices of `truncated_octahedron_vertices` tile space on it at phi = 1."""
    if volume is None:
        from scipy.spatial import ConvexHull
        volume = float(ConvexHull(np.asarray(verts, dtype=np.float64)).volume)
    A = (2.0 * volume / phi) ** (1.0 / 3.0)
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.5]])
    idx = np.stack(np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij"), axis=-1).reshape(-1, 3)
    p = (idx[:, None, :] + basis[None, :, :] + 0.25).reshape(-1, 3) * A - 0.5 * m * A
    N = p.shape[0]
    pos4 = np.zeros((N, 4), dtype=np.float32)
    pos4[:, :3] = p.astype(np.float32)
    L = m * A
    return Workload(name=name, dim=3, N=N, L=(L, L, L), kind=KIND_POLYHEDRON, diameter=0.0, verts=np.asarray(verts, dtype=np.float64),
                    d=d, a=a, n_select=4, sweeps=100, pos4=pos4, quat4=_identity_quats(N), warmup_sweeps=50,
                    notes=f"BCC crystal start at phi = {phi}", extra={"phi": phi, "volume": volume})


def config(k: int, seed: int = 1) -> Workload:
    """BASELINE.json configs[k], k = 0..4."""
    if k == 0:
        return disks(64, seed)
    if k == 1:
        return pentagons(64, seed)
    if k == 2:
        return pentagons(1024, seed)
    if k == 3:
        return cubes(32, seed)
    if k == 4:
        return pentagons(4096, seed)
    raise ValueError("configs are numbered 0..4")


def fcc_polyhedra(verts: np.ndarray, m: int = 4, phi: float = 0.5, volume: float = None, max_tilt: float = 0.03, seed: int = 1,
                  name: str = "fcc_polyhedra", d: float = 0.05, a: float = 0.1) -> Workload:
    """4 m^3 identical convex polyhedra on a face-centred cubic lattice at volume fraction `phi`, all in the body orientation
    up to a random tilt of at most `max_tilt` rad: a dense, overlap-free start that needs no simulation (for dodecahedra of
    circumradius 0.5 at phi = 0.5 the nearest-neighbour distance is 0.995 against an extent of 0.913 along that direction).
    Stands in for the paper's equilibrated phi = 0.5 dodecahedron state in parity tests; the caller checks
    count_overlaps == 0.  `volume`: particle volume (scipy ConvexHull if None)."""
    if volume is None:
        from scipy.spatial import ConvexHull
        volume = float(ConvexHull(np.asarray(verts, dtype=np.float64)).volume)
    A = (4.0 * volume / phi) ** (1.0 / 3.0)                       # cubic cell edge: 4 particles per cell
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    idx = np.stack(np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij"), axis=-1).reshape(-1, 3)
    p = (idx[:, None, :] + basis[None, :, :] + 0.25).reshape(-1, 3) * A - 0.5 * m * A
    N = p.shape[0]
    pos4 = np.zeros((N, 4), dtype=np.float32)
    pos4[:, :3] = p.astype(np.float32)
    rng = _rng(seed, 505)
    z = 2.0 * rng.random(N) - 1.0
    ang_phi = 2.0 * np.pi * rng.random(N)
    rho = np.sqrt(1.0 - z * z)
    axis = np.stack([rho * np.cos(ang_phi), rho * np.sin(ang_phi), z], axis=1)
    ang = max_tilt * rng.random(N)
    q = np.concatenate([np.cos(0.5 * ang)[:, None], np.sin(0.5 * ang)[:, None] * axis], axis=1)
    L = m * A
    return Workload(name=name, dim=3, N=N, L=(L, L, L), kind=KIND_POLYHEDRON, diameter=0.0, verts=np.asarray(verts, dtype=np.float64),
                    d=d, a=a, n_select=4, sweeps=100, pos4=pos4, quat4=q.astype(np.float32), warmup_sweeps=50,
                    notes=f"FCC crystal start at phi = {phi}", extra={"seed": seed, "phi": phi})
