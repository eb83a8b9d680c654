"""Pins of the O9 pressure analysis (oracle/pressure.py + orc_shape_touch_scale / orc_scale_histogram), none of which
re-use the estimator's own formula:
  - the touch scale lambda* is the root of the independently pinned SAT margin (tests/test_oracle_margins.py);
  - closed-form contacts (pentagon vertex-edge 0.904508, edge-edge 0.809017; cube face 1, vertex sqrt 3);
  - the histogram equals a brute-force O(N^2) count of pairs that overlap after compressing separations;
  - hard-disk equation of state: dilute virial series 1 + B2 rho + B3 rho^2 (B2 = pi sigma^2/2, B3 = 0.7820 B2^2)
    and, at config 0's density, the Henderson / Santos-Lopez de Haro-Yuste fluid equations of state
    (P* = beta P sigma^2 = 6.96 .. 7.06).
"""
import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from oracle import pressure as pr
from paper_1509_04692_b200 import workloads as wl


def _rand_quat(rng, dim):
    if dim == 2:
        t = rng.uniform(0, 2 * np.pi)
        return np.array([np.cos(t / 2), 0, 0, np.sin(t / 2)])
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


@pytest.mark.parametrize("dim,kind,verts", [(2, 1, wl.regular_polygon(5, 0.5)), (3, 2, wl.cube_vertices(1.0)),
                                            (2, 1, np.array([[0.5, 0.0], [0.1, 0.4], [-0.4, 0.2], [-0.3, -0.3], [0.2, -0.35]]))])
def test_touch_scale_is_the_root_of_the_margin(dim, kind, verts):
    s = ho.Shape(dim, kind, verts=verts)
    rng = np.random.default_rng(3)
    for _ in range(400):
        r = rng.normal(size=dim); r *= rng.uniform(0.6, 1.6) / np.linalg.norm(r)
        qa, qb = _rand_quat(rng, dim), _rand_quat(rng, dim)
        lam = s.touch_scale(r, qa, qb)
        assert abs(s.margin(lam * r, qa, qb)) < 1e-12
        assert s.margin((lam - 1e-6) * r, qa, qb) < 0 < s.margin((lam + 1e-6) * r, qa, qb)


def test_touch_scale_closed_forms():
    q0 = np.array([1.0, 0, 0, 0])
    pent = ho.Shape(2, 1, verts=wl.regular_polygon(5, 0.5))
    # A's vertex 0 points along +x; B unrotated presents the edge opposite its vertex 0: vertex-edge contact
    assert pent.touch_scale([2.0, 0], q0, q0) * 2.0 == pytest.approx(0.5 + 0.5 * np.cos(np.pi / 5), abs=1e-12)
    # B turned by pi: vertex to vertex at 1.0
    qpi = np.array([0.0, 0, 0, 1.0])
    assert pent.touch_scale([3.0, 0], q0, qpi) * 3.0 == pytest.approx(1.0, abs=1e-12)
    # A turned by pi (edge toward +x), B unrotated (edge toward -x): edge to edge at 2 R cos 36
    assert pent.touch_scale([1.5, 0], qpi, q0) * 1.5 == pytest.approx(2 * 0.5 * np.cos(np.pi / 5), abs=1e-12)
    cube = ho.Shape(3, 2, verts=wl.cube_vertices(1.0))
    assert cube.touch_scale([0, 2.0, 0], q0, q0) * 2.0 == pytest.approx(1.0, abs=1e-12)
    d = np.array([1.0, 1.0, 1.0]) / np.sqrt(3.0)
    assert cube.touch_scale(2.5 * d, q0, q0) * 2.5 == pytest.approx(np.sqrt(3.0), abs=1e-12)
    disk = ho.Shape(2, 0, diameter=1.0)
    assert disk.touch_scale([0.6, 0.8], q0, q0) == pytest.approx(1.0, abs=1e-15)


def _melted(w, sweeps, seed=1):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    o.sweeps(sweeps)
    return o


@pytest.mark.parametrize("w", [wl.pentagons(12), wl.disks(12), wl.cubes(12)], ids=["pentagons", "disks", "cubes"])
def test_histogram_equals_bruteforce_compression_count(w):
    """Pairs with touch scale < s are exactly the pairs that overlap once every separation is scaled by (1 - s)."""
    o = _melted(w, 30 if w.dim == 2 else 6)
    s_max, nb = 0.02, 8
    h = o.scale_histogram(s_max, nb)
    pos, quat = o.get_state()
    shape = ho.Shape(w.dim, w.kind, diameter=w.diameter, verts=w.verts)
    L = np.array(w.L, dtype=np.float32).astype(np.float64)
    x = pos[:, : w.dim].astype(np.float64)
    cum = np.zeros(nb + 1, dtype=np.int64)
    for i in range(w.N):
        r = x[i + 1:] - x[i]
        r -= L * np.round(r / L)
        near = np.nonzero(np.einsum("ij,ij->i", r, r) < (1.05 * shape.dmax) ** 2)[0]
        for jj in near:
            j = i + 1 + jj
            for b in range(nb + 1):
                sc = s_max * b / nb
                if shape.margin((1.0 - sc) * r[jj], quat[i].astype(np.float64), quat[j].astype(np.float64)) < 0.0:
                    cum[b:] += 1
                    break
    assert cum[0] == 0                       # the state itself is overlap-free
    assert h.sum() == cum[nb] and np.array_equal(np.cumsum(h), cum[1:])
    assert h.sum() > (20 if w.dim == 2 else 5)


def _disk_Z(n_lat, spacing, d, sweeps, every, seed=1):
    w = wl.disks(n_lat, spacing=spacing)
    o = ho.Oracle(2, w.L, w.kind, w.N, seed, diameter=1.0)
    o.set_moves(d, 0.0, 4)
    o.set_state(w.pos4, w.quat4)
    o.sweeps(sweeps // 10)
    hist, ns = np.zeros(pr.NBINS), 0
    for _ in range((sweeps - sweeps // 10) // every):
        o.sweeps(every)
        hist += o.scale_histogram(pr.S_MAX, pr.NBINS)
        ns += 1
    assert o.count_overlaps_cells() == 0
    rho = w.N / (w.L[0] * w.L[1])
    return pr.compressibility(hist, ns, w.N, 2), rho


def test_disk_pressure_dilute_virial():
    """rho sigma^2 = 0.0816: beta P/rho = 1 + B2 rho + B3 rho^2 + B4 rho^3 = 1.1389 (B3/B2^2 = 0.7820, B4/B2^3 = 0.5322)."""
    Z, rho = _disk_Z(32, 3.5, 0.45, 3000, 2)
    b2 = 0.5 * np.pi * rho
    expect = 1 + b2 + 0.7820 * b2 ** 2 + 0.5322 * b2 ** 3
    assert rho == pytest.approx(1 / 3.5 ** 2)
    assert Z - 1 == pytest.approx(expect - 1, rel=0.06), (Z, expect)      # ~1.7e4 contact pairs: 2 sigma ~ 3 %


def test_disk_pressure_config0_within_fluid_equations_of_state():
    """Config 0 (phi = 0.6491): Henderson Z = (1 + phi^2/8)/(1 - phi)^2 = 8.55, SHY Z = 8.42 -> P* = Z rho sigma^2."""
    Z, rho = _disk_Z(64, 1.1, 0.15, 1000, 10)
    phi = rho * np.pi / 4
    henderson = (1 + phi ** 2 / 8) / (1 - phi) ** 2
    assert henderson == pytest.approx(8.55, abs=0.01)
    p_star = Z * rho
    assert 6.96 * 0.98 < p_star < 7.06 * 1.02, (Z, p_star)


def test_contact_density_fit_recovers_a_known_quadratic():
    rng = np.random.default_rng(0)
    nb, ns, ds = pr.NBINS, 500, pr.S_MAX / pr.NBINS
    x = (np.arange(nb) + 0.5) * ds
    dens = 6000.0 * (1 + 30 * x + 200 * x * x)
    counts = rng.poisson(dens * ds * ns)
    assert pr.contact_density(counts, ns) == pytest.approx(6000.0, rel=0.02)
