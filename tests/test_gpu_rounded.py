"""GPU parity for rounded shapes -- spheropolygons and convex spheropolyhedra -- against the oracle
(oracle margin = distance of the cores - 2 sweep radius, pinned in tests/test_oracle_rounded.py).  Same bars as
tests/test_gpu_parity.py: grid and cell list bit-exact, every trial of the first sweeps decided as the oracle decides it except
inside the 1e-5 window (counted), positions bit-exact, quaternions within 1e-5, counters equal, zero overlaps; the strict fp64
validator counts planted overlaps as the oracle's O(N^2) brute force does."""
import math

import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu

MARGIN_TOL = 1e-5


def gpu(w, seed=1):
    from paper_1509_04692_b200 import binding as hb
    return hb.from_workload(w, seed=seed)


def orc(w, seed=1, threads=1):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts, sweep_radius=w.sweep_radius)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    if threads > 1:
        o.set_threads(threads)
    return o


CASES = {
    # warp-per-cell pass (small 2-D systems), runtime-vertex-count kernels
    "rounded_pentagons_24": lambda: wl.rounded_polygons(24),
    "rounded_squares_24_dense": lambda: wl.rounded_polygons(24, nv=4, circumradius=0.3, sweep_radius=0.15, spacing=0.92, d=0.05, a=0.2),
    "rounded_triangles_20": lambda: wl.rounded_polygons(20, nv=3, circumradius=0.4, sweep_radius=0.05, spacing=0.95),
    # tile pass (more than 148 x 48 active cells per colour)
    "rounded_pentagons_192": lambda: wl.rounded_polygons(192),
    # 3-D warp-per-cell pass: fp32 XenoCollide with the rounded support function, fp64 GJK on the cores when unsure
    "rounded_cubes_7": lambda: wl.cubes(7, edge=0.7, sweep_radius=0.15, name="rounded_cubes_7"),
    "rounded_cubes_6_big_radius": lambda: wl.cubes(6, edge=0.4, sweep_radius=0.3, name="rounded_cubes_6_big_radius", d=0.15, a=0.3),
    "rounded_dodecahedra_5": lambda: rounded(wl.polyhedra(wl.dodecahedron_vertices(0.4), 5, 1.04, name="rounded_dodecahedra_5"), 0.1),
}


def rounded(w, rho):
    w.sweep_radius = rho
    return w


def lockstep(w, n_sweeps, threads=1):
    g, o = gpu(w), orc(w, threads=threads)
    assert g.d_max == pytest.approx(ho.Shape(w.dim, w.kind, verts=w.verts, sweep_radius=w.sweep_radius).dmax, abs=1e-15)
    assert np.array_equal(g.n, o.n) and g.C == o.C
    assert g.count_overlaps() == 0
    g.enable_trace(True)
    stats = {"marginal": 0, "compared": 0}
    for s in range(n_sweeps):
        cid, cst, mem, shift, perm = g.cell_list(s)
        oshift, operm = o.sweep_header(s)
        ocid, ocst, omem = o.cell_list(oshift)
        assert np.array_equal(cid, ocid) and np.array_equal(cst, ocst) and np.array_equal(mem, omem)
        g.sweep(1)
        f = o.sweep(follow=g.read_trace(), follow_tol=MARGIN_TOL)["follow"]
        assert f["hard_mismatch"] == 0, (s, f)
        stats["marginal"] += f["marginal"]; stats["compared"] += f["compared"]
        gp, gq = g.get_state(); op, oq = o.get_state()
        assert np.array_equal(gp, op), f"sweep {s}: positions differ"
        assert np.max(np.abs(gq.astype(np.float64) - oq.astype(np.float64))) < 1e-5
        o.set_state(op, gq)
    gc, oc = g.counters(), o.counters()
    for k in ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials", "sweeps"):
        assert gc[k] == oc[k], (k, gc, oc)
    assert g.count_overlaps() == 0
    stats.update(trials=gc["trials"], rej=gc["trans_rej_overlap"] + gc["rot_rej_overlap"], acc=gc["trans_acc"] + gc["rot_acc"])
    return stats, g, o


@pytest.mark.parametrize("name,n", [("rounded_pentagons_24", 10), ("rounded_squares_24_dense", 10), ("rounded_triangles_20", 10),
                                    ("rounded_cubes_7", 8), ("rounded_cubes_6_big_radius", 8), ("rounded_dodecahedra_5", 5)])
def test_rounded_shapes_lockstep_with_oracle(name, n):
    w = CASES[name]()
    stats, g, o = lockstep(w, n)
    assert stats["compared"] == n * g.C * w.n_select
    assert stats["marginal"] <= max(3, 2e-3 * stats["trials"]), stats
    assert stats["rej"] > 0.02 * stats["trials"] and stats["acc"] > 0.1 * stats["trials"], stats   # both outcomes occur
    assert o.count_overlaps_bruteforce() == 0
    print(name, g.describe_pass(), stats,
          "fp64 re-runs", g.get_stat("gjk_f64_reruns") if w.dim == 3 else "-")


def test_rounded_pentagons_tile_pass_lockstep():
    """36 864 rounded pentagons: the 2-D tile pass (runtime-vertex-count instantiation) and its dataflow launch."""
    w = CASES["rounded_pentagons_192"]()
    stats, g, o = lockstep(w, 4, threads=8)
    assert "tile2d" in g.describe_pass()
    assert stats["marginal"] <= max(3, 2e-3 * stats["trials"]), stats
    print("rounded_pentagons_192", g.describe_pass(), stats)


@pytest.mark.parametrize("name", ["rounded_pentagons_24", "rounded_cubes_7"])
def test_rounded_colour_pass_variants_agree_bit_for_bit(name):
    """Staged kernels, their overflow fallbacks and the per-thread path run one narrow-phase definition."""
    w = CASES[name]()
    ref = None
    variants = [{}, {"path": 1}, {"tile_cap": 0}]
    if w.dim == 2:
        variants += [{"path": 2}, {"path": 2, "flow": 1}, {"path": 3}]
    for opts in variants:
        g = gpu(w)
        for k, v in opts.items():
            g.set_option(k, v)
        g.sweep(6)
        state = g.get_state() + (g.counters(),)
        if ref is None:
            ref = state
        else:
            assert np.array_equal(ref[0], state[0]) and np.array_equal(ref[1], state[1]) and ref[2] == state[2], opts


def test_rounded_near_contact_crystal_takes_the_fp64_rerun():
    """Rounded cubes (edge 0.7, radius 0.15: width 1.0) in a crystal with face-to-face gaps of 6e-4 and moves of 3e-4: nearly
    every narrow-phase test is a near-contact pair of nearly parallel faces, the case the fp32 run hands to the fp64 GJK on
    the cores (threshold 2 rho + eps_g)."""
    gap = 6e-4
    w = wl.cubes(7, spacing=1.0 + gap, max_tilt=gap / 4, d=gap / 2, a=gap / 2, edge=0.7, sweep_radius=0.15, name="rounded_cubes_near_contact")
    stats, g, o = lockstep(w, 6)
    reruns = g.get_stat("gjk_f64_reruns")
    print("rounded near-contact crystal:", stats, "fp64 re-runs", reruns)
    assert stats["rej"] > 0.05 * stats["trials"] and stats["acc"] > 0.05 * stats["trials"]
    assert stats["marginal"] <= 0.02 * stats["trials"]
    assert reruns > 0


@pytest.mark.parametrize("dim", [2, 3])
def test_validator_counts_planted_rounded_overlaps_like_the_oracle(dim):
    """Pairs whose cores are disjoint but closer than 2 rho overlap; the sharp shapes at the same poses would not."""
    from paper_1509_04692_b200 import binding as hb
    w = wl.rounded_polygons(16) if dim == 2 else wl.cubes(6, edge=0.7, sweep_radius=0.15)
    rng = np.random.default_rng(3)
    pos, quat = w.pos4.copy(), w.quat4.copy()
    spacing = w.L[0] / round(w.N ** (1.0 / dim))
    dmax = 2 * (np.max(np.linalg.norm(w.verts, axis=1)) + w.sweep_radius)
    planted = rng.choice(w.N, size=12, replace=False)
    for i in planted:
        j = (i + 1) if (i + 1) % round(w.N ** (1.0 / dim)) else i - 1     # lattice neighbour along x
        shift = (spacing - rng.uniform(0.55, 0.95) * dmax) * np.sign(pos[j, 0] - pos[i, 0])
        pos[i, 0] += shift
    g = gpu(w); g.bind(pos, quat)
    o = orc(w); o.set_state(pos, quat)
    expect = o.count_overlaps_bruteforce()
    assert expect > 0
    assert g.count_overlaps() == expect
    # the allocation-free entry point runs the same validator
    import torch
    out = torch.full((1,), -7, dtype=torch.int64, device=g.device)
    torch.cuda.synchronize()
    g.count_overlaps_noalloc(torch.from_numpy(pos).to(g.device), torch.from_numpy(quat).to(g.device), out)
    g.stream.synchronize()
    assert int(out.item()) == expect
    sharp = hb.Hpmc(w.dim, w.L, w.kind, w.N, 1, verts=w.verts)
    sharp.bind(pos, quat)
    assert sharp.count_overlaps() < expect


def test_negative_sweep_radius_is_rejected():
    from paper_1509_04692_b200 import binding as hb
    with pytest.raises(hb.HpmcError):
        hb.Hpmc(2, (16.0, 16.0), wl.KIND_POLYGON, 16, 1, verts=wl.regular_polygon(5, 0.35), sweep_radius=-0.1)
    with pytest.raises(hb.HpmcError):
        hb.Hpmc(2, (16.0, 16.0), wl.KIND_POLYGON, 16, 1, verts=wl.regular_polygon(5, 0.35), sweep_radius=float("nan"))
