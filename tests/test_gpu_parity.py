"""GPU parity tests proper: the CUDA path (through the C-ABI binding) against the oracle, element by element,
on the same seeded inputs.  Bars (BASELINE.json north_star): cell assignment and indexing bit-exact; the first
10 sweeps' accept/reject decisions identical except on trials whose contact margin is within 1e-5 of the
threshold (counted); positions within 1e-5 where no decision differed (here: bit-exact); zero overlaps."""
import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu

MARGIN_TOL = 1e-5


def gpu(w, seed=1):
    from paper_1509_04692_b200 import binding as hb
    return hb.from_workload(w, seed=seed)


def orc(w, seed=1):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    return o


CASES = {
    "disks_24": lambda: wl.disks(24),
    "pentagons_24": lambda: wl.pentagons(24),
    "cubes_7": lambda: wl.cubes(7),
    "k0_disks": lambda: wl.config(0),
    "k1_pentagons": lambda: wl.config(1),
    "cubes_12": lambda: wl.cubes(12),
    "spheres_8": lambda: spheres(8),
    "dodecahedra_6": lambda: wl.polyhedra(wl.dodecahedron_vertices(0.5), 6, 1.04, name="dodecahedra_6"),
    "trunc_octahedra_6": lambda: wl.polyhedra(wl.truncated_octahedron_vertices(0.5), 6, 1.04, name="trunc_octahedra_6"),
}


def spheres(n_lat):
    """3-D hard spheres (KIND_DISK in a 3-D box) on the cube lattice of wl.cubes: diameter 1, spacing 1.25."""
    base = wl.cubes(n_lat)
    q = np.zeros((base.N, 4), np.float32); q[:, 0] = 1
    return wl.Workload(name=f"spheres_{n_lat}", dim=3, N=base.N, L=base.L, kind=wl.KIND_DISK, diameter=1.0, verts=None, d=0.2,
                       a=0.0, n_select=4, sweeps=1, pos4=base.pos4, quat4=q)


def test_grid_matches_oracle():
    for name in ("k0_disks", "k1_pentagons", "cubes_12"):
        w = CASES[name]()
        g, o = gpu(w), orc(w)
        assert np.array_equal(g.n, o.n) and g.C == o.C
        assert np.array_equal(g.inv_w[: w.dim], o.inv_w[: w.dim]) and np.array_equal(g.L_f[: w.dim], o.L_f[: w.dim])
        assert g.d_max == pytest.approx(ho.Shape(w.dim, w.kind, diameter=w.diameter, verts=w.verts).dmax, abs=1e-15)


@pytest.mark.parametrize("name", ["disks_24", "pentagons_24", "cubes_7", "k1_pentagons"])
def test_header_and_cell_list_bit_exact(name):
    w = CASES[name]()
    g, o = gpu(w), orc(w)
    for t in (0, 1, 2, 17, 2 ** 32 - 1, 2 ** 32 + 5, 2 ** 40 + 123):
        cid, cst, mem, shift, perm = g.cell_list(t)
        oshift, operm = o.sweep_header(t)
        assert np.array_equal(shift[: w.dim], oshift[: w.dim]) and np.array_equal(perm, operm)   # Philox + R10 + R12
        ocid, ocst, omem = o.cell_list(oshift)
        assert np.array_equal(cid, ocid) and np.array_equal(cst, ocst) and np.array_equal(mem, omem)
    # after some sweeps (off-lattice state, cell-sorted source order inside the library)
    g.sweep(3)
    pos, quat = g.get_state()
    o.set_state(pos, quat)
    for t in (3, 4, 99):
        cid, cst, mem, shift, perm = g.cell_list(t)
        oshift, operm = o.sweep_header(t)
        ocid, ocst, omem = o.cell_list(oshift)
        assert np.array_equal(shift[: w.dim], oshift[: w.dim]) and np.array_equal(perm, operm)
        assert np.array_equal(cid, ocid) and np.array_equal(cst, ocst) and np.array_equal(mem, omem)
    p2, q2 = g.get_state()   # building lists must not change the state
    assert np.array_equal(p2, pos) and np.array_equal(q2, quat)


def lockstep(w, n_sweeps, seed=1):
    """O8: run the GPU one sweep at a time with the trace on; the oracle follows."""
    g, o = gpu(w, seed), orc(w, seed)
    g.enable_trace(True)
    stats = {"marginal": 0, "hard": 0, "compared": 0, "trials": 0}
    for s in range(n_sweeps):
        g.sweep(1)
        tr = g.read_trace()
        res = o.sweep(follow=tr, follow_tol=MARGIN_TOL)
        f = res["follow"]
        stats["marginal"] += f["marginal"]; stats["hard"] += f["hard_mismatch"]; stats["compared"] += f["compared"]
        assert f["hard_mismatch"] == 0, (s, f)
        gp, gq = g.get_state()
        op, oq = o.get_state()
        assert np.array_equal(gp, op), f"sweep {s}: positions differ"          # single-fmaf translations: bit-exact
        assert np.max(np.abs(gq.astype(np.float64) - oq.astype(np.float64))) < 1e-5
        # the oracle adopts the GPU's quaternions so that ulp-level differences cannot accumulate (O8)
        o.set_state(op, gq)
    gc, oc = g.counters(), o.counters()
    stats["trials"] = gc["trials"]
    for k in ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials", "sweeps"):
        assert gc[k] == oc[k], (k, gc, oc)
    assert gc["sweep_counter"] == n_sweeps
    assert g.count_overlaps() == 0
    return stats, g, o


@pytest.mark.parametrize("name,n", [("disks_24", 10), ("pentagons_24", 10), ("cubes_7", 10), ("spheres_8", 10),
                                    ("k0_disks", 10), ("k1_pentagons", 10), ("cubes_12", 4),
                                    ("dodecahedra_6", 6), ("trunc_octahedra_6", 6)])
def test_first_sweeps_lockstep_with_oracle(name, n):
    w = CASES[name]()
    stats, g, o = lockstep(w, n)
    assert stats["compared"] == n * g.C * w.n_select
    # P11: marginal trials should be of order 1e-4 of all trials or fewer
    assert stats["marginal"] <= max(3, 2e-3 * stats["trials"]), stats
    if w.N <= 2000:
        assert o.count_overlaps_bruteforce() == 0
    print(name, stats)


@pytest.mark.parametrize("name", ["disks_24", "pentagons_24", "cubes_7"])
def test_multi_sweep_call_equals_single_sweep_calls(name):
    w = CASES[name]()
    a, b = gpu(w), gpu(w)
    a.sweep(6)
    for _ in range(6):
        b.sweep(1)
    pa, qa = a.get_state(); pb, qb = b.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)
    assert a.counters() == b.counters()


@pytest.mark.parametrize("name", ["disks_24", "pentagons_24", "k1_pentagons", "cubes_7", "spheres_8"])
def test_colour_pass_variants_agree_bit_for_bit(name):
    """The staged kernels (2-D tile, 3-D warp-per-cell), their overflow fallbacks (tile_cap=0 everywhere, a small
    tile_cap on some tiles/cells) and the per-thread path make identical trajectories."""
    w = CASES[name]()
    ref = None
    some = 40 if w.dim == 2 else (84 if w.kind == wl.KIND_POLYHEDRON else 50)   # a capacity only some tiles/cells exceed
    shapes = [{"tile_shape": k} for k in (1, 2, 3)] if w.dim == 2 else []   # every 2-D tile shape
    shapes += [{"path": 2, "flow": 1}, {"tile_shape": 1, "flow": 1}, {"tile_shape": 2, "flow": 1},
               {"path": 2, "flow": 1, "tile_cap": some}] if w.dim == 2 else []
    warp = [{"path": 3}, {"path": 3, "tile_cap": 6}] if w.dim == 2 else []        # 2-D warp-per-cell pass and its fallback
    warp += [{"path": 4}] if w.dim == 2 else []                                   # whole sweeps in one thread-block cluster
    warp += [{"path": 5}, {"path": 5, "tile_cap": 6}] if w.dim == 2 else []       # speculative warp-per-cell pass and its fallback
    builds = [{"small_build": 0}, {"small_build": 0, "path": 2}]                   # the multi-launch cell-list build
    for opts in [{"path": 2}, {"path": 2, "tile_cap": 0}, {"path": 1}, {"path": 2, "tile_cap": some}] + shapes + warp + builds:
        g = gpu(w)
        for k, v in opts.items():
            g.set_option(k, v)
        g.enable_trace(True)
        g.sweep(5)
        out = (g.get_state(), g.counters(), g.read_trace().copy())
        if ref is None:
            ref = out
        else:
            assert np.array_equal(out[0][0], ref[0][0]) and np.array_equal(out[0][1], ref[0][1]), opts
            assert out[1] == ref[1] and np.array_equal(out[2], ref[2]), opts


def test_restart_from_state_and_sweep_counter():
    w = wl.pentagons(24)
    a = gpu(w)
    a.sweep(4)
    p4, q4 = a.get_state()
    a.sweep(3)
    p7, q7 = a.get_state()
    w2 = wl.pentagons(24)
    w2.pos4, w2.quat4 = p4.copy(), q4.copy()
    b = gpu(w2)
    b.set_sweep_counter(4)
    b.sweep(3)
    pb, qb = b.get_state()
    assert np.array_equal(p7, pb) and np.array_equal(q7, qb)


@pytest.mark.parametrize("name", ["disks_24", "pentagons_24", "cubes_7"])
def test_count_overlaps_matches_bruteforce_on_planted_overlaps(name):
    w = CASES[name]()
    rng = np.random.default_rng(5)
    pos, quat = w.pos4.copy(), w.quat4.copy()
    L = np.array(w.L)
    for i in rng.choice(w.N, size=12, replace=False):      # push a dozen particles into their neighbours
        pos[i, : w.dim] += rng.uniform(-0.45, 0.45, size=w.dim).astype(np.float32)
    pos[:, : w.dim] = ((pos[:, : w.dim] + L / 2) % L - L / 2).astype(np.float32)
    w.pos4, w.quat4 = pos, quat
    g, o = gpu(w), orc(w)
    n = o.count_overlaps_bruteforce()
    assert n > 0 and g.count_overlaps() == n


def test_edge_cases_small_and_sparse():
    # one particle, many empty cells, minimal 4x4 grid, large n_select
    pos = np.zeros((1, 4), np.float32); quat = np.zeros((1, 4), np.float32); quat[:, 0] = 1
    w = wl.Workload(name="one", dim=2, N=1, L=(4.2, 4.2), kind=wl.KIND_DISK, diameter=1.0, verts=None, d=0.3, a=0.0,
                    n_select=37, sweeps=1, pos4=pos, quat4=quat)
    stats, g, o = lockstep(w, 5)
    assert list(g.n[:2]) == [4, 4] and stats["trials"] == 5 * 37
    # two pentagons in a box where they keep meeting across the periodic seam
    pos = np.zeros((2, 4), np.float32); pos[0, :2] = [-2.0, 0.1]; pos[1, :2] = [2.0, -0.1]
    quat = np.zeros((2, 4), np.float32); quat[:, 0] = 1
    w = wl.Workload(name="two", dim=2, N=2, L=(5.0, 5.0), kind=wl.KIND_POLYGON, diameter=0.0, verts=wl.regular_polygon(5, 0.5),
                    d=0.4, a=0.5, n_select=8, sweeps=1, pos4=pos, quat4=quat)
    stats, g, o = lockstep(w, 10)
    c = g.counters()
    assert c["trans_rej_overlap"] + c["rot_rej_overlap"] > 0      # they do collide through the seam
    # irregular convex polygon with a vertex count that has no unrolled kernel (runtime-NV path)
    rng = np.random.default_rng(1)
    ang = np.sort(rng.uniform(0, 2 * np.pi, 7)); ang[0] = 0.1
    verts = 0.5 * np.stack([np.cos(ang), np.sin(ang)], axis=1)
    base = wl.disks(12, spacing=1.25)
    w = wl.Workload(name="hept", dim=2, N=base.N, L=base.L, kind=wl.KIND_POLYGON, diameter=0.0, verts=verts, d=0.12, a=0.3,
                    n_select=4, sweeps=1, pos4=base.pos4, quat4=base.quat4)
    lockstep(w, 6)
    # tetrahedra (generic polyhedron path with 4 vertices)
    tet = 0.45 * np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64)
    base = wl.cubes(6)
    quat = np.zeros((base.N, 4), np.float32); quat[:, 0] = 1
    w = wl.Workload(name="tet", dim=3, N=base.N, L=base.L, kind=wl.KIND_POLYHEDRON, diameter=0.0, verts=tet, d=0.15, a=0.3,
                    n_select=4, sweeps=1, pos4=base.pos4, quat4=quat)
    lockstep(w, 6)


def test_empty_system():
    w = wl.Workload(name="none", dim=2, N=0, L=(8.0, 8.0), kind=wl.KIND_DISK, diameter=1.0, verts=None, d=0.1, a=0.0,
                    n_select=4, sweeps=1, pos4=np.zeros((0, 4), np.float32), quat4=np.zeros((0, 4), np.float32))
    g = gpu(w)
    g.sweep(3)
    assert g.counters()["trials"] == 0 and g.count_overlaps() == 0


def test_sweep_host_round_trip():
    import torch
    w = wl.pentagons(24)
    a = gpu(w)
    a.sweep(5)
    pa, qa = a.get_state()
    b = gpu(w)
    hp = torch.from_numpy(w.pos4.copy()).pin_memory(); hq = torch.from_numpy(w.quat4.copy()).pin_memory()
    op = torch.empty_like(hp).pin_memory(); oq = torch.empty_like(hq).pin_memory()
    c = b.sweep_host(hp, hq, 5, op, oq)
    assert np.array_equal(op.numpy(), pa) and np.array_equal(oq.numpy(), qa)
    assert c["trials"] == a.counters()["trials"]


def _lattice_workload(dim, n, spacing, kind, verts=None, diameter=0.0, d=0.1, a=0.2, n_select=4, seed=3):
    """Particles on an n[0] x n[1] (x n[2]) lattice in a box with DIFFERENT edges per axis, random orientations."""
    idx = np.stack(np.meshgrid(*[np.arange(k) for k in n], indexing="ij"), axis=-1).reshape(-1, dim)
    L = np.array([n[k] * spacing[k] for k in range(dim)])
    pos = np.zeros((idx.shape[0], 4), np.float32)
    pos[:, :dim] = ((idx + 0.5) * np.array(spacing) - 0.5 * L).astype(np.float32)
    rng = np.random.default_rng(seed)
    quat = np.zeros((idx.shape[0], 4), np.float32)
    if dim == 2:
        th = rng.uniform(0, 2 * np.pi, idx.shape[0])
        quat[:, 0], quat[:, 3] = np.cos(th / 2), np.sin(th / 2)
    else:
        q = rng.normal(size=(idx.shape[0], 4))
        quat[:] = (q / np.linalg.norm(q, axis=1, keepdims=True)).astype(np.float32)
    return wl.Workload(name="lattice", dim=dim, N=idx.shape[0], L=tuple(L), kind=kind, diameter=diameter, verts=verts, d=d, a=a,
                       n_select=n_select, sweeps=1, pos4=pos, quat4=quat)


@pytest.mark.parametrize("case", ["rect_pentagons_tile", "rect_pentagons_warp", "rect_disks_ns1", "slab_cubes", "slab_spheres_ns9",
                                  "big_step"])
def test_lockstep_on_rectangular_boxes_and_other_move_settings(case):
    """Grids with different cell counts per axis (partial tiles, seams of different lengths), n_select 1 and 9, and a step
    size above half a cell (legal, most trials leave the cell)."""
    pent = wl.regular_polygon(5, 0.5)
    opts = {}
    if case == "rect_pentagons_tile":
        w = _lattice_workload(2, (70, 37), (1.07, 1.12), wl.KIND_POLYGON, verts=pent); opts = {"path": 2}
    elif case == "rect_pentagons_warp":
        w = _lattice_workload(2, (23, 41), (1.1, 1.05), wl.KIND_POLYGON, verts=pent); opts = {"path": 3}
    elif case == "rect_disks_ns1":
        w = _lattice_workload(2, (45, 90), (1.2, 1.08), wl.KIND_DISK, diameter=1.0, d=0.2, n_select=1); opts = {"path": 2, "flow": 1}
    elif case == "slab_cubes":
        w = _lattice_workload(3, (5, 8, 6), (1.8, 1.75, 1.9), wl.KIND_POLYHEDRON, verts=wl.cube_vertices(1.0))
    elif case == "slab_spheres_ns9":
        w = _lattice_workload(3, (9, 6, 12), (1.15, 1.2, 1.1), wl.KIND_DISK, diameter=1.0, d=0.15, n_select=9)
    else:
        w = _lattice_workload(2, (40, 40), (1.15, 1.15), wl.KIND_POLYGON, verts=pent, d=0.8, a=1.5)
    from paper_1509_04692_b200 import binding as hb
    g, o = hb.from_workload(w, seed=5), orc(w, seed=5)
    for k, v in opts.items():
        g.set_option(k, v)
    assert g.n[0] != g.n[1] or case == "big_step"
    g.enable_trace(True)
    marginal = 0
    for s in range(6):
        g.sweep(1)
        f = o.sweep(follow=g.read_trace(), follow_tol=MARGIN_TOL)["follow"]
        assert f["hard_mismatch"] == 0, (case, s, f)
        marginal += f["marginal"]
        gp, gq = g.get_state()
        op, oq = o.get_state()
        assert np.array_equal(gp, op) and np.max(np.abs(gq.astype(np.float64) - oq)) < 1e-5
        o.set_state(op, gq)
    gc, oc = g.counters(), o.counters()
    assert all(gc[k] == oc[k] for k in oc)
    assert g.count_overlaps() == 0 and o.count_overlaps_cells() == 0 and marginal <= 3
    if case == "big_step":
        assert gc["trans_rej_cell"] > 0.4 * (gc["trans_acc"] + gc["trans_rej_overlap"] + gc["trans_rej_cell"])


def test_dataflow_pass_across_the_32_bit_wrap_of_the_sweep_counter():
    """The dataflow launch stamps finished tiles with a value derived from the sweep counter; the stamps must stay distinct
    from sweep to sweep (and from the cleared state) when the low word of the counter wraps."""
    w = wl.pentagons(48)
    out = []
    for flow in (0, 1):
        g = gpu(w)
        g.set_option("path", 2); g.set_option("flow", flow)
        g.sweep(2)
        g.set_sweep_counter(2 ** 32 - 3)
        g.sweep(1); g.sweep(7)                       # plain launches and graph replays: t = 2^32 - 3 .. 2^32 + 4
        assert g.counters()["sweep_counter"] == 2 ** 32 + 5 and g.count_overlaps() == 0
        out.append((g.get_state(), g.counters()))
    assert np.array_equal(out[0][0][0], out[1][0][0]) and np.array_equal(out[0][0][1], out[1][0][1]) and out[0][1] == out[1][1]


@pytest.mark.parametrize("gap,move", [(6e-4, 3e-4), (8e-6, 8e-6)])
def test_near_contact_cubes_match_the_oracle_and_take_the_fp64_rerun(gap, move):
    """A crystal of nearly parallel cubes with face-to-face gaps of `gap` and moves of `move`: almost every narrow-phase test
    is a near-contact pair.  Every decision must be the oracle's (sign of the SAT margin against the guard band) except inside
    the 1e-5 window.  The fp32 GJK certifies a separation itself down to gaps of a few 1e-6 (its certificate n.s >= eps_g is
    evaluated from the support points), but between nearly parallel faces its simplex is often a sliver whose "origin inside"
    verdict cannot be trusted, and with gaps of 8e-6 many trials end inside the guard band or barely overlapping, where the fp32
    run converges without a certificate: both answer "unsure", and the pair must be decided by the fp64 re-run (
    counted on the device: 1243 and 6027 re-runs in 2048 trials).  In the second case most trials lie close to the 1e-5 window.
    Regression for the round-2 finding at full config 3: an fp32 "origin inside the tetrahedron" verdict on a sliver simplex."""
    # 7^3 cubes in 4^3 cells of width 1.75: 145 particles around a cell, inside the staging capacity of the warp-per-cell pass
    w = wl.cubes(7, spacing=1.0 + gap, max_tilt=gap / 4, d=move, a=move, name="cubes_near_contact")
    g, o = gpu(w), orc(w)
    assert g.count_overlaps() == 0 and o.count_overlaps_bruteforce() == 0
    g.enable_trace(True)
    marginal = trials = 0
    for s in range(8):
        g.sweep(1)
        f = o.sweep(follow=g.read_trace(), follow_tol=MARGIN_TOL)["follow"]
        assert f["hard_mismatch"] == 0, (s, f)
        marginal += f["marginal"]
        gp, gq = g.get_state(); op, oq = o.get_state()
        assert np.array_equal(gp, op) and np.max(np.abs(gq.astype(np.float64) - oq)) < 1e-5
        o.set_state(op, gq)
    c = g.counters()
    trials = c["trials"]
    reruns = g.get_stat("gjk_f64_reruns")
    rej = c["trans_rej_overlap"] + c["rot_rej_overlap"]
    print(f"near-contact cubes gap {gap}: {trials} trials, {rej} overlap rejects, {marginal} marginal, {reruns} fp64 re-runs")
    assert rej > 0.05 * trials and c["trans_acc"] + c["rot_acc"] > 0.05 * trials      # both outcomes occur
    assert g.count_overlaps() == 0                                                    # the strict fp64 validator agrees
    assert marginal <= 0.02 * trials
    assert reruns > 0.1 * trials                                                      # the mixed-precision branch carries this case


def test_out_of_box_and_non_finite_coordinates_are_reported_not_fatal():
    """a coordinate outside [-L/2, L/2) or an inf used to index the histogram out of bounds.  Now the cell index is
    clamped, the particle counted, and the next synchronising call reports HPMC_E_ARG; a fresh bind of a valid state works."""
    from paper_1509_04692_b200 import binding as hb
    for w in (wl.pentagons(24), wl.config(2) if False else wl.pentagons(200), wl.cubes(6)):   # single-CTA and multi-launch builds, 3-D
        for bad_value in (0.75 * w.L[0], -3.0 * w.L[0], np.inf, np.nan):
            g = gpu(w)
            pos = w.pos4.copy()
            pos[5, 0] = bad_value
            g.bind(pos, w.quat4)
            g.sweep(2)                                   # must not fault
            with pytest.raises(hb.HpmcError):
                g.count_overlaps()
            g.bind(w.pos4, w.quat4)                      # a valid state clears the condition
            g.sweep(2)
            assert g.count_overlaps() == 0


def test_dataflow_pass_with_many_tiles_and_partial_edges_matches_per_colour_launches():
    """every other forced-dataflow case has 1-4 tiles per colour.  256 x 160 pentagons with the 2-warp tile shape:
    64 x 79 active cells per colour = 2 x 40 tiles with a partial last tile in x and in y, more (colour, tile) tickets than the
    GPU holds CTAs at once is not reached at this size, but tiles do wait on the stamps of their nine neighbours; 20 sweeps,
    including CUDA-graph replay, bit for bit against one launch per colour."""
    base = wl.pentagons(256)
    ny = 160
    keep = np.arange(256 * ny)
    L = (256.0, float(ny))
    pos = base.pos4[keep].copy()
    pos[:, 1] += 0.5 * (256.0 - ny)                      # rows 0..159 recentred in the shorter box
    w = wl.Workload(name="pentagons_256x160", dim=2, N=256 * ny, L=L, kind=base.kind, diameter=0.0, verts=base.verts, d=base.d,
                    a=base.a, n_select=4, sweeps=1, pos4=pos, quat4=base.quat4[keep].copy())
    out = []
    for flow in (1, 0):
        g = gpu(w)
        assert g.count_overlaps() == 0
        g.set_option("tile_shape", 3); g.set_option("flow", flow)
        g.sweep(1); g.sweep(19)
        out.append((g.get_state(), g.counters()))
        assert g.count_overlaps() == 0
    assert np.array_equal(out[0][0][0], out[1][0][0]) and np.array_equal(out[0][0][1], out[1][0][1]) and out[0][1] == out[1][1]


@pytest.mark.parametrize("shape", ["triangle", "square", "hexagon", "irregular_heptagon", "irregular_pentagon"])
@pytest.mark.parametrize("path", [2, 3])
def test_polygon_test_variants_lockstep_with_oracle(shape, path):
    """polygon_separated has three routes: regular pentagons unrolled (every other pentagon test), regular n-gons with a
    runtime n (only the normal closest to the separation is evaluated), and general convex polygons (every axis that passes the
    inscribed-radius test).  The last two through the tile pass and the warp-per-cell pass, against the oracle's full SAT margin."""
    rng = np.random.default_rng(4)
    if shape == "irregular_heptagon":
        ang = np.sort(rng.uniform(0, 2 * np.pi, 7)); ang[0] = 0.1
        verts = 0.5 * np.stack([np.cos(ang), np.sin(ang)], axis=1)
    elif shape == "irregular_pentagon":                      # five vertices, not regular: must NOT take the unrolled pentagon route
        verts = np.array([[0.5, 0.0], [0.1, 0.42], [-0.4, 0.2], [-0.3, -0.3], [0.2, -0.35]])
    else:
        verts = wl.regular_polygon({"triangle": 3, "square": 4, "hexagon": 6}[shape], 0.5)
    w = _lattice_workload(2, (34, 30), (1.06, 1.1), wl.KIND_POLYGON, verts=verts, d=0.15, a=0.4, seed=8)
    from paper_1509_04692_b200 import binding as hb
    g, o = hb.from_workload(w, seed=2), orc(w, seed=2)
    g.set_option("path", path)
    assert g.count_overlaps() == 0 and o.count_overlaps_cells() == 0
    g.enable_trace(True)
    marginal = 0
    for s in range(8):
        g.sweep(1)
        f = o.sweep(follow=g.read_trace(), follow_tol=MARGIN_TOL)["follow"]
        assert f["hard_mismatch"] == 0, (shape, path, s, f)
        marginal += f["marginal"]
        gp, gq = g.get_state(); op, oq = o.get_state()
        assert np.array_equal(gp, op) and np.max(np.abs(gq.astype(np.float64) - oq)) < 1e-5
        o.set_state(op, gq)
    gc, oc = g.counters(), o.counters()
    assert all(gc[k] == oc[k] for k in oc)
    assert gc["trans_rej_overlap"] + gc["rot_rej_overlap"] > 0.05 * gc["trials"]          # the narrow phase decides many trials
    assert g.count_overlaps() == 0 and o.count_overlaps_cells() == 0 and marginal <= 3


def test_lockstep_in_a_box_of_edge_20000():
    """R11/R22: fp32 coordinates of magnitude 10^4 (spacing 1e-3).  The cell width carries 3 ulp(L) of slack there; the CUDA path
    and the oracle must still agree on every cell index and decision, also for the particles at the seam."""
    L = (20000.0, 8.0)
    xs = np.concatenate([np.arange(-10000.0 + 0.6, -10000.0 + 150, 1.05), np.arange(10000.0 - 150, 10000.0 - 0.6, 1.05)])
    ys = np.array([-3.0, -1.9, -0.8, 0.3, 1.4, 2.5])
    P = np.array([[x, y] for x in xs for y in ys])
    N = P.shape[0]
    pos = np.zeros((N, 4), np.float32); pos[:, :2] = P
    rng = np.random.default_rng(2)
    th = rng.uniform(0, 2 * np.pi, N)
    quat = np.zeros((N, 4), np.float32); quat[:, 0] = np.cos(th / 2); quat[:, 3] = np.sin(th / 2)
    w = wl.Workload(name="long_box", dim=2, N=N, L=L, kind=wl.KIND_POLYGON, diameter=0.0, verts=wl.regular_polygon(5, 0.5), d=0.3, a=0.5,
                    n_select=4, sweeps=1, pos4=pos, quat4=quat)
    for path in (2, 3):
        from paper_1509_04692_b200 import binding as hb
        g, o = hb.from_workload(w, seed=4), orc(w, seed=4)
        assert list(g.n[:2]) == [19882, 6] and np.array_equal(g.n, o.n)
        g.set_option("path", path)
        g.enable_trace(True)
        marginal = 0
        for s in range(8):
            cid, cst, mem, shift, perm = g.cell_list(s)
            oshift, _ = o.sweep_header(s)
            ocid, ocst, omem = o.cell_list(oshift)
            assert np.array_equal(cid, ocid) and np.array_equal(cst, ocst) and np.array_equal(mem, omem)
            g.sweep(1)
            f = o.sweep(follow=g.read_trace(), follow_tol=MARGIN_TOL)["follow"]
            assert f["hard_mismatch"] == 0, (path, s, f)
            marginal += f["marginal"]
            gp, gq = g.get_state(); op, oq = o.get_state()
            assert np.array_equal(gp, op) and np.max(np.abs(gq.astype(np.float64) - oq)) < 1e-5
            o.set_state(op, gq)
        assert g.count_overlaps() == 0 and o.count_overlaps_bruteforce() == 0 and marginal <= 3


@pytest.mark.parametrize("case", ["pentagons_ns1", "pentagons_ns3", "pentagons_ns6", "pentagons_ns9", "disks_ns5", "needles_crowded",
                                  "needles_overfull"])
def test_speculative_pass_lockstep_with_oracle(case):
    """k_sweep_spec2d evaluates the decision tree of four trials of a cell at once (sweep_spec2d.cuh).  Against the oracle in lock
    step: batches that are not full (n_select 1, 3), several batches (6, 9), cells with several members -- where a node's
    state differs from the staged one for OTHER members too -- and cells with more members than the tree handles (fallback)."""
    opts = {"path": 5}
    pent = wl.regular_polygon(5, 0.5)
    if case.startswith("pentagons_ns"):
        w = _lattice_workload(2, (26, 30), (1.06, 1.04), wl.KIND_POLYGON, verts=pent, d=0.12, a=0.3, n_select=int(case[-1]), seed=11)
    elif case == "disks_ns5":
        w = _lattice_workload(2, (30, 26), (1.08, 1.1), wl.KIND_DISK, diameter=1.0, d=0.2, n_select=5)
    else:
        # thin rectangles 1.0 x 0.16 stacked at a pitch of 0.5 (crowded: mostly 2-4 per cell) or 0.2 (overfull: most cells above
        # kSpecMaxMem = 4), all nearly parallel: many members per cell, and the moved particle's cell mates are its closest neighbours
        pitch = 0.5 if case == "needles_crowded" else 0.2
        verts = np.array([[0.5, -0.08], [0.5, 0.08], [-0.5, 0.08], [-0.5, -0.08]])
        w = _lattice_workload(2, (20, int(round(20.8 / pitch))), (1.08, pitch), wl.KIND_POLYGON, verts=verts, d=0.03, a=0.05, n_select=4, seed=12)
        rng = np.random.default_rng(13)
        th = rng.uniform(-0.03, 0.03, w.N)
        w.quat4[:, 0], w.quat4[:, 3] = np.cos(th / 2), np.sin(th / 2)
    from paper_1509_04692_b200 import binding as hb
    g, o = hb.from_workload(w, seed=9), orc(w, seed=9)
    for k, v in opts.items():
        g.set_option(k, v)
    assert "spec2d" in g.describe_pass()
    assert g.count_overlaps() == 0 and o.count_overlaps_cells() == 0
    g.enable_trace(True)
    marginal, multi, share = 0, 0, 1.0
    for s in range(8):
        cid, cst, mem, shift, perm = g.cell_list(s)
        cnt = np.diff(cst)
        multi = max(multi, int(cnt.max()))
        share = min(share, float(np.mean((cnt[cnt > 0] >= 2) & (cnt[cnt > 0] <= 4))))
        g.sweep(1)
        f = o.sweep(follow=g.read_trace(), follow_tol=MARGIN_TOL)["follow"]
        assert f["hard_mismatch"] == 0, (case, s, f)
        marginal += f["marginal"]
        gp, gq = g.get_state(); op, oq = o.get_state()
        assert np.array_equal(gp, op) and np.max(np.abs(gq.astype(np.float64) - oq)) < 1e-5
        o.set_state(op, gq)
    gc, oc = g.counters(), o.counters()
    assert all(gc[k] == oc[k] for k in oc)
    assert gc["trans_acc"] > 0.1 * gc["trials"] and g.count_overlaps() == 0 and marginal <= 5
    if case == "needles_crowded":
        assert share > 0.5, share            # most occupied cells hold 2-4 members: the tree runs with cell mates in its states
    if case == "needles_overfull":
        assert multi >= 5


def test_sweep_host_pose2d_equals_sweep_host():
    """The 2-D host-buffer call with one pose (x, y, qw, qz) per particle makes the trajectory of hpmc_sweep_host (pos4 + quat4)
    bit for bit, returns the same counters, leaves the bound device arrays in the pos4 / quat4 layout, and refuses 3-D systems."""
    import torch
    from paper_1509_04692_b200 import binding as hb
    w = wl.pentagons(48)
    a, b = gpu(w), gpu(w)
    hp, hq = torch.from_numpy(w.pos4.copy()).pin_memory(), torch.from_numpy(w.quat4.copy()).pin_memory()
    op, oq = torch.empty(w.N, 4).pin_memory(), torch.empty(w.N, 4).pin_memory()
    pose = torch.from_numpy(np.ascontiguousarray(np.concatenate([w.pos4[:, :2], w.quat4[:, [0, 3]]], axis=1))).pin_memory()
    out = torch.empty(w.N, 4).pin_memory()
    for step in range(3):
        ca = a.sweep_host(hp, hq, 2, op, oq)
        cb = b.sweep_host_pose2d(pose, 2, out)
        assert ca == cb
        assert torch.equal(out[:, :2], op[:, :2]) and torch.equal(out[:, 2], oq[:, 0]) and torch.equal(out[:, 3], oq[:, 3])
        hp.copy_(op); hq.copy_(oq); pose.copy_(out)
    pb, qb = b.get_state()
    assert np.array_equal(pb, op.numpy()) and np.array_equal(qb, oq.numpy())
    assert b.count_overlaps() == 0
    assert b.sweep_host_pose2d(pose, 1, None)["trials"] > ca["trials"]          # no output buffer: counters only
    c3 = gpu(wl.cubes(6))
    with pytest.raises(hb.HpmcError):
        c3.sweep_host_pose2d(pose, 1, out)
