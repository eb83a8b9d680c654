"""Pins for the oracle's cell list and sweep (O2, O3, O5, O6, P2-P4, P8)."""
import math

import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from paper_1509_04692_b200 import workloads as wl


def make(w, seed=1):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    return o


SMALL = {
    "disks": lambda: wl.disks(16),
    "pentagons": lambda: wl.pentagons(16),
    "cubes": lambda: wl.cubes(6),
}


def test_grid_rule_matches_survey_appendix():
    # O2 / R11: even, slack 2^-10 -> 70 / 62 / 1022 / 22 / 4092 cells per side for the five configs
    assert list(make(wl.disks(64)).n[:2]) == [70, 70]
    assert list(make(wl.pentagons(64)).n[:2]) == [62, 62]
    assert list(make(wl.cubes(8)).n) == [4, 4, 4]
    for L, n in ((1024.0, 1022), (4096.0, 4092)):
        o = ho.Oracle(2, (L, L), ho.KIND_POLYGON, 0, 1, verts=wl.regular_polygon(5, 0.5))
        assert list(o.n[:2]) == [n, n]
    o = ho.Oracle(3, (40.0,) * 3, ho.KIND_POLYHEDRON, 0, 1, verts=wl.cube_vertices(1.0))
    assert list(o.n) == [22, 22, 22]
    with pytest.raises(ValueError):   # fewer than 4 cells per side
        ho.Oracle(2, (3.9, 3.9), ho.KIND_DISK, 0, 1, diameter=1.0)


@pytest.mark.parametrize("name", list(SMALL))
def test_cell_list_invariants_and_geometry(name):
    w = SMALL[name]()
    o = make(w)
    o.sweeps(3)                               # off-lattice positions
    pos, _ = o.get_state()
    for t in range(4):
        shift, perm = o.sweep_header(t)
        assert sorted(perm.tolist()) == list(range(1 << w.dim))
        assert np.all(shift[: w.dim] >= 0) and np.all(shift[: w.dim] < o.w_f[: w.dim])
        cid, cst, mem = o.cell_list(shift)
        assert cst[0] == 0 and cst[-1] == w.N and np.all(np.diff(cst) >= 0)       # sum of counts = N
        assert sorted(mem.tolist()) == list(range(w.N))
        for c in np.unique(cid):
            seg = mem[cst[c]:cst[c + 1]]
            assert np.all(cid[seg] == c) and np.all(np.diff(seg) > 0)            # maps back; ascending tag (R8)
        # geometry in fp64: the particle really lies in the half-open box of its cell (up to fp32 rounding)
        L = o.L_f.astype(np.float64); wd = o.w
        f = np.mod(pos[:, :3].astype(np.float64) + 0.5 * L - shift.astype(np.float64), L) / wd
        cc = np.stack([cid % o.n[0], (cid // o.n[0]) % o.n[1], cid // (o.n[0] * o.n[1])], axis=1)
        for k in range(w.dim):
            delta = f[:, k] - cc[:, k]
            delta = np.where(delta < -0.5 * o.n[k], delta + o.n[k], delta)     # periodic wrap of the last cell
            assert np.all(delta > -1e-4) and np.all(delta < 1 + 1e-4)


@pytest.mark.parametrize("name", list(SMALL))
def test_zero_overlap_invariant_bruteforce(name):
    # P8 / P:247: "run short simulations and check for any overlaps"; O5 is all N(N-1)/2 pairs, no cell list
    w = SMALL[name]()
    o = make(w)
    assert o.count_overlaps_bruteforce() == 0
    for _ in range(12 if name != "cubes" else 5):
        o.sweep()
        assert o.count_overlaps_bruteforce() == 0
        assert o.count_overlaps_cells() == 0
    c = o.counters()
    assert c["trials"] == c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"] + c["rot_acc"] + c["rot_rej_overlap"]
    assert c["trans_acc"] > 0 and c["trans_rej_overlap"] > 0 and c["trans_rej_cell"] > 0
    if name != "disks":
        assert c["rot_acc"] > 0 and c["rot_rej_overlap"] > 0


def test_overlap_counters_see_planted_overlaps():
    w = wl.pentagons(8)
    o = make(w)
    pos, quat = w.pos4.copy(), w.quat4.copy()
    pos[5, 0] = pos[4, 0] + 0.3; pos[5, 1] = pos[4, 1]          # particle 5 on top of particle 4
    pos[63, :2] = [-3.9, -3.9]; pos[0, :2] = [3.95, 3.95]         # and one pair across both periodic seams
    o.set_state(pos, quat)
    n = o.count_overlaps_bruteforce()
    assert n >= 2 and o.count_overlaps_cells() == n


@pytest.mark.parametrize("name", list(SMALL))
def test_all_N_twin_makes_identical_decisions(name):
    # O6: scanning all N-1 particles instead of the 3^d cells must not change one decision;
    # pins neighbourhood indexing, the periodic seam and the claim P:59 "only its cell and the neighboring cells"
    w = SMALL[name]()
    a, b = make(w), make(w)
    for _ in range(6 if name != "cubes" else 3):
        ra = a.sweep(neighbour_mode=0, want_trace=True, want_mmin=True)
        rb = b.sweep(neighbour_mode=1, want_trace=True, want_mmin=True)
        assert np.array_equal(ra["trace"], rb["trace"])
        ma, mb = ra["mmin"], rb["mmin"]
        both = np.isfinite(ma) & np.isfinite(mb)
        assert np.array_equal(np.isfinite(ma), np.isfinite(mb)) and np.array_equal(ma[both], mb[both])
    pa, qa = a.get_state(); pb, qb = b.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)


@pytest.mark.parametrize("name", list(SMALL))
def test_same_colour_cells_are_independent(name):
    # P4: any serial order of same-colour cells gives the same result; same-colour particles are >= d_max apart
    w = SMALL[name]()
    a, b = make(w), make(w)
    dmax = ho.Shape(w.dim, w.kind, diameter=w.diameter, verts=w.verts).dmax
    for t in range(5 if name != "cubes" else 3):
        shift, _ = a.sweep_header(t)
        assert a.min_same_colour_distance(shift) >= dmax
        ra = a.sweep(reverse_cells=0, want_trace=True)
        rb = b.sweep(reverse_cells=1, want_trace=True)
        assert np.array_equal(ra["trace"], rb["trace"])
    pa, qa = a.get_state(); pb, qb = b.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)


def test_trace_and_follow_protocol_self_consistency():
    # O8: following one's own trace reports no mismatch; a flipped non-marginal decision is a hard mismatch
    w = wl.pentagons(16)
    a, b = make(w), make(w)
    ra = a.sweep(want_trace=True)
    rb = b.sweep(follow=ra["trace"], want_trace=True)
    assert rb["follow"]["hard_mismatch"] == 0 and rb["follow"]["marginal"] == 0
    assert rb["follow"]["compared"] == a.C * w.n_select
    c, d = make(w), make(w)
    rc = c.sweep(want_trace=True)
    tr = rc["trace"].copy()
    slot = int(np.nonzero((tr[:, 1] >> 8) == 1)[0][0])
    tr[slot, 1] = (tr[slot, 1] & 0xFF) | (3 << 8)
    rd = d.sweep(follow=tr)
    assert rd["follow"]["hard_mismatch"] == 1 and rd["follow"]["first_bad_slot"] == slot


def test_sweep_counter_restart_reproduces_trajectory():
    # counter-based RNG: state + sweep counter reproduce the trajectory bit for bit (no RNG state to save)
    w = wl.pentagons(12)
    a = make(w)
    a.sweeps(5)
    p5, q5 = a.get_state()
    a.sweeps(4)
    p9, q9 = a.get_state()
    b = make(w)
    b.set_state(p5, q5); b.sweep_counter = 5
    b.sweeps(4)
    pb, qb = b.get_state()
    assert np.array_equal(p9, pb) and np.array_equal(q9, qb)
    c = make(w, seed=2)
    c.sweeps(9)
    assert not np.array_equal(c.get_state()[0], p9)


def test_leave_cell_rate_closed_form():
    # P2: the random grid shift makes cell-relative coordinates uniform, so P(trial leaves its cell)
    # = 1 - prod_k (1 - d/(2 w_k)); dilute system so that overlap rejections do not matter
    rng = np.random.default_rng(7)
    L, N = 70.4, 300
    pts = []
    while len(pts) < N:
        p = rng.uniform(-L / 2, L / 2, size=2)
        if all(np.hypot(*(((p - q) + L / 2) % L - L / 2)) > 1.2 for q in pts):
            pts.append(p)
    pos = np.zeros((N, 4), np.float32); pos[:, :2] = np.array(pts)
    quat = np.zeros((N, 4), np.float32); quat[:, 0] = 1
    o = ho.Oracle(2, (L, L), ho.KIND_DISK, N, 3, diameter=1.0)
    o.set_moves(0.15, 0.0, 4); o.set_state(pos, quat)
    o.sweeps(400)
    c = o.counters()
    p_stay = (1 - 0.15 / (2 * o.w[0])) * (1 - 0.15 / (2 * o.w[1]))
    assert p_stay == pytest.approx(0.8564, abs=1e-4)            # SURVEY P2 value for the config-0 grid
    frac = c["trans_rej_cell"] / c["trials"]
    se = math.sqrt(p_stay * (1 - p_stay) / c["trials"])
    assert abs(frac - (1 - p_stay)) < 4 * se
    assert o.count_overlaps_bruteforce() == 0


def test_translation_distribution_uniform_in_cube():
    # R5 + P:243: accepted displacements in a near-empty box are uniform in [-d,d)^2
    L, N = 40.0, 16
    pos = np.zeros((N, 4), np.float32)
    pos[:, 0] = np.linspace(-18, 18, N); pos[:, 1] = np.linspace(-17, 17, N)[::-1]
    quat = np.zeros((N, 4), np.float32); quat[:, 0] = 1
    o = ho.Oracle(2, (L, L), ho.KIND_DISK, N, 5, diameter=1.0)
    o.set_moves(0.05, 0.0, 1); o.set_state(pos, quat)
    disp = []
    prev = pos.copy()
    for _ in range(1500):
        o.sweep()
        cur, _ = o.get_state()
        dd = (cur[:, :2] - prev[:, :2]).astype(np.float64)
        dd = (dd + L / 2) % L - L / 2
        disp.append(dd[np.any(dd != 0, axis=1)])
        prev = cur
    disp = np.concatenate(disp)
    assert disp.shape[0] > 15000 and np.all(np.abs(disp) <= 0.05 + 1e-6)
    # leaving the cell truncates large moves more often -> compare only the central region |delta| < d/2
    core = disp[np.all(np.abs(disp) < 0.025, axis=1)] / 0.025
    h, _, _ = np.histogram2d(core[:, 0], core[:, 1], bins=6, range=[[-1, 1], [-1, 1]])
    expected = core.shape[0] / 36
    # chi^2 with 35 dof (mean 35, sd 8.4); inside the core the leave-cell probability varies by a few
    # per cent with |delta| (w >= 1, d = 0.05), far below what this sample resolves
    assert ((h - expected) ** 2 / expected).sum() < 80.0
    assert abs(core[:, 0].mean()) < 0.03 and abs(core[:, 1].mean()) < 0.03


def test_mutation_dropping_leave_cell_reject_breaks_the_invariant():
    # allowing displacements to cross from an active domain to an inactive one is incorrect
    w = wl.disks(16)
    o = make(w)
    o.set_mutations(no_leave_cell_reject=1)
    o.sweeps(30)
    assert o.count_overlaps_bruteforce() > 0


def test_textbook_metropolis_keeps_zero_overlaps_and_moves_everything():
    w = wl.pentagons(10)
    o = make(w)
    o.textbook_trials(20 * w.N)
    assert o.count_overlaps_bruteforce() == 0
    c = o.counters()
    assert c["trans_rej_cell"] == 0 and c["trials"] == 20 * w.N and c["rot_acc"] > 0 and c["trans_acc"] > 0


def test_large_box_grid_keeps_same_colour_cells_apart():
    # R11/R22: in a box of edge 20 000 the fp32 cell function misplaces boundaries by ~1e-3; the cell width then carries a slack
    # of 3 ulp(L) instead of d_max 2^-10, so that particles of different same-colour cells still cannot come within d_max (P4)
    L = (20000.0, 8.0)
    pent = wl.regular_polygon(5, 0.5)
    o = ho.Oracle(2, L, ho.KIND_POLYGON, 0, 1, verts=pent)
    assert list(o.n[:2]) == [19882, 6] and o.w[0] - 1.0 >= 3 * 2.0 ** -9          # ulp of differences in [16384, 32768) is 2^-9
    # a dense row of pentagons at both ends of the box (largest coordinates: coarsest fp32 spacing) and across the seam
    xs = np.concatenate([np.arange(-10000.0 + 0.6, -10000.0 + 150, 1.05), np.arange(10000.0 - 150, 10000.0 - 0.6, 1.05)])
    ys = np.array([-3.0, -1.9, -0.8, 0.3, 1.4, 2.5])
    P = np.array([[x, y] for x in xs for y in ys])
    N = P.shape[0]
    pos = np.zeros((N, 4), np.float32); pos[:, :2] = P
    rng = np.random.default_rng(2)
    th = rng.uniform(0, 2 * np.pi, N)
    quat = np.zeros((N, 4), np.float32); quat[:, 0] = np.cos(th / 2); quat[:, 3] = np.sin(th / 2)
    o = ho.Oracle(2, L, ho.KIND_POLYGON, N, 3, verts=pent)
    o.set_moves(0.3, 0.5, 4); o.set_state(pos, quat)
    assert o.count_overlaps_bruteforce() == 0
    for t in range(25):
        shift, _ = o.sweep_header(t)
        assert o.min_same_colour_distance(shift) >= 1.0
        o.sweep()
    assert o.count_overlaps_bruteforce() == 0
    c = o.counters()
    assert c["trans_acc"] > 0 and c["trans_rej_overlap"] > 0
