"""S:8(f)-1 / 8(f)-2: the paper's benchmark state points through the existing kernels -- pentagons at phi = 0.676 with move
sizes tuned to 20 % acceptance and dodecahedra at phi = 0.5, truncated octahedra -- LOCKED TO THE
ORACLE at that density: every trial of the following sweeps compared (O8), positions bit-exact, counters equal, zero overlaps
by the oracle's own O(N^2) brute force.  At these densities almost every trial has near-contact neighbours, so the narrow
phase (polygon SAT; fp32 GJK with its fp64 re-run) is exercised where it matters, unlike the dilute lattice cases of
tests/test_gpu_parity.py.

No input of the oracle comes from the CUDA path: the dense pentagon state is tests/golden/pentagons_1024_phi0676.npz, written
by tests/golden/make_dense_pentagons.py with the oracle's own sweeps; the polyhedra start from a seeded FCC crystal at
phi = 0.5 (workloads.fcc_polyhedra), which needs no simulation.  The GPU-side harness that prepares the full-size states for
bench.py (paper_1509_04692_b200/statepoints.py) is tested separately below, against its own invariants only."""
import os

import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def lock(w, sweeps, seed=3):
    from paper_1509_04692_b200 import binding as hb
    g = hb.from_workload(w, seed=seed)
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    o.set_threads(min(os.cpu_count() or 1, 16))
    assert np.array_equal(g.n, o.n)
    assert g.count_overlaps() == 0 and o.count_overlaps_bruteforce() == 0
    g.enable_trace(True)
    marginal = 0
    for s in range(sweeps):
        g.sweep(1)
        f = o.sweep(follow=g.read_trace(), follow_tol=1e-5)["follow"]
        assert f["hard_mismatch"] == 0, (w.name, s, f)
        marginal += f["marginal"]
        gp, gq = g.get_state(); op, oq = o.get_state()
        assert np.array_equal(gp, op) and np.max(np.abs(gq.astype(np.float64) - oq)) < 1e-5
        o.set_state(op, gq)
    gc, oc = g.counters(), o.counters()
    for key in ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials"):
        assert gc[key] == oc[key], (key, gc, oc)
    assert g.count_overlaps() == 0 and o.count_overlaps_bruteforce() == 0
    return g, gc, marginal


def test_pentagons_at_the_papers_density_with_tuned_moves():
    z = np.load(os.path.join(GOLDEN, "pentagons_1024_phi0676.npz"))
    L = float(z["L"])
    w = wl.Workload(name="pentagons_1024_phi0.676", dim=2, N=1024, L=(L, L), kind=wl.KIND_POLYGON, diameter=0.0,
                    verts=wl.regular_polygon(5, 0.5), d=float(z["d"]), a=float(z["a"]), n_select=4, sweeps=10, pos4=z["pos4"], quat4=z["quat4"])
    area = 2.5 * 0.25 * np.sin(2 * np.pi / 5)
    assert abs(w.N * area / L ** 2 - 0.676) < 1e-4
    g, c, marginal = lock(w, 10)
    nt = c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"]
    acc_t, acc_r = c["trans_acc"] / nt, c["rot_acc"] / (c["rot_acc"] + c["rot_rej_overlap"])
    print(f"pentagons phi = 0.676: N = {w.N}, d = {w.d:.4f}, a = {w.a:.4f}, acceptance {acc_t:.3f} / {acc_r:.3f}, {c['trials']} trials "
          f"locked, {marginal} marginal")
    assert abs(acc_t - 0.2) < 0.04                                       # P:47-49 (rotations: capped step, see the golden script)
    assert marginal <= max(3, 2e-3 * c["trials"])


@pytest.mark.parametrize("shape", ["dodecahedra", "truncated_octahedra"])
def test_polyhedra_at_phi_half(shape):
    verts = wl.dodecahedron_vertices(0.5) if shape == "dodecahedra" else wl.truncated_octahedron_vertices(0.5)
    # the crystal leaves gaps of ~0.16 at phi = 0.5 (the fluid is the stable phase): steps large enough to collide from the first sweep
    w = wl.fcc_polyhedra(verts, 4, 0.5, max_tilt=0.03, name=f"{shape}_fcc_256", d=0.2, a=0.5)
    g, c, marginal = lock(w, 8)
    reruns = g.get_stat("gjk_f64_reruns")
    rej = c["trans_rej_overlap"] + c["rot_rej_overlap"]
    print(f"{shape} phi = 0.5: N = {w.N}, {c['trials']} trials locked, {rej} overlap rejects, {marginal} marginal, {reruns} fp64 re-runs")
    assert rej > 0.15 * c["trials"] and c["trans_acc"] + c["rot_acc"] > 0.1 * c["trials"]     # a dense state: both outcomes occur
    assert marginal <= max(3, 5e-3 * c["trials"])


def test_harness_compression_and_move_tuning_reach_the_paper_state():
    """statepoints.py (what bench.py --paper-states uses at 65 536 pentagons): NVT compression by box steps that are kept only
    when hpmc_count_overlaps == 0, periodic replication, move-size tuning.  Checked against its own invariants."""
    from paper_1509_04692_b200 import binding as hb
    from paper_1509_04692_b200 import statepoints as sp
    w = sp.compress(wl.pentagons(32, name="pentagons_1024"), 0.676 * (1 + 2e-4))
    assert abs(sp.packing_fraction(w) / 0.676 - 1.0 - 2e-4) < 1e-5
    big = sp.replicate(w, 2, 0.676, decorrelate_sweeps=20)
    assert big.N == 4096 and abs(sp.packing_fraction(big) - 0.676) < 1e-5
    tuned, (acc_t, acc_r) = sp.tune_moves(big, 0.2)
    assert abs(acc_t - 0.2) < 0.03 and acc_r < 0.5
    g = hb.from_workload(tuned)
    g.sweep(50)
    assert g.count_overlaps() == 0
    p, q = g.get_state()
    assert not np.array_equal(p[:1024, :2] - p[0, :2], p[1024:2048, :2] - p[1024, :2])     # the copies have drifted apart
