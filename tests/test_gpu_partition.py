"""One system on several ranks (paper_1509_04692_b200/partition.py): every rank holds the whole state and
runs the colour-pass tiles of its own slab of cell rows; boundary rows are copied between the ranks after every colour, the
slabs after the last.  Verified on ONE GPU with the ranks as contexts of one process stepped one after the other: the
trajectory must be bit-identical to the single-context one, on every rank, and the per-rank tallies must add up to it."""
import numpy as np
import pytest

from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("nranks", [2, 3, 5])
@pytest.mark.parametrize("case", ["pentagons_96", "disks_rect"])
def test_partitioned_sweeps_equal_the_single_context_trajectory(case, nranks):
    from paper_1509_04692_b200 import binding as hb
    from paper_1509_04692_b200.partition import LocalRanks
    if case == "pentagons_96":
        w = wl.pentagons(96)
    else:
        base = wl.disks(80)
        keep = np.arange(80 * 52)                                   # 80 x 52 lattice rows: a rectangular box, partial last tile row
        pos = base.pos4[keep].copy()
        pos[:, 1] += 0.5 * 1.1 * (80 - 52)
        w = wl.Workload(name="disks_80x52", dim=2, N=keep.size, L=(80 * 1.1, 52 * 1.1), kind=wl.KIND_DISK, diameter=1.0, verts=None,
                        d=0.15, a=0.0, n_select=4, sweeps=1, pos4=pos, quat4=base.quat4[keep].copy())
    ref = hb.from_workload(w, seed=1)
    ref.set_option("path", 2); ref.set_option("flow", 0)
    ranks = LocalRanks(w, nranks, seed=1)
    assert ranks.slabs[0][0] == 0 and ranks.slabs[-1][1] == int(ref.n[1])
    assert all(ranks.slabs[r][1] == ranks.slabs[r + 1][0] for r in range(nranks - 1))      # the slabs tile the rows
    for step in range(4):
        ref.sweep(2)
        ranks.sweep(2)
        rp, rq = ref.get_state()
        for r in range(nranks):
            p, q = ranks.get_state(r)
            assert np.array_equal(p, rp) and np.array_equal(q, rq), (case, nranks, step, r)
    rc, pc = ref.counters(), ranks.counters()
    for k in ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials"):
        assert rc[k] == pc[k], (k, rc, pc)
    assert pc["sweep_counter"] == 8 and ranks.count_overlaps(nranks - 1) == 0


def test_partition_of_one_is_the_plain_sweep_and_3d_is_refused():
    from paper_1509_04692_b200 import binding as hb
    w = wl.pentagons(64)
    a, b = hb.from_workload(w, seed=3), hb.from_workload(w, seed=3)
    a.set_option("path", 2); a.set_option("flow", 0)
    b.set_option("path", 2); b.set_option("flow", 0)
    b.set_partition(0, 1)
    a.sweep(3)
    for _ in range(3):
        b.sweep_phase(-1)
        for ci in range(4):
            b.sweep_phase(ci)
    assert all(np.array_equal(x, y) for x, y in zip(a.get_state(), b.get_state())) and a.counters() == b.counters()
    c = hb.from_workload(wl.cubes(6), seed=1)
    with pytest.raises(hb.HpmcError):
        c.set_partition(0, 2)
