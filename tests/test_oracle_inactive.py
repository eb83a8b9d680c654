"""Pins for the oracle's inactive region (domain decomposition: "only two regions (active and inactive) ...
these particles do not move during substeps"; reading R-strip: whole layers of cells along the last axis).

What the paper and the scheme fix, independent of the oracle's own loop:
  - a particle whose cell lies in an inactive layer keeps its exact state over the sweep; everything else still evolves
  - an all-zero mask is the plain sweep, an all-one mask is the identity
  - trials = n_select x (non-empty cells outside the inactive layers)                                        (R9)
  - the property the decomposition rests on ("There is no need to communicate ghost layer updates"): within one sweep
    nothing crosses an inactive layer, so the outcome in one band does not depend on the particles of another band
  - a mask on the wrong axis, shifted by one layer, or applied to particles instead of cells breaks one of these
"""
import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from paper_1509_04692_b200 import workloads as wl


def make(w, seed=1):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    return o


def layer_of_particles(o, t, dim):
    shift, _ = o.sweep_header(t)
    cid, cst, _ = o.cell_list(shift)
    n0, n1 = int(o.n[0]), int(o.n[1])
    layer = (cid // n0) % n1 if dim == 2 else cid // (n0 * n1)
    return layer, cid, cst


CASES = {"disks": lambda: wl.disks(16), "pentagons": lambda: wl.pentagons(16), "cubes": lambda: wl.cubes(12)}


@pytest.mark.parametrize("name", list(CASES))
def test_inactive_layers_hold_still_and_the_rest_moves(name):
    w = CASES[name]()
    o = make(w)
    o.sweeps(5)
    nl = int(o.n[w.dim - 1])
    mask = np.zeros(nl, dtype=np.uint8)
    mask[[1, nl // 2]] = 1
    o.set_inactive_layers(mask)
    for _ in range(4):
        t = o.sweep_counter
        layer, cid, cst = layer_of_particles(o, t, w.dim)
        p0, q0 = o.get_state()
        o.reset_counters()
        o.sweep()
        p1, q1 = o.get_state()
        frozen = mask[layer] != 0
        assert frozen.any() and (~frozen).any()
        assert np.array_equal(p0[frozen], p1[frozen]) and np.array_equal(q0[frozen], q1[frozen])
        moved = np.any(p0 != p1, axis=1) | np.any(q0 != q1, axis=1)
        assert moved[~frozen].mean() > 0.2               # the active region still evolves
        # R9: exactly n_select trials per non-empty cell outside the inactive layers
        counts = np.diff(cst)
        cells = np.arange(counts.size)
        n0, n1 = int(o.n[0]), int(o.n[1])
        cl = (cells // n0) % n1 if w.dim == 2 else cells // (n0 * n1)
        assert o.counters()["trials"] == w.n_select * int(np.count_nonzero((counts > 0) & (mask[cl] == 0)))
        assert o.count_overlaps_cells() == 0             # (pinned to the brute-force count in test_oracle_sweep.py)


def test_zero_mask_is_the_plain_sweep_and_full_mask_the_identity():
    w = wl.pentagons(16)
    a, b, c = make(w), make(w), make(w)
    nl = int(a.n[1])
    b.set_inactive_layers(np.zeros(nl, dtype=np.uint8))
    c.set_inactive_layers(np.ones(nl, dtype=np.uint8))
    a.sweeps(6); b.sweeps(6); c.sweeps(6)
    pa, qa = a.get_state(); pb, qb = b.get_state(); pc, qc = c.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(qa, qb)
    assert np.array_equal(pc, w.pos4) and np.array_equal(qc, w.quat4) and c.counters()["trials"] == 0
    b.set_inactive_layers(None)                          # cleared again
    a.sweeps(2); b.sweeps(2)
    assert np.array_equal(a.get_state()[0], b.get_state()[0])
    with pytest.raises(AssertionError):
        a.set_inactive_layers(np.zeros(nl + 1, dtype=np.uint8))


@pytest.mark.parametrize("name", ["pentagons", "cubes"])
def test_nothing_crosses_an_inactive_layer_within_a_sweep(name):
    # two inactive layers cut the periodic grid into two bands; replace the particles of band B by a different legal
    # configuration (here: band B after extra sweeps with band A frozen) and band A's sweep must come out bit-identical
    w = CASES[name]()
    base = make(w)
    base.sweeps(5)
    nl = int(base.n[w.dim - 1])
    k1, k2 = 2, nl // 2 + 1
    cut = np.zeros(nl, dtype=np.uint8); cut[[k1, k2]] = 1
    t = base.sweep_counter
    layer, _, _ = layer_of_particles(base, t, w.dim)
    in_a = (layer > k1) & (layer < k2)
    in_b = (layer < k1) | (layer > k2)
    assert in_a.sum() > 10 and in_b.sum() > 10
    p0, q0 = base.get_state()

    # variant: the same system with ONLY band B active for one sweep of the same grid (leave-cell rejection keeps every
    # particle in its cell, so band B's particles stay in band B and the configuration stays legal), counter set back
    other = make(w)
    other.set_state(p0, q0)
    other.sweep_counter = t
    only_b = np.ones(nl, dtype=np.uint8)
    only_b[:k1] = 0; only_b[k2 + 1:] = 0
    other.set_inactive_layers(only_b)
    other.sweep()
    pv, qv = other.get_state()
    changed = np.any(pv != p0, axis=1) | np.any(qv != q0, axis=1)
    assert changed.sum() > 5 and not changed[~in_b].any()
    var = make(w); var.set_state(pv, qv); var.sweep_counter = t
    assert var.count_overlaps_cells() == 0

    base.set_inactive_layers(cut); var.set_inactive_layers(cut)
    base.sweep(); var.sweep()
    pb, qb = base.get_state(); pw, qw = var.get_state()
    assert np.array_equal(pb[in_a], pw[in_a]) and np.array_equal(qb[in_a], qw[in_a])
    # and the cut matters: without it band A does feel band B within a few sweeps
    base2 = make(w); base2.set_state(p0, q0); base2.sweep_counter = t
    var2 = make(w); var2.set_state(pv, qv); var2.sweep_counter = t
    base2.sweeps(30); var2.sweeps(30)
    assert not np.array_equal(base2.get_state()[0][~in_b], var2.get_state()[0][~in_b])
