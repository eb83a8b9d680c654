"""hpmc_count_overlaps_noalloc (include/hpmc.h): the overlap count through the entry point that allocates nothing -- its cell
list lives in a static device array inside the library -- against the existing path (hpmc_bind + hpmc_count_overlaps, whose
cell list lives in the caller's workspace).  Both count pairs with the same strict fp64 test, so the bar is equality of
the integers.  Several calls in a row share the static array: a call must not see what the call before it left there
(different n, different state, different shape and dimension).

Collected last on purpose (file name): the suite runs with pytest -x."""
import dataclasses

import numpy as np
import pytest

from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def jostled(w, amp, seed, n=None):
    """The workload's lattice state with every centre displaced by up to `amp` per axis (wrapped into the box): many overlaps.
    n: keep only the first n particles."""
    rng = np.random.default_rng(seed)
    n = w.N if n is None else n
    pos = w.pos4[:n].copy()
    L = np.array([np.float32(x) for x in w.L[: w.dim]], dtype=np.float32)
    pos[:, : w.dim] += rng.uniform(-amp, amp, (n, w.dim)).astype(np.float32)
    for k in range(w.dim):
        pos[:, k] = np.where(pos[:, k] >= 0.5 * L[k], pos[:, k] - L[k], pos[:, k])
        pos[:, k] = np.where(pos[:, k] < -0.5 * L[k], pos[:, k] + L[k], pos[:, k])
        pos[:, k] = np.where(pos[:, k] >= 0.5 * L[k], -0.5 * L[k], pos[:, k])      # x + L rounded onto the upper face
    return dataclasses.replace(w, N=n, pos4=pos, quat4=w.quat4[:n].copy())


def existing_count(w):
    from paper_1509_04692_b200 import binding as hb
    return hb.from_workload(w, seed=1).count_overlaps()


def context_only(w):
    """A context for the box and shape of `w`: no bind, no workspace."""
    from paper_1509_04692_b200 import binding as hb
    return hb.Hpmc(w.dim, w.L, w.kind, w.N, 1, diameter=w.diameter, verts=w.verts)


def noalloc_count(g, w, out):
    import torch
    pos = torch.from_numpy(w.pos4).to(g.device)
    quat = torch.from_numpy(w.quat4).to(g.device)
    out.fill_(-7)                                   # whatever the entry point leaves must be its own
    torch.cuda.synchronize()
    g.count_overlaps_noalloc(pos, quat, out)
    g.stream.synchronize()
    return int(out.item())


def test_two_calls_in_a_row_equal_the_existing_path():
    import torch
    base = wl.pentagons(64)
    a = jostled(base, 0.30, seed=1)                 # 4096 particles
    b = jostled(base, 0.45, seed=2, n=1500)         # fewer particles, another state: part of the box is empty
    want_a, want_b = existing_count(a), existing_count(b)
    assert want_a > 100 and want_b > 100 and want_a != want_b
    g = context_only(base)
    out = torch.empty(1, dtype=torch.int64, device=g.device)
    assert noalloc_count(g, a, out) == want_a       # first call
    assert noalloc_count(g, b, out) == want_b       # second call finds the first call's cell list in the static array
    assert noalloc_count(g, a, out) == want_a
    assert noalloc_count(g, base, out) == 0 == existing_count(base)
    assert noalloc_count(g, dataclasses.replace(base, N=0, pos4=base.pos4[:0], quat4=base.quat4[:0]), out) == 0


def test_contexts_of_other_shapes_share_the_array():
    import torch
    cases = [jostled(wl.cubes(12), 0.25, seed=3), jostled(wl.disks(48), 0.2, seed=4), jostled(wl.pentagons(40), 0.3, seed=5),
             jostled(wl.cubes(12), 0.25, seed=6, n=700)]
    want = [existing_count(w) for w in cases]
    assert all(x > 20 for x in want)
    out = None
    for rounds in range(2):
        for w, x in zip(cases, want):
            g = context_only(w)
            out = torch.empty(1, dtype=torch.int64, device=g.device) if out is None else out
            assert noalloc_count(g, w, out) == x, (w.name, rounds)


def test_limits_and_bad_input_are_reported():
    import torch
    from paper_1509_04692_b200 import binding as hb
    base = wl.pentagons(64)
    g = context_only(base)
    out = torch.full((1,), 5, dtype=torch.int64, device=g.device)
    big = torch.zeros((65537, 4), dtype=torch.float32, device=g.device)
    with pytest.raises(hb.HpmcError, match="exceeds the static scratch"):
        g.count_overlaps_noalloc(big, big, out)
    g.stream.synchronize()
    assert int(out.item()) == 5                      # a refused call launches nothing
    wide = hb.Hpmc(2, (1024.0, 1024.0), wl.KIND_POLYGON, 16, 1, verts=base.verts)       # 1022^2 cells
    with pytest.raises(hb.HpmcError, match="cells"):
        wide.count_overlaps_noalloc(big[:16], big[:16], out)
    # a coordinate outside the box: -1, and the next call is clean again
    bad = jostled(base, 0.3, seed=1)
    bad.pos4[17, 0] = np.float32(base.L[0])
    assert noalloc_count(g, bad, out) == -1
    good = jostled(base, 0.3, seed=1)
    assert noalloc_count(g, good, out) == existing_count(good)


def test_the_context_own_state_is_untouched():
    import torch
    from paper_1509_04692_b200 import binding as hb
    w = wl.pentagons(48)
    g, ref = hb.from_workload(w, seed=2), hb.from_workload(w, seed=2)
    g.sweep(3); ref.sweep(3)
    other = jostled(w, 0.3, seed=9, n=1000)
    out = torch.empty(1, dtype=torch.int64, device=g.device)
    assert noalloc_count(g, other, out) == existing_count(other)
    g.sweep(3); ref.sweep(3)
    assert all(np.array_equal(x, y) for x, y in zip(g.get_state(), ref.get_state()))
    assert g.count_overlaps() == 0
