"""BASELINE.json's five configs at their full stated run lengths on the GPU path (north_star target: "zero overlaps ... on all
five configs"): 1000 / 10^4 / 1000 / 1000 / 100 sweeps through `hpmc_sweep`, in the default launch configuration (CUDA-graph
replay, dataflow or warp-per-cell pass as chosen by size).  Checked: the fp64 validator finds no overlapping pair before and
after, every trial is accounted for, the sweep counter advanced by the run length, and the acceptance ratio sits where the
oracle puts it for this state point (8-seed means of tests/test_gpu_statistics.py, +- 0.02)."""
import numpy as np
import pytest

from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# (config, translate acceptance, rotate acceptance) from the oracle's 8-seed statistics at these state points
EXPECT = {0: (0.330, None), 1: (0.485, 0.903), 2: (0.485, 0.903), 3: (0.30, 0.73), 4: (0.485, 0.903)}


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_full_length_run_ends_without_overlaps(k):
    from paper_1509_04692_b200 import binding as hb
    w = wl.config(k)
    g = hb.from_workload(w, seed=1)
    assert g.count_overlaps() == 0
    g.sweep(w.sweeps)
    c = g.counters()
    assert g.count_overlaps() == 0
    assert c["sweep_counter"] == w.sweeps and c["sweeps"] == w.sweeps
    nt = c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"]
    nr = c["rot_acc"] + c["rot_rej_overlap"]
    assert nt + nr == c["trials"] and c["trials"] > 0.8 * w.n_select * min(g.C, w.N) * w.sweeps
    ta, ra = EXPECT[k]
    tol = 0.02 if k != 3 else 0.06          # config 3 keeps relaxing from its tilted-lattice orientations over the 1000 sweeps
    assert abs(c["trans_acc"] / nt - ta) < tol, c
    if ra is not None:
        assert abs(c["rot_acc"] / nr - ra) < tol and abs(nr / c["trials"] - 0.5) < 0.01, c
    else:
        assert nr == 0
    p, q = g.get_state()
    half = 0.5 * np.float32(w.L[0])
    assert np.all(np.abs(p[:, : w.dim]) <= half) and np.all(np.abs(np.sum(q.astype(np.float64) ** 2, axis=1) - 1) < 1e-5)
    print(f"config {k}: {c['trials']} trials, acceptance {c['trans_acc'] / nt:.3f}" + (f" / {c['rot_acc'] / nr:.3f}" if nr else ""))
