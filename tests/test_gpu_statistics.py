"""O10: statistical parity of the CUDA path and the oracle (BASELINE.json north_star: "acceptance ratio and
volume-perturbation pressure within 3 standard errors over 8 independent seeds").

Per seed: discard the first 10 % of the sweeps, then sample every 10 sweeps the per-type acceptance (counter
deltas) and the scale-factor histogram of the snapshot (oracle/pressure.py, the same fp64 analysis for both
sides).  Compared: |mean_GPU - mean_oracle| <= 3 sqrt(SE_GPU^2 + SE_oracle^2), SE = std over seeds / sqrt(8).
Two comparisons per workload: the same seeds 1..8 on both sides (trajectories then coincide except for marginal
trials, so the difference is far inside the bar) and GPU seeds 101..108 against oracle seeds 1..8 (independent
samples of the same ensemble).  The cube and pentagon VALUES themselves are "parity unpinned" against the paper
(it prints none for these state points); disks are pinned in tests/test_oracle_pressure.py.
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from oracle import hpmc_oracle as ho
from oracle import pressure as pr
from paper_1509_04692_b200 import workloads as wl

pytestmark = pytest.mark.gpu

EVERY = 10


def _analysis_oracle(w):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, 0, diameter=w.diameter, verts=w.verts, sweep_radius=w.sweep_radius)
    return o


def _summ(counters0, counters1):
    d = {k: counters1[k] - counters0[k] for k in counters1 if k != "sweep_counter"}
    nt = d["trans_acc"] + d["trans_rej_overlap"] + d["trans_rej_cell"]
    nr = d["rot_acc"] + d["rot_rej_overlap"]
    return d["trans_acc"] / max(nt, 1), (d["rot_acc"] / nr if nr else 0.0)


def run_oracle(w, seed, sweeps, pressure=True):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts, sweep_radius=w.sweep_radius)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    o.sweeps(sweeps // 10)
    c0 = o.counters()
    hist, ns = np.zeros(pr.NBINS), 0
    for _ in range((sweeps - sweeps // 10) // EVERY):
        o.sweeps(EVERY)
        if pressure:
            hist += o.scale_histogram(pr.S_MAX, pr.NBINS)
        ns += 1
    ta, ra = _summ(c0, o.counters())
    assert o.count_overlaps_cells() == 0
    return ta, ra, (pr.compressibility(hist, ns, w.N, w.dim) if pressure else 0.0)


def run_gpu(w, seed, sweeps, pressure=True):
    from paper_1509_04692_b200 import binding as hb
    g = hb.from_workload(w, seed=seed)
    an = _analysis_oracle(w)
    g.sweep(sweeps // 10)
    c0 = g.counters()
    hist, ns = np.zeros(pr.NBINS), 0
    for _ in range((sweeps - sweeps // 10) // EVERY):
        g.sweep(EVERY)
        if pressure:
            p, q = g.get_state()
            an.set_state(p, q)
            hist += an.scale_histogram(pr.S_MAX, pr.NBINS)
        ns += 1
    ta, ra = _summ(c0, g.counters())
    assert g.count_overlaps() == 0
    return ta, ra, (pr.compressibility(hist, ns, w.N, w.dim) if pressure else 0.0)


CASES = {
    "k0_disks": (lambda s: wl.config(0, seed=s), 400),
    "k1_pentagons": (lambda s: wl.config(1, seed=s), 600),
    "cubes_12": (lambda s: wl.cubes(12, seed=s), 200),
    # rounded shapes: acceptance only -- the touch scale of a rounded pair is a bisection (oracle), too slow for the
    # snapshots of 24 runs; the pressure estimator itself is shape-independent and pinned on the other cases
    "rounded_pentagons_24": (lambda s: wl.rounded_polygons(24, seed=s), 400),
    "rounded_cubes_6": (lambda s: wl.cubes(6, seed=s, edge=0.7, sweep_radius=0.15, d=0.15, a=0.3), 200),
}


@pytest.mark.parametrize("name", list(CASES))
def test_acceptance_and_pressure_within_3_standard_errors(name):
    make, sweeps = CASES[name]
    pressure = not name.startswith("rounded")
    seeds = list(range(1, 9))
    with ThreadPoolExecutor(8) as ex:       # the oracle is serial C; ctypes releases the GIL, one thread per seed
        fut = [ex.submit(run_oracle, make(s), s, sweeps, pressure) for s in seeds]
        gpu_same = np.array([run_gpu(make(s), s, sweeps, pressure) for s in seeds])
        gpu_indep = np.array([run_gpu(make(100 + s), 100 + s, sweeps, pressure) for s in seeds])
        orc = np.array([f.result() for f in fut])
    report = {}
    for label, gp in (("same seeds", gpu_same), ("independent seeds", gpu_indep)):
        for col, q in enumerate(("translate acceptance", "rotate acceptance", "beta P / rho")):
            mg, sg = pr.mean_and_se(gp[:, col])
            mo, so = pr.mean_and_se(orc[:, col])
            report[(label, q)] = (mg, sg, mo, so)
            if q == "beta P / rho" and not pressure:
                continue
            if q == "rotate acceptance" and mo == 0.0:
                assert mg == 0.0
                continue
            assert abs(mg - mo) <= 3.0 * np.hypot(sg, so) + 1e-12, (name, label, q, mg, sg, mo, so)
            assert so > 0 and so < 0.05 * abs(mo)     # the bar must have teeth: SE below 5 % of the value
    print(name, {k: tuple(round(x, 5) for x in v) for k, v in report.items()})


# ---- configs 2 and 4: the intensive-quantity check of O10 --------------------------------------------------------------
# Configs 1, 2 and 4 are the same state point (pentagons, phi = 0.594, same lattice recipe and moves), so beta P / rho -- an
# ensemble average whose finite-size shift O(1/N) is far below the error bar -- must agree within 3 standard errors between
# the CUDA path on 1 M / 16.8 M particles and the ORACLE on config 1's 4096, under one protocol: the same number of sweeps
# from the lattice start, the same discarded prefix, snapshots at the same sweep numbers (the melting transient is part of
# what is compared).  Protocols (50 sweeps per seed for config 2, 10 for config 4 on 1-2 seeds; 4 here).
#
# The ACCEPTANCE ratios are not intensive in that strict sense, contrary to what SURVEY.md O10 assumed: they depend on the
# cell grid, which differs between the configs (w / d_max = 1.0323 for L = 64, 1.0020 for L = 1024, 1.0010 for L = 4096).
# A translation is rejected outright when it leaves its cell, probability 1 - (1 - d / 2w)^2 (pinned in
# tests/test_oracle_sweep.py), and trials are dealt per CELL, so particles that share a cell get fewer each (R8/R9; seen in
# tests/test_oracle_textbook.py).  Checked instead: the translate acceptance divided by the closed-form stay probability
# (1 - d / 2w)^2 agrees within 1 %, the rotate acceptance within 0.5 % (measured residuals: 0.4 % and 0.1 %).
# (one snapshot of 4096 particles per seed is noisy: config 4's short protocol takes 32 oracle seeds to bring the SE below 2 %)
PROTOCOLS = {2: dict(discard=5, every=15, snapshots=3, gpu_seeds=8, oracle_seeds=8),
             4: dict(discard=1, every=9, snapshots=1, gpu_seeds=4, oracle_seeds=32)}


def _protocol_oracle(seed, discard, every, snapshots):
    w = wl.config(1, seed=seed)
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    o.sweeps(discard)
    c0 = o.counters()
    hist = np.zeros(pr.NBINS)
    for _ in range(snapshots):
        o.sweeps(every)
        hist += o.scale_histogram(pr.S_MAX, pr.NBINS)
    ta, ra = _summ(c0, o.counters())
    return ta, ra, pr.compressibility(hist, snapshots, w.N, w.dim)


def _protocol_gpu(k, seed, discard, every, snapshots, pool):
    from paper_1509_04692_b200 import binding as hb
    w = wl.config(k, seed=seed)
    g = hb.from_workload(w, seed=seed)
    g.sweep(discard)
    c0 = g.counters()
    futs = []
    for _ in range(snapshots):
        g.sweep(every)
        p, q = g.get_state()

        def analyse(p=p, q=q):          # the same fp64 analysis as for the oracle's snapshots, off the GPU thread
            an = _analysis_oracle(w)
            an.set_state(p, q)
            return an.scale_histogram(pr.S_MAX, pr.NBINS)
        futs.append(pool.submit(analyse))
    ta, ra = _summ(c0, g.counters())
    assert g.count_overlaps() == 0
    return ta, ra, futs, w


@pytest.mark.parametrize("k", [2, 4])
def test_large_pentagon_configs_reproduce_config1_oracle_within_3_standard_errors(k):
    pro = PROTOCOLS[k]
    args = (pro["discard"], pro["every"], pro["snapshots"])
    with ThreadPoolExecutor(8) as ex:
        fo = [ex.submit(_protocol_oracle, s, *args) for s in range(1, pro["oracle_seeds"] + 1)]
        runs = [_protocol_gpu(k, s, *args, ex) for s in range(1, pro["gpu_seeds"] + 1)]
        orc = np.array([f.result() for f in fo])
        gpu = []
        for ta, ra, futs, w in runs:
            hist = sum(f.result().astype(np.float64) for f in futs)
            gpu.append((ta, ra, pr.compressibility(hist, len(futs), w.N, w.dim)))
        gpu = np.array(gpu)
    report = {}
    for col, q in enumerate(("translate acceptance", "rotate acceptance", "beta P / rho")):
        mg, sg = pr.mean_and_se(gpu[:, col])
        mo, so = pr.mean_and_se(orc[:, col])
        report[q] = (mg, sg, mo, so)
    print(f"config {k} vs config 1 oracle", {q: tuple(round(x, 5) for x in v) for q, v in report.items()})
    mg, sg, mo, so = report["beta P / rho"]
    assert abs(mg - mo) <= 3.0 * np.hypot(sg, so), (k, report)
    assert 0 < so < 0.02 * abs(mo)                         # the bar has teeth: the oracle's SE is below 2 % of the value
    w1, wk = wl.config(1), runs[0][3]
    stay = lambda w, ncell: (1.0 - w.d / (2.0 * w.L[0] / ncell)) ** 2          # noqa: E731
    n1 = 2 * int(w1.L[0] / (2.0 * (1.0 + 1.0 / 1024.0)))   # R11 with d_max = 1
    nk = 2 * int(wk.L[0] / (2.0 * (1.0 + 1.0 / 1024.0)))
    tg, to = report["translate acceptance"][0] / stay(wk, nk), report["translate acceptance"][2] / stay(w1, n1)
    assert abs(tg / to - 1.0) < 0.01, (k, tg, to)
    assert abs(report["rotate acceptance"][0] / report["rotate acceptance"][2] - 1.0) < 0.005, (k, report)
