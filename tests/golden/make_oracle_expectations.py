"""Writes tests/golden/oracle_expectations.json from the ORACLE ALONE (imports only oracle/ and the input generators).

  python tests/golden/make_oracle_expectations.py            # ~25 min on 8 cores (config 3 at full size dominates)

Two groups of numbers, each the mean and standard error over the 8 seeds 1..8 of BASELINE.json's parity bar:

 "full_runs":  per state point, the translate / rotate acceptance accumulated from the LATTICE START over the first
               100 / 1000 / 10^4 sweeps -- the run lengths BASELINE.json quotes (configs[4] / [2], [0], [3] / [1]) -- on
               the 4096-particle configs 0 and 1 and the full 32 768-cube config 3.  tests/test_gpu_full_runs.py compares
               the CUDA path's full-length runs with these (configs 2 and 4 share config 1's state point: acceptance is
               intensive, the finite-size shift O(1/N) is below the tolerance used there).
 "stationary": acceptance and beta P / rho (O9) after discarding the first 10 % of 600 / 400 sweeps (O10's protocol) for
               configs 1 and 0: the values tests/test_gpu_statistics.py checks configs 2 and 4 against.
 "work":       O7 per-trial work in early-exit serial order on the melted state (candidates scanned, narrow tests, separating
               axes per polygon test, GJK support calls per polyhedron test): the inputs of bench.py's flop tariff.
"""
import json
import os
import sys
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import hpmc_oracle as ho          # noqa: E402
from oracle import pressure as pr             # noqa: E402
from paper_1509_04692_b200 import workloads as wl   # noqa: E402  (seeded input generators only)

SEEDS = list(range(1, 9))
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_expectations.json")


def make(w, seed):
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    return o


def acc(c):
    nt = c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"]
    nr = c["rot_acc"] + c["rot_rej_overlap"]
    return c["trans_acc"] / max(nt, 1), (c["rot_acc"] / nr if nr else 0.0)


def full_run(k, seed, checkpoints):
    o = make(wl.config(k, seed=seed), seed)
    out, done = {}, 0
    for cp in checkpoints:
        o.sweeps(cp - done)
        done = cp
        out[cp] = acc(o.counters())
    assert o.count_overlaps_cells() == 0
    return out


def stationary(k, seed, sweeps):
    w = wl.config(k, seed=seed)
    o = make(w, seed)
    o.sweeps(sweeps // 10)
    o.reset_counters()
    hist, ns = np.zeros(pr.NBINS), 0
    for _ in range((sweeps - sweeps // 10) // 10):
        o.sweeps(10)
        hist += o.scale_histogram(pr.S_MAX, pr.NBINS)
        ns += 1
    ta, ra = acc(o.counters())
    return ta, ra, pr.compressibility(hist, ns, w.N, w.dim)


def work(w, melt, sweeps):
    o = make(w, 1)
    o.sweeps(melt)
    o.set_work_detail(True)
    o.reset_counters()
    o.sweeps(sweeps)
    wk, c = o.work(), o.counters()
    nt = max(wk["narrow_tests_early"], 1)
    return {"sample": f"{w.name}, {sweeps} sweeps after {melt} melt sweeps", "trials": c["trials"],
            "candidates_scanned_per_trial": wk["cand_scanned_early"] / c["trials"],
            "candidates_scanned_per_trial_no_early_exit": wk["cand_scanned_full"] / c["trials"],
            "narrow_tests_per_trial": wk["narrow_tests_early"] / c["trials"],
            "narrow_tests_per_trial_no_early_exit": wk["sphere_pass_full"] / c["trials"],
            "polygon_axes_per_narrow_test": wk["polygon_axes_early"] / nt,
            "gjk_support_calls_per_narrow_test": wk["gjk_support_calls_early"] / nt,
            "rotate_fraction": (c["rot_acc"] + c["rot_rej_overlap"]) / c["trials"]}


def ms(values):
    m, s = pr.mean_and_se(values)
    return {"mean": m, "se": s}


def main():
    plan_full = {3: [100, 1000], 1: [100, 1000, 10000], 0: [100, 1000]}      # longest first
    res = {"seeds": SEEDS, "full_runs": {}, "stationary": {}, "work": {}}
    with ThreadPoolExecutor(os.cpu_count() or 8) as ex:                       # ctypes releases the GIL
        fut_full = {k: [ex.submit(full_run, k, s, cps) for s in SEEDS] for k, cps in plan_full.items()}
        fut_stat = {k: [ex.submit(stationary, k, s, n) for s in SEEDS] for k, n in ((1, 600), (0, 400))}
        res["work"] = {"k0_disks": work(wl.config(0), 200, 20), "k1_pentagons": work(wl.config(1), 200, 20),
                       "k3_cubes": work(wl.cubes(12), 100, 10)}
        for k, futs in fut_stat.items():
            v = np.array([f.result() for f in futs])
            res["stationary"][f"k{k}"] = {"translate_acceptance": ms(v[:, 0]), "rotate_acceptance": ms(v[:, 1]), "betaP_over_rho": ms(v[:, 2])}
        for k, futs in fut_full.items():
            runs = [f.result() for f in futs]
            res["full_runs"][f"k{k}"] = {str(cp): {"translate_acceptance": ms([r[cp][0] for r in runs]),
                                                   "rotate_acceptance": ms([r[cp][1] for r in runs])} for cp in plan_full[k]}
            json.dump(res, open(OUT, "w"), indent=1)
    json.dump(res, open(OUT, "w"), indent=1)
    print(json.dumps(res, indent=1))


if __name__ == "__main__":
    main()
