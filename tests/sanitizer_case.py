"""Small driver for compute-sanitizer (run by hand on a GPU box; not collected by pytest):

    compute-sanitizer --tool racecheck python tests/sanitizer_case.py
    compute-sanitizer --tool memcheck  python tests/sanitizer_case.py

A few sweeps of small systems through every colour-pass variant -- 2-D tile pass (one launch per colour and the persistent
dataflow launch with its ticket / stamp protocol), warp-per-cell pass in 2-D and 3-D (polygon SAT, fp32 GJK + fp64 re-run),
the thread-block-cluster pass, the per-thread path -- and through both cell-list builds, the validator and the un-sort.
profiles/r2_sanitizer.md records the results."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from paper_1509_04692_b200 import binding as hb          # noqa: E402
from paper_1509_04692_b200 import workloads as wl        # noqa: E402

CASES = [(wl.pentagons(40), [{"path": 2}, {"path": 2, "flow": 1}, {"tile_shape": 1, "flow": 1}, {"path": 3}, {"path": 4}, {"path": 1},
                             {"small_build": 0, "path": 2}]),
         (wl.disks(40), [{"path": 2, "flow": 1}, {"path": 3}, {"path": 4}]),
         (wl.cubes(6), [{}, {"path": 1}]),
         (wl.cubes(7, spacing=1.0006, max_tilt=2e-4, d=3e-4, a=3e-4), [{}])]
for w, optsets in CASES:
    for opts in optsets:
        g = hb.from_workload(w, seed=1)
        for k, v in opts.items():
            g.set_option(k, v)
        g.sweep(1)
        g.sweep(3)
        n = g.count_overlaps()
        g.get_state()
        print(w.name, opts, g.describe_pass()[:48], "trials", g.counters()["trials"], "overlaps", n, flush=True)
        assert n == 0
print("sanitizer case done")
