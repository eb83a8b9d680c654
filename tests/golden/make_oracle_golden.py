"""Writes tests/golden/oracle_golden.json.  Calls ONLY oracle/ and the seeded input generators.

Run from the repo root:  python tests/golden/make_oracle_golden.py
The stored values freeze the oracle's trajectory (counters + a hash of the fp32 state) on three small
systems so that any later change to the oracle's arithmetic is visible in review; they are NOT taken
from the CUDA path.  A change here must name the PAPER.md passage / DESIGN.md reading that justifies it.
"""
import hashlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import hpmc_oracle as ho  # noqa: E402
from paper_1509_04692_b200 import workloads as wl  # noqa: E402

CASES = {"disks16": (lambda: wl.disks(16), 20), "pentagons16": (lambda: wl.pentagons(16), 20),
         "cubes6": (lambda: wl.cubes(6), 5)}


def run(name):
    mk, n = CASES[name]
    w = mk()
    o = ho.Oracle(w.dim, w.L, w.kind, w.N, 1, diameter=w.diameter, verts=w.verts)
    o.set_moves(w.d, w.a, w.n_select)
    o.set_state(w.pos4, w.quat4)
    o.sweeps(n)
    p, q = o.get_state()
    return {"sweeps": n, "counters": o.counters(), "pos_sha256": hashlib.sha256(p.tobytes()).hexdigest(),
            "quat_sha256": hashlib.sha256(q.tobytes()).hexdigest(), "header_t3": [o.sweep_header(3)[0].tolist(),
                                                                                   o.sweep_header(3)[1].tolist()]}


if __name__ == "__main__":
    out = {k: run(k) for k in CASES}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_golden.json"), "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
    print(json.dumps(out, indent=1, sort_keys=True))
