"""Writes tests/golden/pentagons_1024_phi0676.npz from the ORACLE ALONE (imports only oracle/ and the input generators):

  python tests/golden/make_dense_pentagons.py            # a few minutes on 8 cores

1024 regular pentagons (circumradius 0.5) compressed from the seeded 32 x 32 lattice start (phi = 0.594) to the paper's
benchmark density phi = 0.676 by NVT compression with the oracle's own sweeps: shrink the box by a small factor,
scale the centres, keep the step only if the oracle's O(N^2) brute-force overlap count is zero, relax, repeat; then the move
sizes are tuned towards 20 % acceptance (the rotation step is capped at half the pentagon's symmetry angle).  The
file holds pos4, quat4 (fp32), the box edge and d, a: the INPUT of tests/test_gpu_statepoints.py's lock-step at that density.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import hpmc_oracle as ho                    # noqa: E402
from paper_1509_04692_b200 import workloads as wl       # noqa: E402  (seeded input generators only)

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "pentagons_1024_phi0676.npz")
PHI, AREA = 0.676, 2.5 * 0.25 * np.sin(2.0 * np.pi / 5.0)


def make(L, pos, quat, d, a, seed):
    o = ho.Oracle(2, (L, L), ho.KIND_POLYGON, pos.shape[0], seed, verts=wl.regular_polygon(5, 0.5))
    o.set_moves(d, a, 4)
    o.set_state(pos, quat)
    o.set_threads(os.cpu_count() or 1)
    return o


def main():
    w = wl.pentagons(32, seed=1)
    L, pos, quat, d, a = float(w.L[0]), w.pos4.copy(), w.quat4.copy(), 0.1, 0.1
    o = make(L, pos, quat, d, a, 1)
    o.sweeps(100)
    step, n = 2e-3, 0
    while w.N * AREA / (L * L) < PHI * (1 - 1e-9):
        pos, quat = o.get_state()
        phi = w.N * AREA / (L * L)
        f = max(1.0 - step, np.sqrt(phi / PHI))
        Lt = float(np.float32(L * f))
        pt = pos.copy()
        pt[:, :2] = (pos[:, :2].astype(np.float64) * f).astype(np.float32)
        half = np.float32(0.5) * np.float32(Lt)
        pt[:, :2] = np.where(pt[:, :2] >= half, pt[:, :2] - np.float32(Lt), pt[:, :2])
        n += 1
        t = make(Lt, pt, quat, d, a, 1 + n)
        if t.count_overlaps_bruteforce() == 0:
            o, L = t, Lt
            step = min(2e-3, step * 1.5)
        else:
            step *= 0.5
            assert step > 1e-7, "compression stalled"
        o.sweeps(10)
        if n % 100 == 0:
            print(f"step {n}: phi = {w.N * AREA / (L * L):.4f}", flush=True)
    a_max = np.pi / 5.0
    for r in range(10):                                   # move sizes towards 20 % acceptance
        o.set_moves(d, a, 4)
        o.reset_counters()
        o.sweeps(40)
        c = o.counters()
        at = c["trans_acc"] / (c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"])
        ar = c["rot_acc"] / (c["rot_acc"] + c["rot_rej_overlap"])
        print(f"tune {r}: d = {d:.4f} ({at:.3f}), a = {a:.4f} ({ar:.3f})", flush=True)
        d = float(np.clip(d * np.clip(np.log(0.2) / np.log(at), 0.5, 2.0), 1e-4, 0.45))
        a = float(np.clip(a * np.clip(np.log(0.2) / np.log(ar), 0.5, 2.0), 1e-4, a_max))
    pos, quat = o.get_state()
    assert o.count_overlaps_bruteforce() == 0
    np.savez_compressed(OUT, pos4=pos, quat4=quat, L=np.float64(L), d=np.float64(d), a=np.float64(a),
                        acceptance=np.array([at, ar]), phi=np.float64(w.N * AREA / (L * L)))
    print("wrote", OUT, "phi", w.N * AREA / (L * L), "d", d, "a", a)


if __name__ == "__main__":
    main()
