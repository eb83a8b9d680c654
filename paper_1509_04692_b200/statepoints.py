"""Harness-side preparation of the paper's own benchmark state points (S:8(f)-1, 8(f)-2) with the existing sweep:

  pentagons at area fraction phi = 0.676, move sizes tuned to 20 % acceptance, 65 536 per GPU
  dodecahedra at volume fraction phi = 0.5

The paper's equilibrated configurations are not available, so a state is produced from the lattice start of `workloads.py` by
NVT compression: shrink the box by a small factor, scale every centre with it, keep the step only if `hpmc_count_overlaps`
finds no overlapping pair (else halve the step), relax with a few sweeps, repeat until the target density is reached.  Then
the translation and rotation step sizes are adjusted until each is accepted at the target ratio ("move sizes are
tuned to 20 % acceptance").  Only library calls are made here (create / bind / set_moves / sweep / count_overlaps /
get_state): no new integrator, no arithmetic of the method.  The result is a `Workload` like any other, so the oracle can be
locked to it (tests/test_gpu_statepoints.py) and bench.py can time it.
"""
import dataclasses

import numpy as np

from . import binding as hb
from . import workloads as wl


def particle_volume(w):
    """Area (2-D) or volume (3-D) of one particle."""
    if w.kind == wl.KIND_DISK:
        return np.pi * 0.25 * w.diameter ** 2 if w.dim == 2 else np.pi / 6.0 * w.diameter ** 3
    v = np.asarray(w.verts, dtype=np.float64)
    if w.dim == 2:
        x, y = v[:, 0], v[:, 1]
        return 0.5 * abs(np.dot(x, np.roll(y, -1)) - np.dot(y, np.roll(x, -1)))
    from scipy.spatial import ConvexHull
    return float(ConvexHull(v).volume)


def packing_fraction(w):
    return w.N * particle_volume(w) / float(np.prod(w.L[: w.dim]))


def _scaled(w, f, pos4, quat4):
    p = pos4.copy()
    p[:, : w.dim] = (pos4[:, : w.dim].astype(np.float64) * f).astype(np.float32)
    L = tuple(float(np.float32(x * f)) for x in w.L)     # the library rounds the box edge to fp32 (R-box): scale to that value
    half = np.array([0.5 * np.float32(x) for x in L[: w.dim]], dtype=np.float32)
    # a centre that rounds onto the upper box face wraps to the lower one (coordinates live in [-L/2, L/2))
    for k in range(w.dim):
        hi = p[:, k] >= half[k]
        p[hi, k] -= np.float32(L[k])
        lo = p[:, k] < -half[k]
        p[lo, k] += np.float32(L[k])
    return dataclasses.replace(w, L=L, pos4=p, quat4=quat4.copy())


def compress(w, phi_target, seed=1, device="cuda:0", step=2e-3, relax_sweeps=10, melt_sweeps=100, max_steps=20000, log=None):
    """NVT compression of workload `w` to packing fraction `phi_target` on the GPU path.  Returns the new Workload."""
    g = hb.from_workload(w, seed=seed, device=device)
    assert g.count_overlaps() == 0
    g.sweep(melt_sweeps)
    cur = w
    taken = rejected = 0
    f_step = step
    while packing_fraction(cur) < phi_target * (1.0 - 1e-9) and taken + rejected < max_steps:
        pos4, quat4 = g.get_state()
        phi = packing_fraction(cur)
        # linear scale factor of this step, not beyond the target
        f = max(1.0 - f_step, (phi / phi_target) ** (1.0 / cur.dim))
        trial = _scaled(cur, f, pos4, quat4)
        gt = hb.from_workload(trial, seed=seed + 1 + taken + rejected, device=device)
        if gt.count_overlaps() == 0:
            cur, g = trial, gt
            g.sweep(relax_sweeps)
            taken += 1
            f_step = min(step, f_step * 1.5)
        else:
            rejected += 1
            f_step *= 0.5
            g.sweep(relax_sweeps)
            if f_step < 1e-7:
                raise RuntimeError(f"compression stalled at phi = {phi:.4f}")
        if log and (taken + rejected) % 500 == 0:
            log(f"compress: phi = {packing_fraction(cur):.4f} after {taken} steps ({rejected} rejected)")
    pos4, quat4 = g.get_state()
    assert g.count_overlaps() == 0
    out = dataclasses.replace(cur, pos4=pos4, quat4=quat4, name=f"{w.name}_phi{phi_target:.3f}", warmup_sweeps=20,
                              notes=f"compressed from the lattice start of {w.name} to phi = {packing_fraction(cur):.4f} in {taken} accepted "
                                    f"box steps ({rejected} rejected); stands in for the paper's equilibrated state (P:183)")
    return out


def tune_moves(w, target=0.2, seed=1, device="cuda:0", rounds=12, sweeps=40, log=None):
    """Adjust d and a until translations and rotations are each accepted at `target`.  Returns the new Workload
    (state advanced by the tuning sweeps) and the measured acceptances of the last round.  The rotation step is capped (see
    a_max): nearly round or highly symmetric particles accept more than `target` of their rotations at any step size."""
    d, a = w.d, w.a
    g = hb.from_workload(w, seed=seed, device=device)
    d_max_move = 0.5 * float(min(g.w[: w.dim]))          # a larger translation mostly leaves its cell
    # rotation steps: at most half the symmetry angle of an n-gon (beyond it larger steps are accepted MORE often), 1 rad in 3-D
    a_max = float(np.pi / w.verts.shape[0]) if (w.kind == wl.KIND_POLYGON) else 1.0
    acc_t = acc_r = 0.0
    for r in range(rounds):
        g.set_moves(d, a if w.kind != wl.KIND_DISK else 0.0, w.n_select)
        g.reset_counters()
        g.sweep(sweeps)
        c = g.counters()
        nt = c["trans_acc"] + c["trans_rej_overlap"] + c["trans_rej_cell"]
        nr = c["rot_acc"] + c["rot_rej_overlap"]
        acc_t = c["trans_acc"] / max(nt, 1)
        acc_r = c["rot_acc"] / nr if nr else target
        if log:
            log(f"tune round {r}: d = {d:.4f} acc {acc_t:.3f}; a = {a:.4f} acc {acc_r:.3f}")
        if abs(acc_t - target) < 0.01 and (abs(acc_r - target) < 0.01 or (a >= a_max and acc_r > target)):
            break
        # acceptance falls roughly exponentially with the step size: scale the step by log(target) / log(acceptance)
        d = float(np.clip(d * np.clip(np.log(target) / np.log(np.clip(acc_t, 1e-3, 0.999)), 0.5, 2.0), 1e-4, d_max_move))
        if nr:
            a = float(np.clip(a * np.clip(np.log(target) / np.log(np.clip(acc_r, 1e-3, 0.999)), 0.5, 2.0), 1e-4, a_max))
    pos4, quat4 = g.get_state()
    assert g.count_overlaps() == 0
    out = dataclasses.replace(w, d=d, a=a, pos4=pos4, quat4=quat4, name=w.name + "_tuned")
    return out, (acc_t, acc_r)


def replicate(w, reps, phi_target, seed=1, device="cuda:0", decorrelate_sweeps=200):
    """Tile `reps`^dim periodic copies of an overlap-free configuration into a box `reps` times larger -- overlap-free by
    periodicity -- expanding it on the way from its own density to `phi_target` (slightly lower), which keeps every gap above
    the fp32 rounding of the larger coordinates; then run sweeps so that the copies drift apart (each cell has its own Philox
    stream).  An affine compression of the large system itself stalls: among 10^5 pairs some gap is always ~1/N."""
    phi = packing_fraction(w)
    assert phi >= phi_target
    f = (phi / phi_target) ** (1.0 / w.dim)
    L0 = np.array(w.L[: w.dim], dtype=np.float64) * f
    base = w.pos4[:, : w.dim].astype(np.float64) * f
    shifts = np.stack(np.meshgrid(*[np.arange(reps)] * w.dim, indexing="ij"), axis=-1).reshape(-1, w.dim)
    pos = np.zeros((w.N * len(shifts), 4), dtype=np.float32)
    quat = np.tile(w.quat4, (len(shifts), 1))
    for t, sh in enumerate(shifts):
        pos[t * w.N:(t + 1) * w.N, : w.dim] = (base + (sh - 0.5 * (reps - 1)) * L0).astype(np.float32)
    L = tuple(float(np.float32(x)) for x in (reps * L0))
    big = dataclasses.replace(w, N=pos.shape[0], L=L, pos4=pos, quat4=quat, name=f"{w.name}_x{reps ** w.dim}")
    half = [0.5 * np.float32(x) for x in L]
    for k in range(w.dim):   # a centre rounded onto the upper face belongs to the lower one
        hi = big.pos4[:, k] >= half[k]
        big.pos4[hi, k] -= np.float32(L[k])
    g = hb.from_workload(big, seed=seed, device=device)
    assert g.count_overlaps() == 0, "replicated configuration overlaps"
    g.sweep(decorrelate_sweeps)
    pos4, quat4 = g.get_state()
    assert g.count_overlaps() == 0
    return dataclasses.replace(big, pos4=pos4, quat4=quat4, notes=w.notes + f"; {reps}^{w.dim} periodic copies, {decorrelate_sweeps} sweeps apart")


def pentagons_paper_state(n_lat=256, seed=1, device="cuda:0", log=None):
    """Pentagons at phi = 0.676 with move sizes tuned to 20 % acceptance; n_lat = 256 is the paper's 65 536 per GPU.
    Systems above 64 x 64 are compressed at 64 x 64 and replicated."""
    base = min(n_lat, 64)
    reps = n_lat // base
    assert base * reps == n_lat
    w = compress(wl.pentagons(base, seed=seed, name=f"pentagons_{base * base}"), 0.676 * (1.0 + (2e-4 if reps > 1 else 0.0)), seed=seed,
                 device=device, log=log)
    if reps > 1:
        w = replicate(w, reps, 0.676, seed=seed, device=device)
    return tune_moves(w, 0.2, seed=seed, device=device, log=log)


def dodecahedra_paper_state(n_lat=16, seed=1, device="cuda:0", log=None):
    """Regular dodecahedra (circumradius 0.5) at phi = 0.5, move sizes tuned to 20 % acceptance (rotations: the step is
    capped at 1 rad, where these nearly spherical particles still accept ~30 %).  Above 8^3 particles: compressed at 8^3 and replicated."""
    base = min(n_lat, 8)
    reps = n_lat // base
    assert base * reps == n_lat
    w0 = wl.polyhedra(wl.dodecahedron_vertices(0.5), base, 1.04, seed=seed, name=f"dodecahedra_{base ** 3}")
    w = compress(w0, 0.5 * (1.0 + (3e-4 if reps > 1 else 0.0)), seed=seed, device=device, step=4e-3, log=log)
    if reps > 1:
        w = replicate(w, reps, 0.5, seed=seed, device=device, decorrelate_sweeps=50)
    return tune_moves(w, 0.2, seed=seed, device=device, log=log)
