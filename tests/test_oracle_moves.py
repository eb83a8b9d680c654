"""Pins for the oracle's move generators and sweep header (R4-R7, R10, R12; "q_trial = q_i . dq",
P:243 "the proper uniform distribution").

The rotation generator is driven through the public sweep on isolated particles (every rotation is accepted), and the
increment dq = q^-1 (x) q' is recovered with this file's own quaternion algebra.  Two kinds of pin:

  * per trial, against the reading R6 evaluated by independent AXIS-ANGLE algebra (not a quaternion product): the random
    words of the trial come from the KAT-pinned Philox with the counter layout R3; the recovered body-frame increment
    must be the rotation by theta = a usym(uc) about (rho cos phi, rho sin phi, z), z = usym(ua), phi = 2 pi u01(ub);
  * distributions: |theta| uniform on [0, a), axis isotropic on S^2 (z-marginal and azimuth uniform), 2-D axis = +-z.

Deliberate breaks of oracle/hpmc_oracle.c that were tried and make these tests fail (each restored afterwards):
  gen_rotate, 3-D: `h = theta` instead of `0.5 * theta` -> test_rotation_3d_per_trial (angle) and _distribution (KS);
  gen_rotate, 3-D: `rho = 1.0`                          -> test_rotation_3d_per_trial (axis not unit / wrong direction);
  gen_rotate: `quat_mul(dq, qd, qn)` (left product)     -> test_rotation_3d_per_trial (body-frame axis mismatch);
  gen_rotate, 2-D: `dq[3] = sin(2 h)`                   -> test_rotation_2d (angle);
  orc_sweep_header: `(uint64_t)i` instead of `(i + 1)`  -> test_colour_permutation_is_uniform (identity never drawn);
  orc_sweep_header: shift from `r[0]` for every axis    -> test_grid_shift_is_uniform (x-y correlation);
  orc_sweep_header: `s->w_f[k] * 0.5f * orc_u01`        -> test_grid_shift_is_uniform (range).
"""
import numpy as np
import pytest
from scipy import stats

from oracle import hpmc_oracle as ho

TAG_TRIAL = 3


def qmul(a, b):
    """Hamilton product, arrays (..., 4) in (w, x, y, z) order."""
    aw, ax, ay, az = np.moveaxis(a, -1, 0)
    bw, bx, by, bz = np.moveaxis(b, -1, 0)
    return np.stack([aw * bw - ax * bx - ay * by - az * bz, aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx, aw * bz + ax * by - ay * bx + az * bw], axis=-1)


def qconj(a):
    return a * np.array([1.0, -1.0, -1.0, -1.0])


def random_unit_quats(rng, n):
    q = rng.normal(size=(n, 4))
    return q / np.linalg.norm(q, axis=1, keepdims=True)


CUBE = np.array([[x, y, z] for x in (-.5, .5) for y in (-.5, .5) for z in (-.5, .5)])
PENTAGON = np.array([[0.5 * np.cos(2 * np.pi * k / 5), 0.5 * np.sin(2 * np.pi * k / 5)] for k in range(5)])


def isolated_system(dim, m, a, seed):
    """m^dim particles 10 apart: no trial can ever overlap, so every rotation is accepted; one trial per cell and sweep."""
    L = 10.0 * m
    idx = np.stack(np.meshgrid(*[np.arange(m)] * dim, indexing="ij"), axis=-1).reshape(-1, dim)
    N = idx.shape[0]
    pos = np.zeros((N, 4), np.float32)
    pos[:, :dim] = (idx + 0.5) * 10.0 - L / 2
    if dim == 3:
        o = ho.Oracle(3, (L,) * 3, ho.KIND_POLYHEDRON, N, seed, verts=CUBE)
    else:
        o = ho.Oracle(2, (L,) * 2, ho.KIND_POLYGON, N, seed, verts=PENTAGON)
    o.set_moves(0.05, a, 1)
    return o, pos, N


def collect_rotations(dim, m, a, seed, sweeps, tilt=True):
    """Returns per accepted rotation trial: q0 (fp64 of the fp32 input), q1 (fp64 of the fp32 result), words (ua, ub, uc)."""
    o, pos, N = isolated_system(dim, m, a, seed)
    rng = np.random.default_rng(seed)
    out_q0, out_q1, out_u = [], [], []
    for t in range(sweeps):
        if dim == 3:
            q0 = random_unit_quats(rng, N) if tilt else np.tile([1.0, 0, 0, 0], (N, 1))
        else:
            th = rng.uniform(0, 2 * np.pi, N)
            q0 = np.stack([np.cos(th / 2), 0 * th, 0 * th, np.sin(th / 2)], axis=1)
        q0 = q0.astype(np.float32)
        o.set_state(pos, q0)
        assert o.sweep_counter == t
        shift, _ = o.sweep_header(t)
        r = o.sweep(want_trace=True)
        tr = r["trace"]
        _, q1 = o.get_state()
        slots = np.nonzero((tr[:, 1] >> 8) != 0)[0]           # n_select = 1: slot = cell id
        for cell in slots:
            i, word1 = int(tr[cell, 0]), int(tr[cell, 1])
            if (word1 & 0xFF) != 1:
                continue                                     # a translation
            assert (word1 >> 8) == 1, "an isolated particle's rotation must be accepted"
            assert o.cell_of(pos[i, :3], shift) == cell
            # R3: ctr = (cell, t_lo, k | block << 16, TAG_TRIAL << 24 | gamma << 16 | t_hi16), key = (seed, 0)
            n0, n1 = int(o.n[0]), int(o.n[1])
            cx, cy, cz = cell % n0, (cell // n0) % n1, cell // (n0 * n1)
            gamma = (cx & 1) | ((cy & 1) << 1) | ((cz & 1) << 2)
            c3 = (TAG_TRIAL << 24) | (gamma << 16)
            b0 = ho.philox4x32_10([cell, t, 0, c3], [seed, 0])
            b1 = ho.philox4x32_10([cell, t, 1 << 16, c3], [seed, 0]) if dim == 3 else [0, 0, 0, 0]
            assert int(b0[1]) >> 31 == 1                      # R7: top bit of word 1 set <=> rotation
            out_q0.append(q0[i].astype(np.float64)); out_q1.append(q1[i].astype(np.float64))
            out_u.append((int(b0[2]), int(b0[3]), int(b1[0])))
        pos = pos.copy()                                     # positions are reset too (translations moved some)
    return np.array(out_q0), np.array(out_q1), out_u


def test_rotation_3d_per_trial_matches_reading_R6_and_is_a_right_product():
    a = 0.4
    q0, q1, words = collect_rotations(3, 3, a, seed=11, sweeps=60)
    assert len(words) > 500
    assert np.max(np.abs(np.linalg.norm(q1, axis=1) - 1.0)) < 2e-7            # renormalised on store
    dq_body = qmul(qconj(q0), q1)                                             # q' = q (x) dq
    dq_world = qmul(q1, qconj(q0))                                            # q' = dq (x) q   (the wrong side)
    bad_world = 0
    for n, (ua, ub, uc) in enumerate(words):
        z = ho.usym(ua)
        phi = 2.0 * np.pi * ho.u01(ub)
        rho = np.sqrt(1.0 - z * z)
        axis = np.array([rho * np.cos(phi), rho * np.sin(phi), z])
        theta = float(np.float32(a) * np.float32(ho.usym(uc)))
        w, v = dq_body[n, 0], dq_body[n, 1:]
        theta_rec = 2.0 * np.arctan2(np.dot(v, axis), w)                      # signed angle about the expected axis
        assert abs(theta_rec - theta) < 2e-6, (n, theta_rec, theta)
        assert np.linalg.norm(np.cross(v, axis)) < 2e-6                       # and about no other axis
        assert abs(np.linalg.norm(v) - abs(np.sin(theta / 2))) < 2e-6
        vw = dq_world[n, 1:]
        bad_world += np.linalg.norm(np.cross(vw, axis)) > 1e-3 * abs(np.sin(theta / 2)) + 2e-6
    assert bad_world > 0.9 * len(words)        # for tilted q the world-frame increment has a different axis


def test_rotation_3d_distribution_uniform_angle_and_isotropic_axis():
    a = 0.5
    q0, q1, words = collect_rotations(3, 3, a, seed=5, sweeps=700)
    assert len(words) > 8000
    dq = qmul(qconj(q0), q1)
    dq = np.where(dq[:, :1] < 0, -dq, dq)                                     # same rotation, w >= 0
    v = dq[:, 1:]
    half = np.arctan2(np.linalg.norm(v, axis=1), dq[:, 0])                    # |theta| / 2
    ang = 2.0 * half
    assert ang.max() < a + 1e-6
    assert stats.kstest(ang / a, "uniform").pvalue > 1e-3                     # |theta| uniform on [0, a)
    ax = v / np.linalg.norm(v, axis=1, keepdims=True)
    # (theta, axis) and (-theta, -axis) are one rotation: fold the sign with an independent coin to test isotropy
    coin = np.random.default_rng(1).integers(0, 2, len(ax)) * 2 - 1
    ax = ax * coin[:, None]
    assert stats.kstest((ax[:, 2] + 1) / 2, "uniform").pvalue > 1e-3          # z-marginal uniform on [-1, 1] (Archimedes)
    az = np.mod(np.arctan2(ax[:, 1], ax[:, 0]), 2 * np.pi) / (2 * np.pi)
    assert stats.kstest(az, "uniform").pvalue > 1e-3                          # azimuth uniform
    assert stats.kstest((ax[:, 0] + 1) / 2, "uniform").pvalue > 1e-3          # and so is any other component
    assert np.all(np.abs(ax.mean(axis=0)) < 4 * np.sqrt(1 / 3 / len(ax)))


def test_rotation_2d_angle_uniform_about_z():
    a = 0.3
    q0, q1, words = collect_rotations(2, 4, a, seed=9, sweeps=900)
    assert len(words) > 6000
    assert np.all(q1[:, 1:3] == 0.0)                                          # R30: x and y components stay exactly 0
    dq = qmul(qconj(q0), q1)
    theta_rec = 2.0 * np.arctan2(dq[:, 3], dq[:, 0])
    theta = np.array([float(np.float32(a) * np.float32(ho.usym(ua))) for ua, _, _ in words])
    assert np.max(np.abs(theta_rec - theta)) < 2e-6                           # R6, 2-D: theta = a usym(ua) about +z
    assert theta_rec.min() >= -a - 1e-6 and theta_rec.max() < a + 1e-6
    assert stats.kstest((theta_rec + a) / (2 * a), "uniform").pvalue > 1e-3   # uniform on [-a, a)
    # orientation angle itself advances by theta (right and left products coincide for a common axis)
    t0 = 2.0 * np.arctan2(q0[:, 3], q0[:, 0]); t1 = 2.0 * np.arctan2(q1[:, 3], q1[:, 0])
    assert np.max(np.abs(np.angle(np.exp(1j * (t1 - t0 - theta))))) < 5e-6


def chi2_p(counts, expected):
    counts = np.asarray(counts, dtype=np.float64)
    x2 = ((counts - expected) ** 2 / expected).sum()
    return stats.chi2.sf(x2, counts.size - 1)


def test_colour_permutation_is_uniform():
    # R12: a fresh uniform random permutation of the 2^d colours per sweep (Fisher-Yates)
    T = 24000
    o2 = ho.Oracle(2, (8.0, 8.0), ho.KIND_DISK, 0, 3, diameter=1.0)
    seen = {}
    for t in range(T):
        _, perm = o2.sweep_header(t)
        seen[tuple(perm.tolist())] = seen.get(tuple(perm.tolist()), 0) + 1
    assert len(seen) == 24                                                    # all 4! orders occur
    assert chi2_p(list(seen.values()), T / 24) > 1e-3
    o3 = ho.Oracle(3, (8.0,) * 3, ho.KIND_DISK, 0, 4, diameter=1.0)
    table = np.zeros((8, 8))
    first_two = np.zeros((8, 8))
    for t in range(T):
        _, perm = o3.sweep_header(t)
        assert sorted(perm.tolist()) == list(range(8))
        table[np.arange(8), perm] += 1                                        # colour at each position
        first_two[perm[0], perm[1]] += 1
    for pos in range(8):
        assert chi2_p(table[pos], T / 8) > 1e-4, pos                          # every position marginal uniform
    off = first_two[~np.eye(8, dtype=bool)]
    assert chi2_p(off, T / 56) > 1e-3                                         # ordered pairs (first, second) uniform over 56
    # successive sweeps are independent draws: the first colour of sweep t+1 does not depend on that of sweep t
    o2b = ho.Oracle(2, (8.0, 8.0), ho.KIND_DISK, 0, 5, diameter=1.0)
    firsts = np.array([o2b.sweep_header(t)[1][0] for t in range(T)])
    joint = np.zeros((4, 4))
    np.add.at(joint, (firsts[:-1], firsts[1:]), 1)
    assert chi2_p(joint.ravel(), (T - 1) / 16) > 1e-3


def test_grid_shift_is_uniform_on_the_cell():
    # R10: s_k = w_k u01(r_k), uniform on [0, w_k), axes independent, fresh each sweep
    T = 30000
    o = ho.Oracle(3, (9.0, 13.0, 17.0), ho.KIND_DISK, 0, 7, diameter=1.0)     # three different cell widths
    s = np.array([o.sweep_header(t)[0] for t in range(T)], dtype=np.float64)
    w = o.w
    assert np.all(s >= 0) and np.all(s < w[None, :])
    u = s / w[None, :]
    for k in range(3):
        assert u[:, k].max() > 0.999 and u[:, k].min() < 0.001                # the whole cell width is used
        assert stats.kstest(u[:, k], "uniform").pvalue > 1e-3
    for k, l in ((0, 1), (0, 2), (1, 2)):                                     # pairwise independent
        h, _, _ = np.histogram2d(u[:, k], u[:, l], bins=6, range=[[0, 1], [0, 1]])
        assert chi2_p(h.ravel(), T / 36) > 1e-3
        assert abs(np.corrcoef(u[:, k], u[:, l])[0, 1]) < 4 / np.sqrt(T)
    assert abs(np.corrcoef(u[:-1, 0], u[1:, 0])[0, 1]) < 4 / np.sqrt(T)       # and from sweep to sweep
    o2 = ho.Oracle(2, (9.0, 9.0), ho.KIND_DISK, 0, 7, diameter=1.0)
    assert o2.sweep_header(5)[0][2] == 0.0                                    # no z shift in 2-D


def test_select_and_move_type_are_uniform():
    # R7/R8: member floor(sel n / 2^32) uniform over the cell's members; translate/rotate 50/50 from the top bit of word 1
    L = 8.0
    o = ho.Oracle(2, (L, L), ho.KIND_POLYGON, 3, 2, verts=PENTAGON)           # three pentagons on top of each other: every trial is rejected,
    # but the trace still records which member was picked and the move type
    pos = np.zeros((3, 4), np.float32)
    pos[:, 0] = [-0.3, 0.0, 0.3]
    quat = np.zeros((3, 4), np.float32); quat[:, 0] = 1
    o.set_moves(1e-4, 1e-4, 64)
    picks = np.zeros(3); rot = 0; n = 0
    for t in range(400):
        o.set_state(pos, quat)
        shift, _ = o.sweep_header(t)
        cells = [o.cell_of(pos[i, :3], shift) for i in range(3)]
        if len(set(cells)) != 1:
            o.sweep()
            continue
        tr = o.sweep(want_trace=True)["trace"]
        sl = tr[(tr[:, 1] >> 8) != 0]
        assert len(sl) == 64
        picks += np.bincount(sl[:, 0].astype(int), minlength=3)
        rot += int(np.sum(sl[:, 1] & 0xFF)); n += 64
    assert n > 10000
    assert chi2_p(picks, n / 3) > 1e-3
    assert abs(rot / n - 0.5) < 4 * 0.5 / np.sqrt(n)


def test_work_counters_polygon_axes_and_gjk_support_calls():
    # O7: axes evaluated up to the first separating axis; GJK support calls.  Closed-form checks on two-particle systems.
    L = 12.0
    o = ho.Oracle(2, (L, L), ho.KIND_POLYGON, 2, 1, verts=PENTAGON)
    o.set_work_detail(True)
    o.set_moves(1e-6, 1e-6, 1)
    quat = np.zeros((2, 4), np.float32); quat[:, 0] = 1
    pos = np.zeros((2, 4), np.float32); pos[1, 0] = 0.95                      # B along +x of A: A's normal 0 (angle 36 deg) ...
    o.set_state(pos, quat)
    for _ in range(20):
        o.set_state(pos, quat); o.sweep()
    wk = o.work()
    assert wk["narrow_tests_early"] > 0
    per = wk["polygon_axes_early"] / wk["narrow_tests_early"]
    assert 1.0 <= per <= 10.0
    # a pair that certainly overlaps evaluates all 2n = 10 axes
    o2 = ho.Oracle(2, (L, L), ho.KIND_POLYGON, 2, 1, verts=PENTAGON)
    o2.set_work_detail(True); o2.set_moves(1e-6, 1e-6, 1)
    pos2 = pos.copy(); pos2[1, 0] = 0.5
    o2.set_state(pos2, quat); o2.sweep()
    wk2 = o2.work()
    assert wk2["narrow_tests_early"] > 0 and wk2["polygon_axes_early"] == 10 * wk2["narrow_tests_early"]
    # cubes far enough apart to be separated by the first support plane: exactly 1 support call per narrow test
    o3 = ho.Oracle(3, (L,) * 3, ho.KIND_POLYHEDRON, 2, 1, verts=CUBE)
    o3.set_work_detail(True); o3.set_moves(1e-6, 1e-6, 1)
    pos3 = np.zeros((2, 4), np.float32); pos3[1, 0] = 1.6                     # inside the circumsphere range sqrt(3), gap 0.6
    o3.set_state(pos3, quat); o3.sweep()
    wk3 = o3.work()
    assert wk3["narrow_tests_early"] > 0 and wk3["gjk_support_calls_early"] == wk3["narrow_tests_early"]
    # off by default
    o4 = ho.Oracle(3, (L,) * 3, ho.KIND_POLYHEDRON, 2, 1, verts=CUBE)
    o4.set_moves(1e-6, 1e-6, 1); o4.set_state(pos3, quat); o4.sweep()
    assert o4.work()["gjk_support_calls_early"] == 0 and o4.work()["narrow_tests_early"] > 0


@pytest.mark.parametrize("nt", [2, 5])
def test_threaded_colour_loop_is_bit_identical_to_serial(nt):
    # P4 in practice: the cells of one colour as a parallel-for give the serial result, trace, counters and work
    from paper_1509_04692_b200 import workloads as wl
    for w in (wl.pentagons(24), wl.cubes(6)):
        def make():
            o = ho.Oracle(w.dim, w.L, w.kind, w.N, 1, diameter=w.diameter, verts=w.verts)
            o.set_moves(w.d, w.a, w.n_select); o.set_state(w.pos4, w.quat4)
            return o
        a, b = make(), make()
        b.set_threads(nt)
        for _ in range(4):
            ra = a.sweep(want_trace=True, want_mmin=True); rb = b.sweep(want_trace=True, want_mmin=True)
            assert np.array_equal(ra["trace"], rb["trace"])
            assert np.array_equal(np.nan_to_num(ra["mmin"], nan=-7.0), np.nan_to_num(rb["mmin"], nan=-7.0))
        assert all(np.array_equal(x, y) for x, y in zip(a.get_state(), b.get_state()))
        assert a.counters() == b.counters() and a.work() == b.work()
