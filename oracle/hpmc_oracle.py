"""ctypes face of the C oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Argument marshalling only; all arithmetic is in hpmc_oracle.c.  Imports nothing from the
product package.
"""
import ctypes as C

import numpy as np

from . import build as _build

KIND_DISK, KIND_POLYGON, KIND_POLYHEDRON = 0, 1, 2

_lib = None


class Counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in
                ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials", "sweeps")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class Work(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in
                ("cand_scanned_full", "sphere_pass_full", "cand_scanned_early", "narrow_tests_early",
                 "polygon_axes_early", "gjk_support_calls_early")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class FollowStats(C.Structure):
    _fields_ = [("compared", C.c_uint64), ("marginal", C.c_uint64), ("hard_mismatch", C.c_uint64),
                ("first_bad_slot", C.c_int64), ("first_bad_mine", C.c_uint32 * 2),
                ("first_bad_theirs", C.c_uint32 * 2), ("first_bad_mmin", C.c_double)]

    def as_dict(self):
        return {"compared": int(self.compared), "marginal": int(self.marginal),
                "hard_mismatch": int(self.hard_mismatch), "first_bad_slot": int(self.first_bad_slot),
                "first_bad_mine": list(self.first_bad_mine), "first_bad_theirs": list(self.first_bad_theirs),
                "first_bad_mmin": float(self.first_bad_mmin)}


class Probe(C.Structure):
    _fields_ = [("slot", C.c_int64), ("particle", C.c_int64), ("rotate", C.c_int32), ("ncand", C.c_int32),
                ("xt", C.c_float * 3), ("qt", C.c_float * 4), ("cand", C.c_int64 * 64), ("r", (C.c_double * 3) * 64),
                ("qb", (C.c_float * 4) * 64), ("margin", C.c_double * 64)]


def lib():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(_build.build())
    vp, dp, fp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_float)
    u32p, i32p = C.POINTER(C.c_uint32), C.POINTER(C.c_int32)
    L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
    L.orc_u01.argtypes = [C.c_uint32]; L.orc_u01.restype = C.c_float
    L.orc_usym.argtypes = [C.c_uint32]; L.orc_usym.restype = C.c_float
    L.orc_shape_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_int, dp]; L.orc_shape_create.restype = vp
    L.orc_shape_create_rounded.argtypes = [C.c_int, C.c_int, C.c_double, C.c_int, dp]; L.orc_shape_create_rounded.restype = vp
    L.orc_shape_sweep_radius.argtypes = [vp]; L.orc_shape_sweep_radius.restype = C.c_double
    L.orc_create_rounded.argtypes = [C.c_int, dp, C.c_int, C.c_double, C.c_int, dp, C.c_int64, C.c_uint64]
    L.orc_create_rounded.restype = vp
    L.orc_shape_destroy.argtypes = [vp]
    L.orc_shape_dmax.argtypes = [vp]; L.orc_shape_dmax.restype = C.c_double
    L.orc_shape_nfaces.argtypes = [vp]; L.orc_shape_nfaces.restype = C.c_int
    L.orc_shape_nedgedirs.argtypes = [vp]; L.orc_shape_nedgedirs.restype = C.c_int
    L.orc_shape_faces.argtypes = [vp, dp, dp]
    L.orc_shape_margin.argtypes = [vp, dp, dp, dp]; L.orc_shape_margin.restype = C.c_double
    L.orc_shape_gjk.argtypes = [vp, dp, dp, dp]; L.orc_shape_gjk.restype = C.c_int
    L.orc_shape_touch_scale.argtypes = [vp, dp, dp, dp]; L.orc_shape_touch_scale.restype = C.c_double
    L.orc_scale_histogram.argtypes = [vp, C.c_double, C.c_int, C.POINTER(C.c_uint64)]; L.orc_scale_histogram.restype = C.c_int64
    L.orc_create.argtypes = [C.c_int, dp, C.c_int, C.c_double, C.c_int, dp, C.c_int64, C.c_uint64]
    L.orc_create.restype = vp
    L.orc_destroy.argtypes = [vp]
    L.orc_sys_shape.argtypes = [vp]; L.orc_sys_shape.restype = vp
    L.orc_set_moves.argtypes = [vp, C.c_double, C.c_double, C.c_int]; L.orc_set_moves.restype = C.c_int
    L.orc_set_eps_guard.argtypes = [vp, C.c_double]
    L.orc_set_state.argtypes = [vp, fp, fp]
    L.orc_get_state.argtypes = [vp, fp, fp]
    L.orc_set_sweep_counter.argtypes = [vp, C.c_uint64]
    L.orc_get_sweep_counter.argtypes = [vp]; L.orc_get_sweep_counter.restype = C.c_uint64
    L.orc_get_counters.argtypes = [vp, C.POINTER(Counters)]
    L.orc_get_work.argtypes = [vp, C.POINTER(Work)]
    L.orc_reset_counters.argtypes = [vp]
    L.orc_get_grid.argtypes = [vp, i32p, dp, fp, fp, fp]
    L.orc_num_cells.argtypes = [vp]; L.orc_num_cells.restype = C.c_int64
    L.orc_sweep_header.argtypes = [vp, C.c_uint64, fp, i32p]
    L.orc_cell_of.argtypes = [vp, fp, fp]; L.orc_cell_of.restype = C.c_int32
    L.orc_cell_list.argtypes = [vp, fp, i32p, i32p, i32p]
    L.orc_sweep.argtypes = [vp, C.c_int, C.c_int, u32p, C.c_double, u32p, dp, C.POINTER(FollowStats)]
    L.orc_sweep.restype = C.c_int
    L.orc_sweeps.argtypes = [vp, C.c_int64]; L.orc_sweeps.restype = C.c_int
    L.orc_set_mutations.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    L.orc_set_work_detail.argtypes = [vp, C.c_int]
    L.orc_set_threads.argtypes = [vp, C.c_int]
    L.orc_get_threads.argtypes = [vp]; L.orc_get_threads.restype = C.c_int
    L.orc_set_inactive_layers.argtypes = [vp, C.c_void_p, C.c_int32]; L.orc_set_inactive_layers.restype = C.c_int
    L.orc_set_probe.argtypes = [vp, C.c_int64]
    L.orc_get_probe.argtypes = [vp, C.POINTER(Probe)]
    L.orc_textbook_trials.argtypes = [vp, C.c_int64]; L.orc_textbook_trials.restype = C.c_int
    L.orc_count_overlaps_bruteforce.argtypes = [vp]; L.orc_count_overlaps_bruteforce.restype = C.c_int64
    L.orc_count_overlaps_cells.argtypes = [vp]; L.orc_count_overlaps_cells.restype = C.c_int64
    L.orc_min_margin_cells.argtypes = [vp]; L.orc_min_margin_cells.restype = C.c_double
    L.orc_min_same_colour_distance.argtypes = [vp, fp]; L.orc_min_same_colour_distance.restype = C.c_double
    _lib = L
    return L


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _i32p(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _u32p(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint32))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_u32p(c), _u32p(k), _u32p(out))
    return out


def u01(r):
    return float(lib().orc_u01(int(r)))


def usym(r):
    return float(lib().orc_usym(int(r)))


class Shape:
    """One hard shape (O1): disk/sphere, convex polygon (CCW) or convex polyhedron (vertex list); sweep_radius > 0 rounds
    the polygon / polyhedron (spheropolygon / spheropolyhedron)."""

    def __init__(self, dim, kind, diameter=0.0, verts=None, sweep_radius=0.0):
        self.dim, self.kind = dim, kind
        v = np.zeros(1) if verts is None else np.ascontiguousarray(verts, dtype=np.float64)
        nv = 0 if verts is None else v.shape[0]
        if sweep_radius:
            self._h = lib().orc_shape_create_rounded(dim, kind, float(sweep_radius), nv, _dp(v))
        else:
            self._h = lib().orc_shape_create(dim, kind, float(diameter), nv, _dp(v))
        if not self._h:
            raise ValueError("oracle rejected the shape (non-convex, not CCW, too many vertices, bad dim)")

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None:
            lib().orc_shape_destroy(self._h)
            self._h = None

    @property
    def dmax(self):
        return lib().orc_shape_dmax(self._h)

    @property
    def sweep_radius(self):
        return lib().orc_shape_sweep_radius(self._h)

    @property
    def nfaces(self):
        return lib().orc_shape_nfaces(self._h)

    @property
    def nedgedirs(self):
        return lib().orc_shape_nedgedirs(self._h)

    def faces(self):
        n = self.nfaces
        nn, cc = np.zeros((n, 3)), np.zeros(n)
        lib().orc_shape_faces(self._h, _dp(nn), _dp(cc))
        return nn, cc

    def margin(self, r_ab, qa, qb):
        r = np.zeros(3); r[:len(r_ab)] = r_ab
        a = np.ascontiguousarray(qa, dtype=np.float64); b = np.ascontiguousarray(qb, dtype=np.float64)
        return lib().orc_shape_margin(self._h, _dp(r), _dp(a), _dp(b))

    def touch_scale(self, r_ab, qa, qb):
        """O9: lambda* such that the pair at separation lambda * r_ab overlaps iff lambda < lambda*."""
        r = np.zeros(3); r[:len(r_ab)] = r_ab
        a = np.ascontiguousarray(qa, dtype=np.float64); b = np.ascontiguousarray(qb, dtype=np.float64)
        return lib().orc_shape_touch_scale(self._h, _dp(r), _dp(a), _dp(b))

    def gjk(self, r_ab, qa, qb):
        r = np.zeros(3); r[:len(r_ab)] = r_ab
        a = np.ascontiguousarray(qa, dtype=np.float64); b = np.ascontiguousarray(qb, dtype=np.float64)
        return lib().orc_shape_gjk(self._h, _dp(r), _dp(a), _dp(b))


class Oracle:
    """The serial checkerboard-sweep oracle (O1-O8, O11)."""

    def __init__(self, dim, L, kind, N, seed, diameter=0.0, verts=None, sweep_radius=0.0):
        Ld = np.ones(3); Ld[:dim] = np.asarray(L, dtype=np.float64)[:dim]
        v = np.zeros(1) if verts is None else np.ascontiguousarray(verts, dtype=np.float64)
        nv = 0 if verts is None else v.shape[0]
        self.dim, self.N, self.kind = dim, int(N), kind
        if sweep_radius:
            self._h = lib().orc_create_rounded(dim, _dp(Ld), kind, float(sweep_radius), nv, _dp(v), int(N), int(seed))
        else:
            self._h = lib().orc_create(dim, _dp(Ld), kind, float(diameter), nv, _dp(v), int(N), int(seed))
        if not self._h:
            raise ValueError("oracle rejected the system (shape invalid or fewer than 4 cells per side)")
        n = np.zeros(3, np.int32); w = np.zeros(3); wf = np.zeros(3, np.float32)
        iw = np.zeros(3, np.float32); Lf = np.zeros(3, np.float32)
        lib().orc_get_grid(self._h, _i32p(n), _dp(w), _fp(wf), _fp(iw), _fp(Lf))
        self.n, self.w, self.w_f, self.inv_w, self.L_f = n, w, wf, iw, Lf
        self.C = int(lib().orc_num_cells(self._h))
        self.n_select = 4

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None:      # `lib` is gone during interpreter shutdown
            lib().orc_destroy(self._h)
            self._h = None

    def set_moves(self, d, a, n_select):
        if lib().orc_set_moves(self._h, d, a, n_select) != 0:
            raise ValueError("bad move parameters")
        self.n_select = n_select

    def set_eps_guard(self, e):
        lib().orc_set_eps_guard(self._h, e)

    def set_state(self, pos4, quat4):
        p = np.ascontiguousarray(pos4, dtype=np.float32); q = np.ascontiguousarray(quat4, dtype=np.float32)
        assert p.shape == (self.N, 4) and q.shape == (self.N, 4)
        lib().orc_set_state(self._h, _fp(p), _fp(q))

    def get_state(self):
        p = np.zeros((self.N, 4), np.float32); q = np.zeros((self.N, 4), np.float32)
        lib().orc_get_state(self._h, _fp(p), _fp(q))
        return p, q

    @property
    def sweep_counter(self):
        return int(lib().orc_get_sweep_counter(self._h))

    @sweep_counter.setter
    def sweep_counter(self, t):
        lib().orc_set_sweep_counter(self._h, int(t))

    def counters(self):
        c = Counters(); lib().orc_get_counters(self._h, C.byref(c)); return c.as_dict()

    def work(self):
        w = Work(); lib().orc_get_work(self._h, C.byref(w)); return w.as_dict()

    def reset_counters(self):
        lib().orc_reset_counters(self._h)

    def sweep_header(self, t):
        s = np.zeros(3, np.float32); p = np.zeros(8, np.int32)
        lib().orc_sweep_header(self._h, int(t), _fp(s), _i32p(p))
        return s, p[: 1 << self.dim].copy()

    def cell_of(self, x, shift):
        xx = np.zeros(3, np.float32); xx[:len(x)] = x
        ss = np.ascontiguousarray(shift, dtype=np.float32)
        return int(lib().orc_cell_of(self._h, _fp(xx), _fp(ss)))

    def cell_list(self, shift):
        ss = np.ascontiguousarray(shift, dtype=np.float32)
        cid = np.zeros(max(self.N, 1), np.int32); cst = np.zeros(self.C + 1, np.int32)
        mem = np.zeros(max(self.N, 1), np.int32)
        lib().orc_cell_list(self._h, _fp(ss), _i32p(cid), _i32p(cst), _i32p(mem))
        return cid[: self.N], cst, mem[: self.N]

    def sweep(self, neighbour_mode=0, reverse_cells=0, follow=None, follow_tol=1e-5, want_trace=False,
              want_mmin=False):
        nslots = self.C * self.n_select
        tr = np.zeros((nslots, 2), np.uint32) if want_trace else None
        mm = np.zeros(nslots, np.float64) if want_mmin else None
        fs = FollowStats()
        fol = None
        if follow is not None:
            fol = np.ascontiguousarray(follow, dtype=np.uint32)
            assert fol.size == 2 * nslots
        rc = lib().orc_sweep(self._h, neighbour_mode, reverse_cells,
                             _u32p(fol) if fol is not None else None, float(follow_tol),
                             _u32p(tr) if tr is not None else None, _dp(mm) if mm is not None else None, C.byref(fs))
        assert rc == 0
        return {"trace": tr, "mmin": mm, "follow": fs.as_dict()}

    def sweeps(self, n):
        assert lib().orc_sweeps(self._h, int(n)) == 0

    def set_mutations(self, no_shift=0, fixed_colour_order=0, no_leave_cell_reject=0):
        lib().orc_set_mutations(self._h, no_shift, fixed_colour_order, no_leave_cell_reject)

    def set_work_detail(self, on=True):
        """O7: also count separating axes (polygons) / GJK support calls (polyhedra) per early-exit narrow test."""
        lib().orc_set_work_detail(self._h, int(bool(on)))

    def set_threads(self, n):
        """n > 1: same-colour cells as an OpenMP parallel-for (identical results, P4); 1 = serial (default)."""
        lib().orc_set_threads(self._h, int(n))

    def set_inactive_layers(self, mask):
        """layers of cells along the last axis that make no trials (mask: n[dim-1] bytes; None clears)."""
        if mask is None:
            assert lib().orc_set_inactive_layers(self._h, None, 0) == 0
            return
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        assert lib().orc_set_inactive_layers(self._h, m.ctypes.data_as(C.c_void_p), int(m.size)) == 0, "mask size != grid extent"

    def set_probe(self, slot):
        """O8 dump: record the trial pose and candidates of `slot` during the following sweeps (-1 = off)."""
        lib().orc_set_probe(self._h, int(slot))

    def get_probe(self):
        p = Probe(); lib().orc_get_probe(self._h, C.byref(p))
        n = int(p.ncand)
        return {"slot": int(p.slot), "particle": int(p.particle), "rotate": int(p.rotate), "xt": np.array(p.xt[:]),
                "qt": np.array(p.qt[:]), "cand": np.array(p.cand[:n]), "r": np.array([list(x) for x in p.r[:n]]),
                "qb": np.array([list(x) for x in p.qb[:n]]), "margin": np.array(p.margin[:n])}

    def textbook_trials(self, n):
        assert lib().orc_textbook_trials(self._h, int(n)) == 0

    def count_overlaps_bruteforce(self):
        return int(lib().orc_count_overlaps_bruteforce(self._h))

    def count_overlaps_cells(self):
        return int(lib().orc_count_overlaps_cells(self._h))

    def scale_histogram(self, s_max=0.02, nbins=40):
        """O9: counts of pairs whose touch scale s = 1 - lambda* falls in each of nbins bins on [0, s_max)."""
        h = np.zeros(nbins, dtype=np.uint64)
        n = lib().orc_scale_histogram(self._h, float(s_max), int(nbins), h.ctypes.data_as(C.POINTER(C.c_uint64)))
        assert n >= 0, "scale_histogram needs >= 5 cells per side"
        return h

    def min_margin_cells(self):
        return float(lib().orc_min_margin_cells(self._h))

    def min_same_colour_distance(self, shift):
        ss = np.ascontiguousarray(shift, dtype=np.float32)
        return float(lib().orc_min_same_colour_distance(self._h, _fp(ss)))
