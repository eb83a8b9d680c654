"""Thin ctypes binding over libhpmc.so (C-ABI: include/hpmc.h).  Argument marshalling only.

PyTorch is used for device memory and the CUDA stream; every step of the sweep runs in the library's
CUDA kernels.  There is NO fallback: if libhpmc.so is missing or a call fails, this module raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhpmc.so")

KIND_DISK, KIND_POLYGON, KIND_POLYHEDRON = 0, 1, 2

# every symbol include/hpmc.h declares (checked by tests/test_abi.py)
ABI_SYMBOLS = ["hpmc_create", "hpmc_destroy", "hpmc_last_error", "hpmc_get_grid", "hpmc_workspace_bytes", "hpmc_bind",
               "hpmc_set_moves", "hpmc_sweep", "hpmc_count_overlaps", "hpmc_get_state", "hpmc_set_sweep_counter",
               "hpmc_reset_counters", "hpmc_set_trace", "hpmc_get_cell_list", "hpmc_sweep_host", "hpmc_sweep_host_pose2d", "hpmc_set_option", "hpmc_set_profile",
               "hpmc_get_profile", "hpmc_launch_count", "hpmc_describe_pass", "hpmc_get_stat", "hpmc_measure_fp32_peak", "hpmc_set_partition", "hpmc_sweep_phase",
               "hpmc_partition_rows", "hpmc_row_offsets", "hpmc_sorted_pose", "hpmc_set_inactive_layers", "hpmc_dist_load",
               "hpmc_dist_route", "hpmc_dist_append", "hpmc_local_count", "hpmc_sorted_tags", "hpmc_count_overlaps_noalloc"]


class HpmcError(RuntimeError):
    pass


class Box(C.Structure):
    _fields_ = [("dim", C.c_int), ("L", C.c_double * 3)]


class ShapeDesc(C.Structure):
    _fields_ = [("kind", C.c_int), ("diameter", C.c_double), ("nverts", C.c_int), ("verts", C.POINTER(C.c_double)),
                ("sweep_radius", C.c_double)]


class Counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in
                ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials", "sweeps")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class GridInfo(C.Structure):
    _fields_ = [("dim", C.c_int), ("n", C.c_int * 3), ("w", C.c_double * 3), ("L_f", C.c_float * 3),
                ("inv_w", C.c_float * 3), ("d_max", C.c_double), ("num_cells", C.c_int64), ("N", C.c_int64)]


_lib = None


def load_library():
    """Load libhpmc.so; raises HpmcError if it has not been built (no CPU fallback exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise HpmcError(f"{LIB_PATH} is missing: build it with `python -m paper_1509_04692_b200.build` "
                        "(there is no CPU fallback for the sweep)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.hpmc_create.argtypes = [C.POINTER(Box), C.POINTER(ShapeDesc), C.c_int64, C.c_uint64, vp, C.POINTER(vp)]
    L.hpmc_destroy.argtypes = [vp]
    L.hpmc_last_error.argtypes = [vp]; L.hpmc_last_error.restype = C.c_char_p
    L.hpmc_get_grid.argtypes = [vp, C.POINTER(GridInfo)]
    L.hpmc_workspace_bytes.argtypes = [vp]; L.hpmc_workspace_bytes.restype = C.c_size_t
    L.hpmc_bind.argtypes = [vp, vp, vp, vp, C.c_size_t]
    L.hpmc_set_moves.argtypes = [vp, C.c_double, C.c_double, C.c_int]
    L.hpmc_sweep.argtypes = [vp, C.c_int64]
    L.hpmc_count_overlaps.argtypes = [vp, C.POINTER(C.c_int64)]
    L.hpmc_get_state.argtypes = [vp, vp, vp, C.POINTER(Counters), C.POINTER(C.c_int64)]
    L.hpmc_set_sweep_counter.argtypes = [vp, C.c_uint64]
    L.hpmc_reset_counters.argtypes = [vp]
    L.hpmc_set_trace.argtypes = [vp, vp, C.c_int64]
    L.hpmc_get_cell_list.argtypes = [vp, C.c_uint64, vp, vp, vp, C.POINTER(C.c_float), C.POINTER(C.c_int32)]
    L.hpmc_sweep_host.argtypes = [vp, vp, vp, C.c_int64, vp, vp, C.POINTER(Counters)]
    L.hpmc_sweep_host_pose2d.argtypes = [vp, vp, C.c_int64, vp, C.POINTER(Counters)]
    L.hpmc_set_option.argtypes = [vp, C.c_char_p, C.c_int64]
    L.hpmc_set_profile.argtypes = [vp, C.c_int]
    L.hpmc_get_profile.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.hpmc_launch_count.argtypes = [vp]; L.hpmc_launch_count.restype = C.c_int64
    L.hpmc_get_stat.argtypes = [vp, C.c_char_p, C.POINTER(C.c_int64)]
    L.hpmc_measure_fp32_peak.argtypes = [vp, C.POINTER(C.c_double)]
    L.hpmc_set_partition.argtypes = [vp, C.c_int, C.c_int]
    L.hpmc_sweep_phase.argtypes = [vp, C.c_int]
    L.hpmc_partition_rows.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.hpmc_row_offsets.argtypes = [vp, C.POINTER(C.c_int32), C.c_int, C.POINTER(C.c_int64)]
    L.hpmc_sorted_pose.argtypes = [vp, C.POINTER(vp)]
    L.hpmc_sorted_tags.argtypes = [vp, C.POINTER(vp)]
    L.hpmc_set_inactive_layers.argtypes = [vp, vp, C.c_int32]
    L.hpmc_dist_load.argtypes = [vp, vp, vp, C.c_int64]
    L.hpmc_dist_route.argtypes = [vp, C.c_int, vp, vp, C.c_int64, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
    L.hpmc_dist_append.argtypes = [vp, vp, vp, C.c_int64]
    L.hpmc_local_count.argtypes = [vp]; L.hpmc_local_count.restype = C.c_int64
    L.hpmc_count_overlaps_noalloc.argtypes = [vp, vp, vp, C.c_int64, vp]
    L.hpmc_describe_pass.argtypes = [vp, C.c_char_p, C.c_size_t]
    for name in ABI_SYMBOLS:
        if name not in ("hpmc_last_error", "hpmc_workspace_bytes", "hpmc_launch_count", "hpmc_local_count"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


class Hpmc:
    """One NVT hard-particle system on one GPU.  Mirrors the C-ABI names one to one."""

    def __init__(self, dim, L, kind, N, seed, diameter=0.0, verts=None, device="cuda:0", stream=None, sweep_radius=0.0):
        import torch  # device memory + streams only
        self._torch = torch
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise HpmcError("no CUDA device: the sweep has no CPU implementation")
        self.device = torch.device(device)
        self.dim, self.N, self.kind = int(dim), int(N), int(kind)
        box = Box(); box.dim = self.dim
        for k in range(3):
            box.L[k] = float(L[k]) if k < self.dim else 1.0
        sd = ShapeDesc(); sd.kind = self.kind; sd.diameter = float(diameter); sd.sweep_radius = float(sweep_radius)
        self._verts = None
        if verts is not None:
            self._verts = np.ascontiguousarray(verts, dtype=np.float64)
            sd.nverts = int(self._verts.shape[0])
            sd.verts = self._verts.ctypes.data_as(C.POINTER(C.c_double))
        with torch.cuda.device(self.device):
            # a stream of our own: the legacy default stream cannot be captured into a CUDA graph
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            h = C.c_void_p()
            rc = self._lib.hpmc_create(C.byref(box), C.byref(sd), self.N, int(seed), C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc != 0:
            raise HpmcError(f"hpmc_create failed ({rc}): {self._lib.hpmc_last_error(None).decode()}")
        self._h = h
        gi = GridInfo(); self._check(self._lib.hpmc_get_grid(self._h, C.byref(gi)))
        self.n = np.array(list(gi.n), dtype=np.int32)
        self.w = np.array(list(gi.w)); self.L_f = np.array(list(gi.L_f), dtype=np.float32)
        self.inv_w = np.array(list(gi.inv_w), dtype=np.float32)
        self.d_max, self.C = float(gi.d_max), int(gi.num_cells)
        self.n_select = 4
        self.pos4 = self.quat4 = self.workspace = self._trace = None

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            raise HpmcError(f"libhpmc error {rc}: {self._lib.hpmc_last_error(self._h).decode()}")

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.hpmc_destroy(self._h)
            self._h = None

    # -- C-ABI mirror ----------------------------------------------------------------------------
    def workspace_bytes(self):
        return int(self._lib.hpmc_workspace_bytes(self._h))

    def bind(self, pos4, quat4):
        """pos4/quat4: (N,4) float32, numpy (copied to the device) or CUDA torch tensors (used in place)."""
        torch = self._torch
        def dev(a):
            if isinstance(a, np.ndarray):
                a = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(self.device)
            assert a.is_cuda and a.dtype == torch.float32 and a.is_contiguous() and tuple(a.shape) == (self.N, 4)
            return a
        torch.cuda.current_stream(self.device).synchronize()      # caller's tensors are ready
        with torch.cuda.stream(self.stream):                       # every torch op on the state runs on OUR stream
            self.pos4, self.quat4 = dev(pos4), dev(quat4)
            if self.workspace is None:
                self.workspace = torch.empty(self.workspace_bytes() + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        off = (-base) % 256
        self.stream.synchronize()
        self._check(self._lib.hpmc_bind(self._h, self.pos4.data_ptr(), self.quat4.data_ptr(), base + off, self.workspace.numel() - off))

    def set_moves(self, d, a, n_select):
        self._check(self._lib.hpmc_set_moves(self._h, float(d), float(a), int(n_select)))
        self.n_select = int(n_select)

    def sweep(self, n=1):
        self._check(self._lib.hpmc_sweep(self._h, int(n)))

    def count_overlaps(self):
        out = C.c_int64(-1)
        self._check(self._lib.hpmc_count_overlaps(self._h, C.byref(out)))
        return int(out.value)

    def get_state(self, to_host=True):
        """Un-sort into the bound arrays; returns (pos4, quat4) as numpy (to_host) or the CUDA tensors."""
        self._check(self._lib.hpmc_get_state(self._h, self.pos4.data_ptr(), self.quat4.data_ptr(), None, None))
        self.stream.synchronize()
        if to_host:
            return self.pos4.cpu().numpy(), self.quat4.cpu().numpy()
        return self.pos4, self.quat4

    def counters(self):
        c = Counters(); t = C.c_int64()
        self._check(self._lib.hpmc_get_state(self._h, None, None, C.byref(c), C.byref(t)))
        d = c.as_dict(); d["sweep_counter"] = int(t.value)
        return d

    def set_sweep_counter(self, t):
        self._check(self._lib.hpmc_set_sweep_counter(self._h, int(t)))

    def reset_counters(self):
        self._check(self._lib.hpmc_reset_counters(self._h))

    def enable_trace(self, on=True):
        torch = self._torch
        if on:
            words = 2 * self.C * self.n_select
            with torch.cuda.stream(self.stream):
                self._trace = torch.zeros(words, dtype=torch.int32, device=self.device)
            self.stream.synchronize()
            self._check(self._lib.hpmc_set_trace(self._h, self._trace.data_ptr(), words))
        else:
            self._trace = None
            self._check(self._lib.hpmc_set_trace(self._h, None, 0))

    def read_trace(self):
        self.stream.synchronize()
        return self._trace.cpu().numpy().view(np.uint32).reshape(-1, 2)

    def cell_list(self, t):
        """Cell list of sweep t's grid shift for the current state: (cell_of_tag, cell_start, member_tags, shift, perm)."""
        torch = self._torch
        with torch.cuda.stream(self.stream):
            cst = torch.empty(self.C + 1, dtype=torch.int32, device=self.device)
            mem = torch.empty(max(self.N, 1), dtype=torch.int32, device=self.device)
            cid = torch.empty(max(self.N, 1), dtype=torch.int32, device=self.device)
        shift = (C.c_float * 3)(); perm = (C.c_int32 * 8)()
        self._check(self._lib.hpmc_get_cell_list(self._h, int(t), cst.data_ptr(), mem.data_ptr(), cid.data_ptr(), shift, perm))
        self.stream.synchronize()
        return (cid.cpu().numpy()[: self.N], cst.cpu().numpy(), mem.cpu().numpy()[: self.N],
                np.array(list(shift), dtype=np.float32), np.array(list(perm), dtype=np.int32)[: 1 << self.dim])

    def sweep_host(self, h_pos4, h_quat4, n, h_pos4_out, h_quat4_out):
        """End-to-end call with HOST buffers (torch CPU tensors, ideally pinned): H2D, n sweeps, D2H."""
        c = Counters()
        self._check(self._lib.hpmc_sweep_host(self._h, h_pos4.data_ptr(), h_quat4.data_ptr(), int(n),
                                              h_pos4_out.data_ptr(), h_quat4_out.data_ptr(), C.byref(c)))
        return c.as_dict()

    def sweep_host_pose2d(self, h_pose4, n, h_pose4_out):
        """End-to-end call for 2-D systems with HOST poses (N, 4) = (x, y, qw, qz) (torch CPU tensors, ideally pinned): half the
        bytes of sweep_host each way.  h_pose4_out may be None."""
        c = Counters()
        self._check(self._lib.hpmc_sweep_host_pose2d(self._h, h_pose4.data_ptr(), int(n),
                                                     h_pose4_out.data_ptr() if h_pose4_out is not None else None, C.byref(c)))
        return c.as_dict()

    def set_option(self, name, value):
        self._check(self._lib.hpmc_set_option(self._h, name.encode(), int(value)))

    def set_profile(self, on=True):
        self._check(self._lib.hpmc_set_profile(self._h, 1 if on else 0))

    def get_profile(self):
        """{'build_ms', 'build_n', 'colour_ms', 'colour_n'} since set_profile (synchronises)."""
        mb, mc = C.c_double(), C.c_double()
        nb, nc = C.c_int64(), C.c_int64()
        self._check(self._lib.hpmc_get_profile(self._h, C.byref(mb), C.byref(nb), C.byref(mc), C.byref(nc)))
        return {"build_ms": mb.value, "build_n": int(nb.value), "colour_ms": mc.value, "colour_n": int(nc.value)}

    def describe_pass(self):
        buf = C.create_string_buffer(256)
        n = self._lib.hpmc_describe_pass(self._h, buf, 256)
        if n < 0:
            raise HpmcError("hpmc_describe_pass failed")
        return buf.value.decode()

    def launch_count(self):
        return int(self._lib.hpmc_launch_count(self._h))

    def measure_fp32_peak(self):
        """TFLOP/s of the library's pure-FMA microkernel on this device (the measured FP32 roofline denominator)."""
        v = C.c_double()
        self._check(self._lib.hpmc_measure_fp32_peak(self._h, C.byref(v)))
        return float(v.value)

    # -- partitioned compute (one system on several GPUs / contexts), see paper_1509_04692_b200/partition.py -----------
    def set_partition(self, rank, nranks):
        self._check(self._lib.hpmc_set_partition(self._h, int(rank), int(nranks)))

    def sweep_phase(self, phase):
        self._check(self._lib.hpmc_sweep_phase(self._h, int(phase)))

    def partition_rows(self, rank, nranks):
        a, b = C.c_int32(), C.c_int32()
        self._check(self._lib.hpmc_partition_rows(self._h, int(rank), int(nranks), C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def row_offsets(self, rows):
        r = (C.c_int32 * len(rows))(*[int(x) for x in rows])
        o = (C.c_int64 * len(rows))()
        self._check(self._lib.hpmc_row_offsets(self._h, r, len(rows), o))
        return [int(x) for x in o]

    def sorted_pose(self):
        """The current cell-sorted pose array as a torch view (local count, 4) into the workspace (valid until the next build)."""
        p = C.c_void_p()
        self._check(self._lib.hpmc_sorted_pose(self._h, C.byref(p)))
        n = self.local_count()
        off = int(p.value) - self.workspace.data_ptr()
        assert 0 <= off and off + 16 * n <= self.workspace.numel()
        return self.workspace[off:off + 16 * n].view(self._torch.float32).view(n, 4)

    def sorted_tags(self):
        """The tags that go with sorted_pose(), as a torch int32 view into the workspace."""
        p = C.c_void_p()
        self._check(self._lib.hpmc_sorted_tags(self._h, C.byref(p)))
        n = self.local_count()
        off = int(p.value) - self.workspace.data_ptr()
        assert 0 <= off and off + 4 * n <= self.workspace.numel()
        return self.workspace[off:off + 4 * n].view(self._torch.int32)

    def local_count(self):
        return int(self._lib.hpmc_local_count(self._h))

    def set_inactive_layers(self, mask):
        """layers of cells along the last axis that make no trials (n[dim-1] bytes; None clears)."""
        if mask is None:
            self._check(self._lib.hpmc_set_inactive_layers(self._h, None, 0))
            return
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        self._check(self._lib.hpmc_set_inactive_layers(self._h, m.ctypes.data_as(C.c_void_p), int(m.size)))

    def dist_load(self, pose4, tags):
        """Distributed state: `pose4` (n, 4) float32 (x, y, qw, qz) and `tags` (n,) int32 global ids, device tensors."""
        assert pose4.is_cuda and tags.is_cuda and pose4.dtype == self._torch.float32 and tags.dtype == self._torch.int32
        pose4, tags = pose4.contiguous(), tags.contiguous()
        with self._torch.cuda.stream(self.stream):
            self._check(self._lib.hpmc_dist_load(self._h, pose4.data_ptr(), tags.data_ptr(), int(tags.numel())))
        self.stream.synchronize()            # the sources may be temporaries

    def dist_route(self, owned_only, up_pose, up_tags, down_pose, down_tags):
        """Classify for the next sweep's grid; fills the caller's send buffers; returns (kept, up, down, unclassified)."""
        cnt = (C.c_int64 * 4)()
        self._check(self._lib.hpmc_dist_route(self._h, int(bool(owned_only)), up_pose.data_ptr(), up_tags.data_ptr(), int(up_tags.numel()),
                                              down_pose.data_ptr(), down_tags.data_ptr(), int(down_tags.numel()), cnt))
        return tuple(int(x) for x in cnt)

    def dist_append(self, pose4, tags, n):
        if n:
            self._check(self._lib.hpmc_dist_append(self._h, pose4.data_ptr(), tags.data_ptr(), int(n)))

    def count_overlaps_noalloc(self, pos4, quat4, out):
        """Overlapping pairs among the particles of the CUDA tensors pos4 / quat4 ((n, 4) float32, tag order) in this context's
        box, through the entry point that allocates nothing (static scratch inside the library; n <= 65 536).  `out`: a CUDA
        int64 tensor of one element that receives the count (-1: a coordinate outside the box).  No bind is needed.
        Asynchronous on the context's stream: synchronise it before reading `out`."""
        torch = self._torch
        assert pos4.is_cuda and pos4.dtype == torch.float32 and pos4.is_contiguous() and pos4.shape[1] == 4
        assert quat4 is None or (quat4.is_cuda and quat4.dtype == torch.float32 and quat4.is_contiguous() and quat4.shape == pos4.shape)
        assert out.is_cuda and out.dtype == torch.int64 and out.numel() == 1
        torch.cuda.current_stream(self.device).synchronize()      # the caller's tensors are ready
        self._check(self._lib.hpmc_count_overlaps_noalloc(self._h, pos4.data_ptr(), quat4.data_ptr() if quat4 is not None else None,
                                                          int(pos4.shape[0]), out.data_ptr()))

    def get_stat(self, name):
        v = C.c_int64()
        self._check(self._lib.hpmc_get_stat(self._h, name.encode(), C.byref(v)))
        return int(v.value)


def from_workload(w, seed=1, device="cuda:0"):
    """Create + bind + set_moves for a workloads.Workload."""
    h = Hpmc(w.dim, w.L, w.kind, w.N, seed, diameter=w.diameter, verts=w.verts, device=device, sweep_radius=w.sweep_radius)
    h.set_moves(w.d, w.a, w.n_select)
    h.bind(w.pos4, w.quat4)
    return h
