"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/hpmc.h declares,
and the argument validation that needs no GPU behaves as the header states."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1509_04692_b200 import binding as hb
from paper_1509_04692_b200 import build as hbuild
from paper_1509_04692_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    hbuild.build()
    return hb.load_library()


def test_header_symbols_all_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "hpmc.h")).read()
    declared = sorted(set(re.findall(r"\b(hpmc_[a-z0-9_]+)\s*\(", hdr)))
    assert declared == sorted(hb.ABI_SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None


def _create(lib, dim, L, kind, N, diameter=0.0, verts=None, sweep_radius=0.0):
    box = hb.Box(); box.dim = dim
    for k in range(3):
        box.L[k] = L[k] if k < len(L) else 1.0
    sd = hb.ShapeDesc(); sd.kind = kind; sd.diameter = diameter; sd.sweep_radius = sweep_radius
    keep = None
    if verts is not None:
        keep = np.ascontiguousarray(verts, dtype=np.float64)
        sd.nverts = keep.shape[0]; sd.verts = keep.ctypes.data_as(C.POINTER(C.c_double))
    h = C.c_void_p()
    rc = lib.hpmc_create(C.byref(box), C.byref(sd), N, 1, None, C.byref(h))
    return rc, h


def test_create_validation_and_grid(lib):
    rc, h = _create(lib, 2, (70.4, 70.4), hb.KIND_DISK, 4096, diameter=1.0)
    assert rc == 0
    gi = hb.GridInfo(); assert lib.hpmc_get_grid(h, C.byref(gi)) == 0
    assert list(gi.n)[:2] == [70, 70] and gi.num_cells == 4900 and gi.N == 4096
    assert np.float32(gi.L_f[0]) == np.float32(70.4)
    assert lib.hpmc_workspace_bytes(h) > 4096 * (2 * 20 + 8)     # 2-D: two pose+tag buffers and the (cell, rank) keys
    # unbound context: sweeping is an error, not a crash
    assert lib.hpmc_sweep(h, 1) == -4
    assert b"not bound" in lib.hpmc_last_error(h)
    assert lib.hpmc_set_moves(h, -1.0, 0.1, 4) == -1 and lib.hpmc_set_moves(h, 0.1, 0.1, 0) == -1
    assert lib.hpmc_set_moves(h, 0.1, 0.1, 70000) == -1 and lib.hpmc_set_moves(h, 0.15, 0.0, 4) == 0
    assert lib.hpmc_destroy(h) == 0

    for L, n in ((64.0, 62), (1024.0, 1022), (4096.0, 4092)):
        rc, h = _create(lib, 2, (L, L), hb.KIND_POLYGON, 16, verts=wl.regular_polygon(5, 0.5))
        assert rc == 0
        assert lib.hpmc_get_grid(h, C.byref(gi)) == 0 and list(gi.n)[:2] == [n, n]
        lib.hpmc_destroy(h)
    rc, h = _create(lib, 3, (40.0,) * 3, hb.KIND_POLYHEDRON, 8, verts=wl.cube_vertices(1.0))
    assert rc == 0 and lib.hpmc_get_grid(h, C.byref(gi)) == 0 and list(gi.n) == [22, 22, 22]
    assert gi.d_max == pytest.approx(3 ** 0.5)
    lib.hpmc_destroy(h)


def test_rounded_shapes_grid_and_validation(lib):
    """Spheropolygons / spheropolyhedra: d_max = 2 (circumradius + sweep_radius) sets the grid (R11)."""
    gi = hb.GridInfo()
    rc, h = _create(lib, 2, (64.0, 64.0), hb.KIND_POLYGON, 16, verts=wl.regular_polygon(5, 0.35), sweep_radius=0.1)
    assert rc == 0 and lib.hpmc_get_grid(h, C.byref(gi)) == 0
    assert gi.d_max == pytest.approx(0.9, abs=1e-15) and list(gi.n)[:2] == [70, 70]        # 2 floor(64 / (2 x 0.9 (1 + 2^-10)))
    lib.hpmc_destroy(h)
    rc, h = _create(lib, 3, (40.0,) * 3, hb.KIND_POLYHEDRON, 8, verts=wl.cube_vertices(0.7), sweep_radius=0.15)
    assert rc == 0 and lib.hpmc_get_grid(h, C.byref(gi)) == 0
    assert gi.d_max == pytest.approx(2 * (0.35 * 3 ** 0.5 + 0.15)) and list(gi.n) == [26, 26, 26]
    lib.hpmc_destroy(h)
    for bad in (-0.1, float("nan"), float("inf")):
        assert _create(lib, 2, (64.0, 64.0), hb.KIND_POLYGON, 16, verts=wl.regular_polygon(5, 0.35), sweep_radius=bad)[0] == -2
    assert _create(lib, 2, (64.0, 64.0), hb.KIND_DISK, 16, diameter=1.0, sweep_radius=-1.0)[0] == 0     # ignored for disks


def test_create_rejects_bad_input(lib):
    assert _create(lib, 4, (10, 10), hb.KIND_DISK, 4, diameter=1.0)[0] == -1                     # dim
    assert _create(lib, 2, (3.9, 3.9), hb.KIND_DISK, 4, diameter=1.0)[0] == -3                   # < 4 cells per side
    assert _create(lib, 2, (10, 10), hb.KIND_DISK, 4, diameter=0.0)[0] == -2
    assert _create(lib, 2, (10, 10), hb.KIND_POLYGON, 4, verts=wl.regular_polygon(5, 0.5)[::-1])[0] == -2   # clockwise
    concave = np.array([[0, 0], [1, 0], [0.2, 0.2], [0, 1.0]]) - 0.25
    assert _create(lib, 2, (10, 10), hb.KIND_POLYGON, 4, verts=concave)[0] == -2
    assert _create(lib, 2, (10, 10), hb.KIND_POLYGON, 4, verts=wl.regular_polygon(40, 0.5))[0] == -2        # > 32 vertices
    inner = np.vstack([wl.cube_vertices(1.0), [[0.1, 0.0, 0.0]]])
    assert _create(lib, 3, (10,) * 3, hb.KIND_POLYHEDRON, 4, verts=inner)[0] == -2                           # not a hull vertex
    assert _create(lib, 2, (10, 10), hb.KIND_POLYHEDRON, 4, verts=wl.cube_vertices(1.0))[0] == -2            # wrong dim
    assert b"" != lib.hpmc_last_error(None)
    # R11/R22: in boxes so large that d_max 2^-10 no longer covers the fp32 rounding of cell_of the cells get wider, not the box refused
    gi = hb.GridInfo()
    import math
    for L, n in ((4096.0, 4092), (8192.0, 8180), (65536.0, 64776)):
        rc, h = _create(lib, 2, (L, 8.0), hb.KIND_POLYGON, 4, verts=wl.regular_polygon(5, 0.5))
        assert rc == 0 and lib.hpmc_get_grid(h, C.byref(gi)) == 0 and gi.n[0] == n, (L, gi.n[0])
        ulp = math.ldexp(1.0, math.frexp(math.nextafter(L, 0.0))[1] - 24)        # fp32 ulp of coordinate differences just below L
        assert gi.w[0] - 1.0 >= max(2.0 ** -10, 3 * ulp) and gi.n[0] % 2 == 0
        lib.hpmc_destroy(h)

def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    w = wl.disks(8)
    with pytest.raises(hb.HpmcError):
        hb.from_workload(w)


def test_options_and_pass_description_need_no_gpu(lib):
    """hpmc_set_option validates names and ranges; hpmc_describe_pass names the kernel the options select."""
    def describe(h):
        buf = C.create_string_buffer(256)
        assert lib.hpmc_describe_pass(h, buf, 256) > 0
        return buf.value.decode()
    rc, h = _create(lib, 2, (1024.0, 1024.0), hb.KIND_POLYGON, 1 << 20, verts=wl.regular_polygon(5, 0.5))
    assert rc == 0
    assert describe(h).startswith("k_sweep_tile2d_flow<4 warps x 1 row")          # 1.7 waves of tiles: dataflow launch
    assert lib.hpmc_set_option(h, b"flow", 0) == 0 and describe(h).startswith("k_sweep_tile2d<")
    assert lib.hpmc_set_option(h, b"path", 1) == 0 and describe(h).startswith("k_sweep_colour")
    assert lib.hpmc_set_option(h, b"path", 7) == -1 and lib.hpmc_set_option(h, b"flow", 2) == -1
    assert lib.hpmc_set_option(h, b"tile_shape", 4) == -1 and lib.hpmc_set_option(h, b"no_such_option", 1) == -1
    assert lib.hpmc_destroy(h) == 0
    rc, h = _create(lib, 2, (64.0, 64.0), hb.KIND_POLYGON, 4096, verts=wl.regular_polygon(5, 0.5))
    assert rc == 0 and describe(h).startswith("k_sweep_warpcell")                  # 961 active cells per colour
    assert lib.hpmc_set_option(h, b"path", 2) == 0 and describe(h).startswith("k_sweep_tile2d<")   # below one wave: per colour
    assert lib.hpmc_destroy(h) == 0
    rc, h = _create(lib, 3, (40.0, 40.0, 40.0), hb.KIND_POLYHEDRON, 32768, verts=wl.cube_vertices(1.0))
    assert rc == 0 and describe(h).startswith("k_sweep_warpcell")
    assert lib.hpmc_destroy(h) == 0
