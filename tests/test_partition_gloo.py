"""CPU checks of the multi-rank host logic of paper_1509_04692_b200/partition.py: the exchange plan (pure index arithmetic)
and the two collectives on CPU tensors with two gloo ranks.  Each rank plays the colour passes by writing a rank- and
colour-specific pattern into the rows of its own slab; after the plan's copies every rank must hold what a single owner of
all rows would hold wherever the next colour pass reads (own slab + one row either side), and everything after the gather."""
import os
import subprocess
import sys

import numpy as np

from paper_1509_04692_b200 import partition as pt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slabs_tile_the_rows_and_the_plan_covers_every_boundary():
    for n1, th, nr in ((62, 2, 2), (1022, 4, 8), (70, 2, 3), (26, 2, 5), (8, 2, 4), (4, 2, 3)):
        slabs = pt.reference_rows(n1, th, nr)
        assert slabs[0][0] == 0 and slabs[-1][1] == n1
        assert all(slabs[r][1] == slabs[r + 1][0] for r in range(nr - 1))
        per_row = 3                                                   # particles per cell row (any layout works for the arithmetic)
        boundary, gather = pt.exchange_plan(slabs, lambda r: per_row * r, n1)
        owners = [r for r, (a, b) in enumerate(slabs) if b > a]
        covered = sorted((lo, hi) for _, lo, hi in gather)
        assert covered[0][0] == 0 and covered[-1][1] == per_row * n1 and all(covered[i][1] == covered[i + 1][0] for i in range(len(covered) - 1))
        for i, r in enumerate(owners):
            if len(owners) < 2:
                assert boundary == []
                continue
            a, b = slabs[r]
            below, above = owners[i - 1], owners[(i + 1) % len(owners)]
            # what rank r reads beyond its slab: the row under its first row and the row over its last row (periodic)
            need = {((a - 1) % n1, below), (b % n1, above)}
            for row, owner in need:
                assert any(src == owner and dst == r and lo == per_row * row and hi == per_row * (row + 1) for src, dst, lo, hi in boundary), (n1, nr, r, row)


WORKER = r'''
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_1509_04692_b200 import partition as pt
dist.init_process_group("gloo")
rank, n = dist.get_rank(), dist.get_world_size()
n1, th, per_row = 26, 2, 5
slabs = pt.reference_rows(n1, th, n)
boundary, gather = pt.exchange_plan(slabs, lambda r: per_row * r, n1)
pose = torch.zeros(per_row * n1, 4)
truth = torch.zeros(per_row * n1, 4)                # what one owner of all rows would hold
for ci in range(4):
    for r, (a, b) in enumerate(slabs):                # every slab's owner rewrites the rows of parity ci & 1 in its slab
        for row in range(a, b):
            if (row & 1) == (ci & 1):
                val = 100.0 * (ci + 1) + row
                truth[per_row * row: per_row * (row + 1)] = val
                if r == rank:
                    pose[per_row * row: per_row * (row + 1)] = val
    if ci < 3:
        pt.exchange_boundaries(dist, rank, pose, boundary)
        a, b = slabs[rank]
        if b > a:                                     # the rows the next pass reads: own slab and one row either side
            for row in [(a - 1) % n1] + list(range(a, b)) + [b % n1]:
                assert torch.equal(pose[per_row * row: per_row * (row + 1)], truth[per_row * row: per_row * (row + 1)]), (rank, ci, row)
    else:
        pt.gather_slabs(dist, pose, gather)
assert torch.equal(pose, truth)
dist.destroy_process_group()
print("rank", rank, "ok")
'''


def test_exchange_and_gather_with_two_gloo_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    for world in (2, 3):
        r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}", "--master-addr", "127.0.0.1",
                            "--master-port", str(29640 + world), str(script), ROOT], capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
        assert r.stdout.count("ok") == world


MIGRANT_WORKER = r'''
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_1509_04692_b200 import partition as pt
dist.init_process_group("gloo")
rank, n = dist.get_rank(), dist.get_world_size()
slabs = pt.reference_rows(26, 2, n)
below, above = pt.neighbours(rank, slabs)
assert below == (rank - 1) % n and above == (rank + 1) % n

def payload(r, which, step):                       # what rank r sends up (which = 0) / down (1) in `step`: sizes vary, some empty
    k = (3 * r + 5 * which + 2 * step) % 7
    tags = (1000 * r + 500 * which + 10 * step + torch.arange(k)).to(torch.int32)
    pose = tags.to(torch.float32)[:, None] * torch.tensor([1.0, -1.0, 0.5, 0.25])
    return pose, tags

cap = 16
for step in range(4):
    up = (torch.zeros(cap, 4), torch.zeros(cap, dtype=torch.int32)); down = (torch.zeros(cap, 4), torch.zeros(cap, dtype=torch.int32))
    pu, tu = payload(rank, 0, step); pd, td = payload(rank, 1, step)
    up[0][:len(tu)] = pu; up[1][:len(tu)] = tu; down[0][:len(td)] = pd; down[1][:len(td)] = td
    got_below, got_above = pt.exchange_migrants(dist, below, above, up, len(tu), down, len(td))
    eb = payload(below, 0, step); ea = payload(above, 1, step)        # the rank below sends UP to me, the rank above DOWN
    assert torch.equal(got_below[1], eb[1]) and torch.equal(got_below[0], eb[0]), (rank, step)
    assert torch.equal(got_above[1], ea[1]) and torch.equal(got_above[0], ea[0]), (rank, step)
dist.destroy_process_group()
print("rank", rank, "ok")
'''


def test_inactive_mask_and_neighbours():
    slabs = pt.reference_rows(26, 2, 3)
    mask = pt.inactive_mask(slabs, 26)
    assert mask.sum() == 3 and all(mask[b - 1] == 1 for _, b in slabs)
    assert pt.neighbours(0, slabs) == (2, 1) and pt.neighbours(2, slabs) == (1, 0)
    slabs = pt.reference_rows(4, 2, 3)                     # more ranks than tile rows: empty slabs own nothing
    owners = [r for r, (a, b) in enumerate(slabs) if b > a]
    assert pt.inactive_mask(slabs, 4).sum() == len(owners)
    for r in owners:
        lo, hi = pt.neighbours(r, slabs)
        assert lo in owners and hi in owners
    pos = np.arange(12, dtype=np.float32).reshape(3, 4); quat = np.arange(12, 24, dtype=np.float32).reshape(3, 4)
    assert np.array_equal(pt.pose_of(pos, quat), np.array([[0, 1, 12, 15], [4, 5, 16, 19], [8, 9, 20, 23]], dtype=np.float32))


def test_migrant_exchange_with_gloo_ranks(tmp_path):
    script = tmp_path / "migrants.py"
    script.write_text(MIGRANT_WORKER)
    for world in (2, 3):
        r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}", "--master-addr", "127.0.0.1",
                            "--master-port", str(29650 + world), str(script), ROOT], capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
        assert r.stdout.count("ok") == world
