"""One system on several GPUs: partitioned compute over a replicated state (include/hpmc.h).

The checkerboard makes the cells of one colour independent.  Every rank holds the whole state, builds the same
cell list (deterministic: members of a cell in ascending tag), and runs the colour-pass tiles of its own slab of cell rows.
Between the colour passes a rank needs the one cell row on either side of its slab as the neighbouring ranks left it, and
before the next build it needs everything.  Rows of cells are contiguous in the cell-sorted pose array and sit at the same
offsets on every rank, so the exchange is a handful of copies of contiguous float ranges:

    after each colour:  first row of my slab -> the rank below, last row of my slab -> the rank above (periodic)
    after the last:     every slab -> every rank

The trajectory is bit-identical to the single-GPU one (tests/test_gpu_partition.py).  The paper distributes the STATE over MPI
ranks with an inactive strip and one exchange per step; with NVLink 5 between the GPUs of a node the few MB to 1 GB
of these systems are cheap to replicate, and the per-colour exchange keeps the single-GPU trajectory exactly.

Two communicators with one interface:
  LocalRanks     the ranks are contexts of ONE process on one GPU, run one after the other (how the scheme is verified on a
                 single GPU; kernels of different ranks never wait on one another);
  DistributedRank one rank per process / GPU, `torch.distributed` (NCCL over NVLink; gloo on CPU tensors in the tests).
No method arithmetic lives here: only which float ranges go where.
"""
import numpy as np


def exchange_plan(slabs, offsets_of_row, nrows):
    """Pure index arithmetic, shared by both communicators and tested on CPU.

    slabs: [(row_begin, row_end)] per rank (cell rows; empty slabs allowed).  offsets_of_row(r) -> index of the first particle
    of cell row r in the cell-sorted arrays (row nrows = N).  Returns (boundary, gather):
      boundary: list of (src_rank, dst_rank, lo, hi): after every colour pass src sends poses [lo, hi) to dst
      gather:   list of (src_rank, lo, hi): after the last colour pass src's slab [lo, hi) goes to every other rank
    """
    owners = [r for r, (a, b) in enumerate(slabs) if b > a]
    boundary, gather = [], []
    for i, r in enumerate(owners):
        a, b = slabs[r]
        gather.append((r, offsets_of_row(a), offsets_of_row(b)))
        if len(owners) < 2:
            continue
        below, above = owners[i - 1], owners[(i + 1) % len(owners)]
        first = (r, below, offsets_of_row(a), offsets_of_row(a + 1))          # my first row: read by the slab that ends at it
        last = (r, above, offsets_of_row(b - 1), offsets_of_row(b))           # my last row: read by the slab that starts after it
        boundary.append(first)
        if not (below == above and b - a == 1):                               # two owners and a one-row slab: same row twice
            boundary.append(last)
    assert sum(hi - lo for _, lo, hi in gather) == offsets_of_row(nrows) - offsets_of_row(0)
    return boundary, gather


class LocalRanks:
    """`n` ranks as `n` library contexts of this process on one device, stepped one after the other."""

    def __init__(self, workload, n, seed=1, device="cuda:0", binding=None):
        from . import binding as hb
        hb = binding or hb
        self.n = n
        self.g = [hb.from_workload(workload, seed=seed, device=device) for _ in range(n)]
        for r, g in enumerate(self.g):
            g.set_partition(r, n)
        self.nrows = int(self.g[0].n[1])
        self.slabs = [self.g[0].partition_rows(r, n) for r in range(n)]

    def sweep(self, nsweeps=1):
        torch = self.g[0]._torch
        for _ in range(nsweeps):
            for g in self.g:
                g.sweep_phase(-1)
            rows = sorted({x for a, b in self.slabs if b > a for x in (a, a + 1, b - 1, b)})
            off = dict(zip(rows, self.g[0].row_offsets(rows)))
            boundary, gather = exchange_plan(self.slabs, lambda r: off[r], self.nrows)
            poses = [g.sorted_pose() for g in self.g]
            for ci in range(4):
                for g in self.g:
                    g.sweep_phase(ci)
                torch.cuda.synchronize()          # the ranks use streams of their own
                if ci < 3:
                    for src, dst, lo, hi in boundary:
                        poses[dst][lo:hi].copy_(poses[src][lo:hi])
                else:
                    for src, lo, hi in gather:
                        for dst in range(self.n):
                            if dst != src:
                                poses[dst][lo:hi].copy_(poses[src][lo:hi])
                torch.cuda.synchronize()

    def get_state(self, rank=0):
        return self.g[rank].get_state()

    def counters(self):
        """Tallies summed over the ranks (each counts the trials of its own tiles); sweeps and the sweep counter are per rank."""
        out = None
        for g in self.g:
            c = g.counters()
            if out is None:
                out = dict(c)
            else:
                for k in ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials"):
                    out[k] += c[k]
        return out

    def count_overlaps(self, rank=0):
        return self.g[rank].count_overlaps()


class DistributedRank:
    """This process is rank `dist.get_rank()` of `dist.get_world_size()`; one GPU each.  `hpmc` is this rank's context, created
    from the SAME workload and seed on every rank."""

    def __init__(self, hpmc, dist):
        self.g, self.dist = hpmc, dist
        self.rank, self.n = dist.get_rank(), dist.get_world_size()
        hpmc.set_partition(self.rank, self.n)
        self.nrows = int(hpmc.n[1])
        self.slabs = [hpmc.partition_rows(r, self.n) for r in range(self.n)]

    def sweep(self, nsweeps=1):
        for _ in range(nsweeps):
            self.g.sweep_phase(-1)
            rows = sorted({x for a, b in self.slabs if b > a for x in (a, a + 1, b - 1, b)})
            off = dict(zip(rows, self.g.row_offsets(rows)))       # identical on every rank: the builds are
            boundary, gather = exchange_plan(self.slabs, lambda r: off[r], self.nrows)
            pose = self.g.sorted_pose()
            for ci in range(4):
                self.g.sweep_phase(ci)
                with self.g._torch.cuda.stream(self.g.stream):
                    if ci < 3:
                        exchange_boundaries(self.dist, self.rank, pose, boundary)
                    else:
                        gather_slabs(self.dist, pose, gather)


def exchange_boundaries(dist, rank, pose, boundary):
    """Point-to-point copies of the plan's boundary rows that involve `rank` (all posted, then waited for)."""
    ops = []
    for src, dst, lo, hi in boundary:
        if hi <= lo or src == dst:
            continue
        if src == rank:
            ops.append(dist.P2POp(dist.isend, pose[lo:hi], dst))
        elif dst == rank:
            ops.append(dist.P2POp(dist.irecv, pose[lo:hi], src))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


def gather_slabs(dist, pose, gather):
    """Every slab to every rank: one broadcast per owning rank of its contiguous range (sizes are known everywhere)."""
    for src, lo, hi in gather:
        if hi > lo:
            dist.broadcast(pose[lo:hi], src=src)


def reference_rows(n1, tile_rows, nranks):
    """The slab rule of hpmc_partition_rows restated for the CPU tests: tile rows of `tile_rows` active rows dealt evenly."""
    nay = n1 // 2
    tiles_y = (nay + tile_rows - 1) // tile_rows
    out = []
    for r in range(nranks):
        ty0, ty1 = tiles_y * r // nranks, tiles_y * (r + 1) // nranks
        out.append((min(2 * tile_rows * ty0, n1), min(2 * tile_rows * ty1, n1)))
    return out
