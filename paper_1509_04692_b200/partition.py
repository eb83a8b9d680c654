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

A second scheme DISTRIBUTES the state, the paper's way: the last cell row of every slab is an inactive region for
the sweep (`inactive_mask`), so a rank reads no row that another rank changes, holds only its slab plus one ghost row, and
exchanges particles once per sweep (`LocalDistributed`, `DistributedState`; include/hpmc.h hpmc_dist_*).  Its trajectory is
the single-GPU one with the same inactive rows.

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


# ---- distributed state with an inactive region ------------------------------------------------------------------

def inactive_mask(slabs, nrows):
    """The inactive region of a slab decomposition: the last cell row of every non-empty slab (R-strip)."""
    mask = np.zeros(nrows, dtype=np.uint8)
    for a, b in slabs:
        if b > a:
            mask[b - 1] = 1
    return mask


def pose_of(pos4, quat4):
    """(x, y, qw, qz) rows of a 2-D state given as pos4 = (x, y, 0, 0), quat4 = (w, 0, 0, z): layout only."""
    return np.ascontiguousarray(np.stack([pos4[:, 0], pos4[:, 1], quat4[:, 0], quat4[:, 3]], axis=1), dtype=np.float32)


def neighbours(rank, slabs):
    """(below, above) among the ranks that own rows, periodic."""
    owners = [r for r, (a, b) in enumerate(slabs) if b > a]
    i = owners.index(rank)
    return owners[i - 1], owners[(i + 1) % len(owners)]


class LocalDistributed:
    """`n` ranks with a DISTRIBUTED state as `n` contexts of this process on one device, stepped one after the other: each holds
    its slab of cell rows plus one ghost row; once per sweep particles are routed between them.  `capacity`: particles a rank
    can hold (default: all of them, so that any decomposition of a small test system fits)."""

    def __init__(self, workload, n, seed=1, device="cuda:0", capacity=None, binding=None):
        import dataclasses
        from . import binding as hb
        import torch
        hb = binding or hb
        self.n, self.N = n, workload.N
        cap = int(capacity or workload.N)
        wcap = dataclasses.replace(workload, N=cap, pos4=workload.pos4[:cap], quat4=workload.quat4[:cap]) if cap != workload.N else workload
        self.g = [hb.from_workload(wcap, seed=seed, device=device) for _ in range(n)]
        for r, g in enumerate(self.g):
            g.set_partition(r, n)
        self.nrows = int(self.g[0].n[1])
        self.slabs = [self.g[0].partition_rows(r, n) for r in range(n)]
        self.mask = inactive_mask(self.slabs, self.nrows)
        dev = torch.device(device)
        pose = torch.from_numpy(pose_of(workload.pos4, workload.quat4)).to(dev)
        tags = torch.arange(workload.N, dtype=torch.int32, device=dev)
        self.buf = []
        for g in self.g:
            g.set_inactive_layers(self.mask)
            up = (torch.empty((cap, 4), dtype=torch.float32, device=dev), torch.empty(cap, dtype=torch.int32, device=dev))
            down = (torch.empty((cap, 4), dtype=torch.float32, device=dev), torch.empty(cap, dtype=torch.int32, device=dev))
            self.buf.append((up, down))
            # every rank is offered the whole system and keeps the rows of its slab and its ghost row in the first sweep's grid
            if workload.N <= cap:
                g.dist_load(pose, tags)
                g.dist_route(False, up[0], up[1], down[0], down[1])
            else:
                g.dist_load(pose[:0], tags[:0])
                for lo in range(0, workload.N, cap // 2):
                    hi = min(lo + cap // 2, workload.N)
                    g.dist_append(pose[lo:hi], tags[lo:hi], hi - lo)
                    g.dist_route(False, up[0], up[1], down[0], down[1])
        self.migrated = 0

    def sweep(self, nsweeps=1):
        torch = self.g[0]._torch
        for _ in range(nsweeps):
            for g in self.g:
                g.sweep_phase(-1)
                for ci in range(4):
                    g.sweep_phase(ci)             # no exchange between the colours: nothing a rank reads changes elsewhere
            counts = []
            for g, (up, down) in zip(self.g, self.buf):
                counts.append(g.dist_route(True, up[0], up[1], down[0], down[1]))
            torch.cuda.synchronize()
            for r, g in enumerate(self.g):
                below, above = neighbours(r, self.slabs)
                (up, down), (_, n_up, n_down, _) = self.buf[r], counts[r]
                self.g[above].dist_append(up[0], up[1], n_up)
                self.g[below].dist_append(down[0], down[1], n_down)
                self.migrated += n_up + n_down
            torch.cuda.synchronize()

    def gather(self):
        """Whole state by global tag, (N, 4) poses (x, y, qw, qz), from the rows every rank OWNS in the grid of the next sweep
        (after a sweep a rank holds them plus its ghost row; a particle is owned by exactly one rank)."""
        out = np.full((self.N, 4), np.nan, dtype=np.float32)
        seen = np.zeros(self.N, dtype=np.int32)
        for r, g in enumerate(self.g):
            g.sweep_phase(-1)                                    # cell list of the next sweep: rows are contiguous ranges
            a, b = self.slabs[r]
            lo, hi = g.row_offsets([a, b])
            pose = g.sorted_pose()[lo:hi].cpu().numpy()
            tags = g.sorted_tags()[lo:hi].cpu().numpy()
            out[tags] = pose
            seen[tags] += 1
            g.set_sweep_counter(g.counters()["sweep_counter"] - 1)   # the build advanced it: put it back, the next sweep rebuilds
        assert np.all(seen == 1), "every particle must be owned by exactly one rank"
        return out

    def counters(self):
        out = None
        for g in self.g:
            c = g.counters()
            if out is None:
                out = dict(c)
            else:
                for k in ("trans_acc", "trans_rej_overlap", "trans_rej_cell", "rot_acc", "rot_rej_overlap", "trials"):
                    out[k] += c[k]
        return out

    def local_counts(self):
        return [g.local_count() for g in self.g]


def exchange_migrants(dist, below, above, up, n_up, down, n_down):
    """The once-per-sweep exchange of a distributed state (the paper's stage 9) for one rank: the first n_up rows of
    up = (pose, tags) go to the rank `above`, the first n_down rows of `down` to the rank `below`; returns what the rank below
    sent up and what the rank above sent down, as ((pose, tags), (pose, tags)).  Counts first, then payloads of exactly that
    size.  Every rank posts its operations in the same order (up before down), so the two messages between the same pair of
    ranks when there are only two of them cannot be confused."""
    import torch
    dev, (up_pose, up_tags), (down_pose, down_tags) = up[0].device, up, down
    c_send_up = torch.tensor([n_up], dtype=torch.int64, device=dev)
    c_send_down = torch.tensor([n_down], dtype=torch.int64, device=dev)
    c_from_below = torch.zeros(1, dtype=torch.int64, device=dev)
    c_from_above = torch.zeros(1, dtype=torch.int64, device=dev)
    ops = [dist.P2POp(dist.isend, c_send_up, above), dist.P2POp(dist.isend, c_send_down, below),
           dist.P2POp(dist.irecv, c_from_below, below), dist.P2POp(dist.irecv, c_from_above, above)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    nb, na = int(c_from_below.item()), int(c_from_above.item())
    got_below = (torch.empty((nb, 4), dtype=torch.float32, device=dev), torch.empty(nb, dtype=torch.int32, device=dev))
    got_above = (torch.empty((na, 4), dtype=torch.float32, device=dev), torch.empty(na, dtype=torch.int32, device=dev))
    ops = []
    if n_up:
        ops += [dist.P2POp(dist.isend, up_pose[:n_up], above), dist.P2POp(dist.isend, up_tags[:n_up], above)]
    if n_down:
        ops += [dist.P2POp(dist.isend, down_pose[:n_down], below), dist.P2POp(dist.isend, down_tags[:n_down], below)]
    if nb:
        ops += [dist.P2POp(dist.irecv, got_below[0], below), dist.P2POp(dist.irecv, got_below[1], below)]
    if na:
        ops += [dist.P2POp(dist.irecv, got_above[0], above), dist.P2POp(dist.irecv, got_above[1], above)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    return got_below, got_above


class DistributedState:
    """This process is rank `dist.get_rank()` of a system whose STATE is distributed over the ranks (one GPU each).  `hpmc` is
    this rank's context (capacity = the N it was created with); `pose`, `tags`: device tensors with any superset of the
    particles this rank needs for the first sweep (the whole system, or its y range with a margin of two cell widths)."""

    def __init__(self, hpmc, dist, pose, tags):
        import torch
        self.g, self.dist = hpmc, dist
        self.rank, self.n = dist.get_rank(), dist.get_world_size()
        hpmc.set_partition(self.rank, self.n)
        self.nrows = int(hpmc.n[1])
        self.slabs = [hpmc.partition_rows(r, self.n) for r in range(self.n)]
        self.mask = inactive_mask(self.slabs, self.nrows)
        hpmc.set_inactive_layers(self.mask)
        self.below, self.above = neighbours(self.rank, self.slabs)
        cap, dev = hpmc.N, pose.device
        self.up = (torch.empty((cap, 4), dtype=torch.float32, device=dev), torch.empty(cap, dtype=torch.int32, device=dev))
        self.down = (torch.empty((cap, 4), dtype=torch.float32, device=dev), torch.empty(cap, dtype=torch.int32, device=dev))
        hpmc.dist_load(pose, tags)
        hpmc.dist_route(False, self.up[0], self.up[1], self.down[0], self.down[1])

    def sweep(self, nsweeps=1):
        g = self.g
        for _ in range(nsweeps):
            g.sweep_phase(-1)
            for ci in range(4):
                g.sweep_phase(ci)
            _, n_up, n_down, _ = g.dist_route(True, self.up[0], self.up[1], self.down[0], self.down[1])   # synchronises
            with g._torch.cuda.stream(g.stream):
                got_below, got_above = exchange_migrants(self.dist, self.below, self.above, self.up, n_up, self.down, n_down)
                g.dist_append(got_below[0], got_below[1], got_below[1].numel())
                g.dist_append(got_above[0], got_above[1], got_above[1].numel())
            g.stream.synchronize()
