"""N > 1: "replicas only".

BASELINE.json north_star scopes this build to one GPU per system ("one GPU (no sharding, no collectives)"), so
`bench.py --gpus N` runs N independent replicas -- replica r has Philox seed and orientation seed 1 + r -- with no
data-path collective.  The only communication is the bench protocol itself: a barrier on both sides of the timed
region, MAX over ranks of the device time and SUM over ranks of the trial counters.  This module holds that host
logic so that it can be exercised on CPU with the gloo backend (tests/test_replicas_gloo.py).
"""
import os


class Replicas:
    def __init__(self, backend="nccl"):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.on = self.world > 1
        self.backend = backend
        self.dist = None
        if self.on:
            import torch
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            if backend == "nccl":
                torch.cuda.set_device(self.local)
                dist.init_process_group("nccl", device_id=torch.device(f"cuda:{self.local}"))
            else:
                dist.init_process_group(backend)
            self.dist = dist

    @property
    def seed(self):
        """Philox / orientation seed of this rank's replica."""
        return 1 + self.rank

    def barrier(self):
        if self.on:
            self.dist.barrier()

    def reduce(self, x, op):
        """All-reduce one float over the ranks; op is 'MAX' or 'SUM'."""
        if not self.on:
            return float(x)
        import torch
        dev = f"cuda:{self.local}" if self.backend == "nccl" else "cpu"
        t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
        self.dist.all_reduce(t, op=getattr(self.dist.ReduceOp, op))
        return float(t.item())

    def aggregate(self, trials_local, seconds_local):
        """Whole-job throughput: trials of all replicas / the slowest replica's time."""
        t_max = self.reduce(seconds_local, "MAX")
        trials_all = self.reduce(trials_local, "SUM")
        return trials_all / t_max, trials_all, t_max

    def close(self):
        if self.on:
            self.dist.destroy_process_group()
