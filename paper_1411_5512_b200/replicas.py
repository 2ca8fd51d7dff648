"""Multi-GPU plumbing: REPLICAS ONLY.

The path does not shard: one batch of 64 samples at L = 128 is 40-64 MiB and a half-sweep lasts a few
microseconds, so a spatial split would be latency-bound.  The paper itself used its two GPUs for independent
batches.  N GPUs therefore run N independent sims (different seed / p / T); there is no
collective on the data path.  The only communication is host-side bookkeeping, done with `torch.distributed`
(NCCL on GPUs, gloo in the CPU tests): which work items a rank owns, the max-over-ranks step time, and the
concatenation of the per-sample integer observables.

Nothing here touches the method's arithmetic.
"""
import os

import numpy as np


def world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def shard(items, rank, world_size):
    """Round-robin split of independent work items (seeds, (p, T) points) over ranks: item k -> rank k % world.
    Every item is owned by exactly one rank; ranks differ by at most one item."""
    if not (0 <= rank < world_size):
        raise ValueError("rank %d outside [0, %d)" % (rank, world_size))
    return [it for k, it in enumerate(items) if k % world_size == rank]


def replica_seed(base_seed, rank):
    """Independent batches: rank r simulates the batch with seed base + r (workloads.seed_for variants)."""
    return int(base_seed) + int(rank)


def init(backend=None):
    """Join the process group torchrun set up (no-op for a single process).  Returns (rank, local_rank, world)."""
    rank, local_rank, ws = world()
    if ws > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            if backend is None:
                import torch
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            dist.init_process_group(backend=backend, rank=rank, world_size=ws)
    return rank, local_rank, ws


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _device_for_collectives():
    import torch
    import torch.distributed as dist
    if dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def max_over_ranks(value):
    """max of a host float over all ranks (the step time of a multi-GPU run is its slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device_for_collectives())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device_for_collectives())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_lanes(per_lane):
    """Concatenate per-sample integer observables of all ranks: int64 [..., lanes] per rank ->
    [world, ..., lanes] on every rank (rank-major; the samples of different ranks are independent batches)."""
    import torch
    import torch.distributed as dist
    a = np.ascontiguousarray(per_lane, dtype=np.int64)
    if not (dist.is_available() and dist.is_initialized()):
        return a[None]
    dev = _device_for_collectives()
    t = torch.from_numpy(a).to(dev)
    out = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return np.stack([o.cpu().numpy() for o in out])


def aggregate_throughput(units_per_rank, seconds_per_rank):
    """Whole-job throughput bookkeeping: (total units over ranks, max time over ranks)."""
    return sum_over_ranks(units_per_rank), max_over_ranks(seconds_per_rank)
