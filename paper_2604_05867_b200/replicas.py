"""Host-side logic of the multi-GPU arm (replicas only, no data-path collective).

Rank r runs an independent BA problem (one d of BASELINE.json configs[2]'s sweep); the only exchange is
the max-over-ranks of the device time.  No method arithmetic lives here.
"""

D_REPLICAS = (0.70, 0.64, 0.75, 0.80, 0.85, 0.90, 0.95, 0.60)   # rank r runs d = D_REPLICAS[r % 8]


def replica_d(rank, world, d_single):
    """d of the problem rank `rank` runs: the headline d alone, one d of the sweep per rank otherwise."""
    return d_single if world == 1 else D_REPLICAS[rank % len(D_REPLICAS)]


def max_over_ranks(value, world, device=None):
    """MAX all-reduce of one float over the default process group (gloo on CPU, nccl on GPUs)."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank, seconds_local, world, device=None):
    """Whole-job throughput: units all ranks processed / max-over-ranks time (weak scaling)."""
    t = max_over_ranks(seconds_local, world, device)
    return units_per_rank * world / t, t
