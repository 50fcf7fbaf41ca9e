"""Channel sharding across ranks: coarse channels are independent
(PAPER.md:47, :53 -- one channel per GPU in the paper), so multi-GPU is plain data parallelism
with no collective on the data path.  Host logic only; used by bench.py and tested on gloo."""


def shard_channels(n_coarse_total, world, rank):
    """Contiguous, balanced partition of channels [0, n_coarse_total) over `world` ranks.
    Returns (first_channel, count); the first n_coarse_total % world ranks get one extra."""
    if world < 1 or not (0 <= rank < world) or n_coarse_total < 0:
        raise ValueError("bad sharding arguments")
    base, extra = divmod(n_coarse_total, world)
    count = base + (1 if rank < extra else 0)
    first = rank * base + min(rank, extra)
    return first, count


def weak_scaling_shard(channels_per_rank, rank):
    """bench.py's weak-scaling layout: every rank owns `channels_per_rank` channels."""
    return rank * channels_per_rank, channels_per_rank


def job_throughput_gbs(bytes_per_rank_per_step, steps, elapsed_ms_per_rank, dist=None):
    """Whole-job input GB/s = bytes all ranks processed / the slowest rank's time.  With a
    process group, sums the bytes and takes the max of the times over ranks."""
    total_bytes = float(bytes_per_rank_per_step) * steps
    ms = float(elapsed_ms_per_rank)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        import torch
        t = torch.tensor([total_bytes], dtype=torch.float64)
        m = torch.tensor([ms], dtype=torch.float64)
        if dist.get_backend() == "nccl":
            t, m = t.cuda(), m.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        dist.all_reduce(m, op=dist.ReduceOp.MAX)
        total_bytes, ms = float(t.item()), float(m.item())
    return total_bytes / (ms * 1e-3) / 1e9, ms
