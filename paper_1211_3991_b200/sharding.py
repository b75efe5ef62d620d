"""Multi-GPU plumbing: graph samples are independent (PAPER.md:165,
Eq. 12 is a plain average over topologies), so the path shards BY SAMPLE, one process per GPU, with no
data-path collective.  The only exchange is a gather of the [S][R][XY_NACC] fp64 accumulators (a few KB)
when the caller wants the graph average.  No Monte-Carlo arithmetic lives here.
"""
import numpy as np


def shard_samples(S_total, world_size, rank):
    """Contiguous block of global sample ids owned by `rank`: (sample_base, S_local).  Ranks 0..rem-1 get
    one extra sample when world_size does not divide S_total; a rank may own zero samples."""
    if S_total < 0 or world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("need S_total >= 0, world_size >= 1, 0 <= rank < world_size")
    q, rem = divmod(S_total, world_size)
    base = rank * q + min(rank, rem)
    return base, q + (1 if rank < rem else 0)


def weak_shard(S_per_gpu, rank):
    """Weak scaling (bench.py): every rank runs S_per_gpu samples, global ids rank*S_per_gpu ..."""
    return rank * S_per_gpu, S_per_gpu


def gather_accumulators(acc_local, S_total, group=None):
    """All ranks contribute their [S_local][R][C] fp64 accumulators (global sample order = rank order);
    every rank gets the full [S_total][R][C] array.  Works on any torch.distributed backend (NCCL on the
    GPUs, gloo in the CPU tests); without an initialised process group it is the identity."""
    import torch
    import torch.distributed as dist
    acc_local = np.ascontiguousarray(acc_local, np.float64)
    if not (dist.is_available() and dist.is_initialized()):
        if acc_local.shape[0] != S_total:
            raise ValueError("single process must hold all samples")
        return acc_local.copy()
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    R, Ccols = acc_local.shape[1], acc_local.shape[2]
    counts = [shard_samples(S_total, world, r)[1] for r in range(world)]
    if acc_local.shape[0] != counts[rank]:
        raise ValueError(f"rank {rank} holds {acc_local.shape[0]} samples, its shard has {counts[rank]}")
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    smax = max(counts)
    pad = torch.zeros((smax, R, Ccols), dtype=torch.float64, device=dev)
    if counts[rank]:
        pad[: counts[rank]] = torch.from_numpy(acc_local).to(dev)
    out = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(out, pad, group=group)
    return np.concatenate([o[:c].cpu().numpy() for o, c in zip(out, counts)], axis=0)


def graph_average(acc_all):
    """Eq. 12: mean over samples of the per-sample time averages.  acc_all [S][R][C] with column 0 = n.
    Returns [R][C-1] (columns 1..): overline{<E>}, overline{<E^2>}, overline{<|m|>}, ..."""
    acc_all = np.asarray(acc_all, np.float64)
    n = acc_all[..., :1]
    return (acc_all[..., 1:] / n).mean(axis=0)
