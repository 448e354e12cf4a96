"""Multi-GPU plumbing.  The checkpoint path shards with NO data exchange (
PAPER.md:L223, L392-396: every rank checkpoints its own regions into its own log at the same
collective boundary).  What ranks share is control only: the epoch id of a boundary and, for
measurement, the max-over-ranks time.  Works with any torch.distributed backend (nccl on GPUs,
gloo in the CPU tests)."""
import torch
import torch.distributed as dist


def rank_seed(base_seed: int, rank: int) -> int:
    """Every rank owns a different region: distinct, reproducible seed per rank."""
    return base_seed + 7919 * rank


def agree_epoch(local_epoch: int, device="cpu", group=None) -> int:
    """All ranks must checkpoint the same boundary: returns the common epoch id, raises if they differ.
    Control plane only (one 16-byte all-reduce); no checkpoint data crosses GPUs."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return local_epoch
    t = torch.tensor([local_epoch, -local_epoch], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    hi, lo = int(t[0].item()), -int(t[1].item())
    if hi != lo:
        raise RuntimeError("ranks disagree on the checkpoint epoch: min %d max %d" % (lo, hi))
    return hi


def job_throughput(local_units: float, local_ms: float, device="cpu", group=None):
    """Whole-job throughput = units processed by all ranks / max-over-ranks time.
    Returns (units_per_second, max_ms)."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return local_units / (local_ms * 1e-3), local_ms
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    m = torch.tensor([local_ms], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(m, op=dist.ReduceOp.MAX, group=group)
    return float(u.item()) / (float(m.item()) * 1e-3), float(m.item())
