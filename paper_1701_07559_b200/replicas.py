"""Multi-GPU = replicas only: the path's independent units are right-hand sides; every rank
holds the gauge field and solves its own sources, with no collective on the data path.  This module holds the
rank -> right-hand-side assignment and the aggregation of the ranks' counters that bench.py reports; it works on
any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
import torch


def columns_for_rank(n_columns: int, rank: int, world: int):
    """Indices of the right-hand sides (e.g. the 12 spin-colour columns of a point source) rank `rank` solves:
    round-robin, so that the ranks' counts differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world of %d" % (rank, world))
    return list(range(rank, n_columns, world))


def source_seed(base_seed: int, rank: int) -> int:
    """Seed of the Gaussian source of rank `rank` (distinct right-hand sides, same gauge field)."""
    return base_seed + 17 * rank


def aggregate(work: float, seconds: float, device="cpu"):
    """(sum over ranks of work, max over ranks of seconds): whole-job throughput = sum / max."""
    import torch.distributed as dist
    w = torch.tensor([work], dtype=torch.float64, device=device)
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(w, op=dist.ReduceOp.SUM)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(w.item()), float(t.item())
