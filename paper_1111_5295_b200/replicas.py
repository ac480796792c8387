"""Multi-GPU = replicas only: the path has no exchange step on one node, so N ranks
run N independent copies of the workload.  This module holds the only cross-rank logic there
is: the max-over-ranks time and the whole-job unit count that bench.py reports."""
import torch
import torch.distributed as dist


def aggregate(ms, e2e_s, n_sub, n_cross, device="cpu"):
    """-> (max ms, max e2e seconds, total sub-steps, total crossings) over all ranks.
    Works on any initialised process group (nccl on GPUs, gloo in the CPU tests); without a
    process group it returns its arguments."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), float(e2e_s), float(n_sub), float(n_cross)
    t = torch.tensor([ms, e2e_s, float(n_sub), float(n_cross)], dtype=torch.float64, device=device)
    tmax, tsum = t.clone(), t.clone()
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(tmax[1]), float(tsum[2]), float(tsum[3])


def rank_seed(base_seed, rank):
    """Every replica draws its own particles and field phases."""
    return int(base_seed) + int(rank)
