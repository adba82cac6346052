"""Multi-GPU host logic ("Multi-GPU"): the path shards over disorder realisations
(PAPER.md:266-270 adds n_dis as a pure batch axis), one process per GPU, no data-path collective.
Rank r owns the global disorders [r * n_dis, (r + 1) * n_dis); the Philox counters and the instance
seeds are indexed by the GLOBAL disorder, so a sharded job draws exactly what one process would.
The only communication is the reduction of the job's wall time (max) and counts (sum) for the report.
No arithmetic of the method lives here."""
import torch
import torch.distributed as dist


def first_disorder(rank, n_dis_per_rank):
    """global index of this rank's disorder 0 (passed to tnmc_create as first_disorder)"""
    return int(rank) * int(n_dis_per_rank)


def reduce_job(ms_local, count_local, device="cpu"):
    """(max over ranks of ms_local, sum over ranks of count_local); identity without a process group"""
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    a = torch.tensor([float(count_local)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(a, op=dist.ReduceOp.SUM)
    return t.item(), a.item()
