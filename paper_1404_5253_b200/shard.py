"""Host-side logic of the multi-GPU run: the path shards over independent
problems, one process per GPU, no data-path collective.  Only the timing and the unit count are
reduced over the ranks.  Works with any torch.distributed backend (nccl on the GPUs, gloo in the
CPU tests)."""
import os


def rank_world():
    """(rank, local_rank, world_size) from the torchrun environment (1-process defaults)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def lattice_seed_offset(rank):
    """Every rank builds its own lattice: same recipe, jitter seed shifted by the rank (weak scaling)."""
    return int(rank)


def assign_round_robin(items, rank, world):
    """Items (e.g. the J^pi matrices of a sweep) owned by `rank` when a job list is split over ranks."""
    return [it for k, it in enumerate(items) if k % world == rank]


def assign_balanced(items, costs, rank, world):
    """Items dealt largest cost first to the least loaded rank (ties: lowest rank); the items of `rank`, in the order of `items`.
    Every rank computes the same assignment from the same (items, costs)."""
    load = [0.0] * world
    owner = {}
    for k in sorted(range(len(items)), key=lambda k: (-float(costs[k]), k)):
        r = min(range(world), key=lambda r: (load[r], r))
        owner[k] = r
        load[r] += float(costs[k])
    return [it for k, it in enumerate(items) if owner[k] == rank]


def reduce_step(dist, device, ms_local, units_local):
    """(max over ranks of the step time in ms, sum over ranks of the units processed)."""
    import torch

    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return t.item(), u.item()


def throughput(ms_max, units_sum):
    """Whole-job units per second: all ranks' units over the slowest rank's time."""
    return units_sum / (ms_max * 1e-3)
