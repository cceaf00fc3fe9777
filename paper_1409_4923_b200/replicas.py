"""Host-side logic of the N > 1 launch ("replicas only").

BASELINE.json fixes the path to one GPU with no sharding and no collective, so `bench.py --gpus N` runs N independent
replicas of the workload, one process per GPU.  What the ranks share is plumbing only: a distinct seed per rank
(distinct ensembles), and the MAX over ranks of the device-timed duration.  No arithmetic of the method lives here.
"""


def replica_seed(base_seed, rank):
    """Seed of replica `rank`: Philox keys differ in their low word, so the ensembles are independent."""
    return (int(base_seed) + int(rank)) & 0xFFFFFFFFFFFFFFFF


def max_over_ranks(value, dist=None, device=None):
    """MAX all-reduce of a scalar (elapsed milliseconds); identity when there is no process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank, world, ms_per_step):
    """Aggregate throughput of `world` replicas that each process `units_per_rank` units per step."""
    return world * units_per_rank / (ms_per_step * 1e-3)
