"""Host-side plumbing for running the path on several GPUs: replicas only.

Events are independent and the path has no exchange step, so
ranks never communicate on the data path.  What is shared
is (a) which events a rank processes and (b) the reduction of the timings:
the job's time is the MAX over ranks, its throughput the SUM of the events all
ranks processed divided by that time.  torch.distributed is used for (b) only.
"""


def event_range(rank: int, world: int, events_per_rank: int):
    """Weak scaling: rank r owns events [r*n, (r+1)*n) of the (seeded, unbounded) event stream."""
    if not (0 <= rank < world) or events_per_rank < 0:
        raise ValueError("bad rank/world/events_per_rank")
    first = rank * events_per_rank
    return first, first + events_per_rank


def max_over_ranks(values, device=None):
    """Element-wise MAX of a list of floats over all ranks (identity when not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1):
        return [float(x) for x in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def job_throughput(events_per_rank: int, world: int, ms_max_over_ranks: float) -> float:
    """events/s of the whole job: all ranks' events over the slowest rank's time."""
    return world * events_per_rank / (ms_max_over_ranks * 1e-3)
