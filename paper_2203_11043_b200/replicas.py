"""N > 1 GPUs: replicas only.  BASELINE.json's north_star fixes one GPU per event with no sharding or
collectives, so the multi-GPU path is host logic: which events a rank runs, which seed its event uses, and how the
per-rank timings and work counts combine into the whole-job number (max over ranks of the device time, sum of the
work).  No data-path collective exists; torch.distributed is used for the timing barrier and these two reductions,
on whatever backend the caller initialised (nccl on the GPU box, gloo in the CPU tests)."""
import numpy as np


def rank_seed(base_seed, rank):
    """One independent event per rank: rank r simulates the workload drawn with seed base_seed + r."""
    return int(base_seed) + int(rank)


def shard_events(n_events, rank, world):
    """Contiguous, balanced slice [lo, hi) of a batch of independent events for this rank (sizes differ by <= 1)."""
    n_events, rank, world = int(n_events), int(rank), int(world)
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    base, extra = divmod(n_events, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_offsets(offsets, rank, world):
    """Event offsets (n_events+1) -> (carrier_lo, carrier_hi, local offsets starting at 0) of this rank's slice."""
    off = np.asarray(offsets, dtype=np.uint64)
    lo, hi = shard_events(len(off) - 1, rank, world)
    return int(off[lo]), int(off[hi]), (off[lo:hi + 1] - off[lo]).astype(np.uint64)


def aggregate(ms_local, units_local, device="cpu"):
    """(max over ranks of ms, sum over ranks of units).  Without an initialised process group: the inputs."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def whole_job_rate(ms_local, units_local, device="cpu"):
    """Whole-job throughput in units/s: all ranks' units over the slowest rank's device time."""
    ms, units = aggregate(ms_local, units_local, device)
    return units / (ms * 1e-3), ms, units
