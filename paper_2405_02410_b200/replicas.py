"""Multi-GPU host logic: REPLICAS ONLY.

Every FFT of the step couples all lattice sites, so the path does not shard without an all-to-all per
transform, and north_star fixes one GPU per realisation with no collective.  What parallelises is the
ensemble: rank r advances its own realisation (seed + r).  The only cross-rank traffic is the timing
reduction below (max over ranks of the device-timed totals); it is not on the data path.

No arithmetic of the method lives here.  Works on any torch.distributed backend (nccl on the GPU box,
gloo in the CPU tests).
"""
import torch
import torch.distributed as dist


def rank_config(cfg, rank):
    """the workload of rank ``rank``: the same equation and lattice, an independent noise/IC seed"""
    out = dict(cfg)
    out["seed"] = int(cfg["seed"]) + int(rank)
    return out


def reduce_timings(times, units, device=None):
    """times: list of this rank's timed totals (ms or s); units: work units this rank processed.
    Returns ([max over ranks of each time], total units of all ranks)."""
    t = torch.tensor([float(x) for x in times], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], float(u.item())
