"""How the path runs on N GPUs: one process per GPU, one independent repertoire (donor) per rank,
no data-path collective.  Only the bookkeeping of the timing contract crosses ranks: the step time
is the MAX over ranks, the work units are SUMMED.  Works on any torch.distributed backend (nccl on
GPUs, gloo in the CPU tests); with no process group it is the identity."""
from __future__ import annotations

import torch
import torch.distributed as dist


def rank_seed(rank: int) -> int:
    """Seed of the repertoire rank `rank` draws (rank r = donor r)."""
    return int(rank)


def aggregate(step_ms: float, units: dict, device=None) -> tuple[float, dict]:
    """(max over ranks of step_ms, {name: sum over ranks}) -- every rank gets the result."""
    names = sorted(units)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(step_ms), {k: float(units[k]) for k in names}
    t = torch.tensor([float(step_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units[k]) for k in names], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), {k: float(v) for k, v in zip(names, u.tolist())}


def whole_job_value(step_ms_max: float, total_units: float) -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's step time."""
    return total_units / (step_ms_max * 1e-3)
