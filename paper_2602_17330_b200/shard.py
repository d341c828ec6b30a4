"""How the path runs on N GPUs.  One process per GPU.

Two partitionings, both without a collective on the data path:

* by repertoire (bench.py's weak-scaling arm): one independent repertoire (donor) per rank.
* ONE repertoire over G ranks (`sharded_candidates`): every rank packs and sketches the whole
  repertoire and runs band keys, bucket sort and bucket scan on it (replicated: about a sixth of the
  step), then emits, orders and verifies only the candidate rows it owns -- the batches b of
  `batch_rows` consecutive ids with b % G == rank (block-cyclic: row i pairs only with j > i, so low
  ids carry more pairs).  Pairs never cross ranks, so nothing is exchanged; what crosses ranks is
  bookkeeping: the per-rank counts (one all-gather) and the timing contract's max / sum.

Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests); with no process group
every helper is the identity.  Argument marshalling and bookkeeping only -- no arithmetic of the
method lives here."""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def rank_seed(rank: int) -> int:
    """Seed of the repertoire rank `rank` draws (rank r = donor r)."""
    return int(rank)


def _active() -> bool:
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def aggregate(step_ms: float, units: dict, device=None) -> tuple[float, dict]:
    """(max over ranks of step_ms, {name: sum over ranks}) -- every rank gets the result."""
    names = sorted(units)
    if not _active():
        return float(step_ms), {k: float(units[k]) for k in names}
    t = torch.tensor([float(step_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units[k]) for k in names], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), {k: float(v) for k, v in zip(names, u.tolist())}


def whole_job_value(step_ms_max: float, total_units: float) -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's step time."""
    return total_units / (step_ms_max * 1e-3)


# ---- one repertoire over G ranks -----------------------------------------------------------------
def batch_owner(batch: int, world: int) -> int:
    """Rank that emits and verifies batch `batch` (rows [batch * batch_rows, (batch + 1) * batch_rows))."""
    return int(batch) % int(world)


def owned_batches(n: int, batch_rows: int, rank: int, world: int) -> list[tuple[int, int]]:
    """Row ranges [lo, hi) rank `rank` owns, ascending."""
    nb = (n + batch_rows - 1) // batch_rows if n > 0 else 0
    return [(b * batch_rows, min(n, (b + 1) * batch_rows)) for b in range(rank, nb, world)]


def default_batch_rows(n: int, world: int, batches_per_rank: int = 16) -> int:
    """Batch size that deals every rank `batches_per_rank` batches (a multiple of 32 rows)."""
    per = max(1, -(-n // (world * batches_per_rank)))
    return (per + 31) // 32 * 32


def gather_counts(count: int, device=None) -> list[int]:
    """Every rank's pair count, on every rank (the one collective of the sharded path)."""
    if not _active():
        return [int(count)]
    t = torch.tensor([int(count)], dtype=torch.int64, device=device)
    out = [torch.zeros_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return [int(x.item()) for x in out]


def merge_parts(parts: list[tuple[np.ndarray, np.ndarray]], batch_rows: int):
    """Interleave the ranks' outputs back into the single ascending (i, j) list: rank r holds its
    batches in ascending order, each batch ascending in (i, j); batch b precedes batch b + 1.
    parts[r] = (pairs uint32[c_r][2], dist uint16[c_r]).  Bookkeeping for consumers and tests."""
    pairs = np.concatenate([p for p, _ in parts]) if parts else np.zeros((0, 2), np.uint32)
    dists = np.concatenate([d for _, d in parts]) if parts else np.zeros(0, np.uint16)
    order = np.argsort(pairs[:, 0].astype(np.int64) // int(batch_rows), kind="stable")
    return pairs[order], dists[order]


def sharded_candidates(sq, sig, P: dict, max_d: int, pairs_host, dist_host, block_capacity: int,
                       batch_rows: int, rank: int | None = None, world: int | None = None):
    """This rank's share of ONE repertoire's candidates + distances, into its host buffers, through
    sq_candidates_stream_host.  `sq` must hold the WHOLE repertoire (sq.pack) and `sig` all its
    signatures.  Returns (count of this rank, raw pairs over all rows, every rank's count)."""
    if rank is None:
        rank = dist.get_rank() if _active() else 0
    if world is None:
        world = dist.get_world_size() if _active() else 1
    cnt, raw = sq.candidates_stream_host(sig, P["bands"], P["rows"], P["cap"], max_d, pairs_host, dist_host,
                                         block_capacity, batch_rows=batch_rows, part=rank, n_parts=world)
    return cnt, raw, gather_counts(cnt, device=None if not torch.cuda.is_available() else sig.device
                                   if dist.is_initialized() and dist.get_backend() == "nccl" else None)
