"""N > 1 paths on CPU: world-size-2 gloo.

(1) by repertoire: one donor per rank, no data-path collective; what crosses ranks is the timing
    contract's max / sum.
(2) ONE repertoire over two ranks: the block-cyclic ownership of row batches, the count all-gather
    and the merge -- the host-side logic of paper_2602_17330_b200/shard.py.  The ranks' shares are
    produced here by the oracle restricted to the rows a rank owns (the CUDA path produces them in
    tests/test_gpu_multirank.py); merged, they must be the oracle's whole list."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2602_17330_b200 import datagen as dg
from paper_2602_17330_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # every rank draws its own repertoire and (here, on CPU) counts its work units with the oracle
    import oracle
    P = dg.PARAMS["config2"]
    rep = dg.config2(4000, seed=shard.rank_seed(rank))
    sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], dg.DEFAULT_SEED64)
    pairs, _, _ = oracle.lsh_sorted(sig, P["bands"], P["rows"], P["cap"])
    step_ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
    t, tot = shard.aggregate(step_ms, {"pairs": pairs.shape[0], "seqs": rep.n})
    dist.barrier()
    q.put((rank, t, tot, int(pairs.shape[0]), int(rep.seqs[:64].astype(np.int64).sum())))
    dist.destroy_process_group()


def _spawn(target, world, extra=()):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=target, args=(r, world, port, q) + tuple(extra)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return res


def test_two_ranks_shard_by_repertoire_and_aggregate():
    res = _spawn(_worker, 2)
    (r0, t0, tot0, c0, h0), (r1, t1, tot1, c1, h1) = res
    assert h0 != h1                                   # different donors on different ranks
    assert t0 == t1 == 20.0                           # max over ranks
    assert tot0 == tot1
    assert tot0["pairs"] == c0 + c1 and tot0["seqs"] == 8000   # sum over ranks
    assert shard.whole_job_value(t0, tot0["pairs"]) == (c0 + c1) / 0.020


def test_single_process_is_the_identity():
    t, tot = shard.aggregate(3.5, {"pairs": 7, "seqs": 2})
    assert t == 3.5 and tot == {"pairs": 7.0, "seqs": 2.0}
    assert shard.gather_counts(11) == [11]


def test_block_cyclic_ownership_partitions_the_rows():
    for n, br, world in [(10, 3, 2), (1000, 32, 8), (60_013, 6016, 2), (5, 100, 4), (0, 8, 2)]:
        seen = np.zeros(n, np.int32)
        for r in range(world):
            prev_hi = -1
            for lo, hi in shard.owned_batches(n, br, r, world):
                assert 0 <= lo < hi <= n and lo % br == 0 and lo > prev_hi
                assert shard.batch_owner(lo // br, world) == r
                seen[lo:hi] += 1
                prev_hi = hi - 1
        assert (seen == 1).all()
    assert shard.default_batch_rows(10_000_000, 8) % 32 == 0
    assert 16 * 8 * shard.default_batch_rows(10_000_000, 8) >= 10_000_000


def _shard_worker(rank, world, port, q, n, batch_rows):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    P = dg.PARAMS["config4"]
    rep = dg.config4(n, seed=5)                        # the SAME repertoire on every rank
    sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], dg.DEFAULT_SEED64)
    pairs, _, _ = oracle.lsh_sorted(sig, P["bands"], P["rows"], P["cap"])
    own = np.zeros(n, bool)
    for lo, hi in shard.owned_batches(n, batch_rows, rank, world):
        own[lo:hi] = True
    mine = pairs[own[pairs[:, 0]]]                     # this rank's share: the rows it owns
    d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, mine, P["max_d"])
    counts = shard.gather_counts(mine.shape[0])
    t, tot = shard.aggregate(5.0 + rank, {"pairs": mine.shape[0]})
    q.put((rank, counts, tot["pairs"], mine, d, int(pairs.shape[0])))
    dist.barrier()
    dist.destroy_process_group()


def test_one_repertoire_over_two_ranks_merges_to_the_whole_list():
    import oracle
    n, world = 6000, 2
    batch_rows = shard.default_batch_rows(n, world, batches_per_rank=4)
    res = _spawn(_shard_worker, world, extra=(n, batch_rows))
    counts0 = res[0][1]
    total = res[0][5]
    assert [r[3].shape[0] for r in res] == counts0 == res[1][1]        # the all-gather of the counts
    assert sum(counts0) == total == res[0][2] == res[1][2]              # disjoint shares, all pairs
    assert min(counts0) > 0.3 * total                                   # block-cyclic: balanced
    mp_, md_ = shard.merge_parts([(r[3], r[4]) for r in res], batch_rows)
    P = dg.PARAMS["config4"]
    rep = dg.config4(n, seed=5)
    sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], dg.DEFAULT_SEED64)
    want, _, _ = oracle.lsh_sorted(sig, P["bands"], P["rows"], P["cap"])
    assert np.array_equal(mp_, want)
    assert np.array_equal(md_, oracle.edit_distance_pairs(rep.seqs, rep.offsets, want, P["max_d"]))
