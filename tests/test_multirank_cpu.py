"""N > 1 path on CPU: world-size-2 gloo.  The path shards by repertoire (one donor per rank, no
data-path collective); what crosses ranks is the timing contract's max / sum."""
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


def test_two_ranks_shard_by_repertoire_and_aggregate():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, tot0, c0, h0), (r1, t1, tot1, c1, h1) = res
    assert h0 != h1                                   # different donors on different ranks
    assert t0 == t1 == 20.0                           # max over ranks
    assert tot0 == tot1
    assert tot0["pairs"] == c0 + c1 and tot0["seqs"] == 8000   # sum over ranks
    assert shard.whole_job_value(t0, tot0["pairs"]) == (c0 + c1) / 0.020


def test_single_process_is_the_identity():
    t, tot = shard.aggregate(3.5, {"pairs": 7, "seqs": 2})
    assert t == 3.5 and tot == {"pairs": 7.0, "seqs": 2.0}
