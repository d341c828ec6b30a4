"""ONE repertoire over two ranks through the CUDA path: two processes, one per rank,
each with its own context -- here both on cuda:0 (the box has one GPU; the ranks' kernels never wait
on one another, the only collective is the all-gather of the counts, gloo on the host here, nccl on
a multi-GPU node).  The two shares, merged by batch, must equal oracle.lsh_sorted + Wagner-Fischer on
the whole repertoire, bit for bit."""
import os
import socket
import tempfile

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2602_17330_b200 import datagen as dg
from paper_2602_17330_b200 import shard

pytestmark = pytest.mark.gpu
N, WORLD, BLOCK = 80_021, 2, 600_000


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _rank(rank, world, port, outdir, batch_rows):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2602_17330_b200 import binding
    P = dg.PARAMS["config4"]
    rep = dg.config4(N, seed=9)                        # every rank holds the whole repertoire
    sq = binding.SubQuad(0)
    max_len = int(rep.lengths.max())
    sq.set_workspace(sq.workspace_bytes(binding.OP_LSH, rep.n, int(rep.offsets[-1]), max_len, P["H"], P["bands"],
                                        P["cap"], BLOCK) + 20 * BLOCK + 4096)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    sig = sq.minhash(P["k"], P["H"], dg.DEFAULT_SEED64)
    cap = 200 * N
    ph = torch.zeros((cap, 2), dtype=torch.int32).pin_memory()
    dh = torch.zeros(cap, dtype=torch.int16).pin_memory()
    cnt, raw, counts = shard.sharded_candidates(sq, sig, P, P["max_d"], ph, dh, BLOCK, batch_rows, rank, world)
    assert counts[rank] == cnt
    np.save(os.path.join(outdir, f"pairs{rank}.npy"), ph.numpy().view(np.uint32)[:cnt])
    np.save(os.path.join(outdir, f"dist{rank}.npy"), dh.numpy().view(np.uint16)[:cnt])
    np.save(os.path.join(outdir, f"meta{rank}.npy"), np.array([raw] + counts, np.int64))
    if rank == 0:
        np.save(os.path.join(outdir, "sig.npy"), sig.cpu().numpy().view(np.uint32))
    sq.close()
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_one_repertoire_equal_the_oracle():
    import oracle
    batch_rows = shard.default_batch_rows(N, WORLD, batches_per_rank=6)
    port = _free_port()
    ctx = mp.get_context("spawn")
    with tempfile.TemporaryDirectory() as outdir:
        procs = [ctx.Process(target=_rank, args=(r, WORLD, port, outdir, batch_rows)) for r in range(WORLD)]
        for p in procs:
            p.start()
        for p in procs:
            p.join(timeout=600)
            assert p.exitcode == 0
        parts = [(np.load(os.path.join(outdir, f"pairs{r}.npy")), np.load(os.path.join(outdir, f"dist{r}.npy")))
                 for r in range(WORLD)]
        metas = [np.load(os.path.join(outdir, f"meta{r}.npy")) for r in range(WORLD)]
        sig = np.load(os.path.join(outdir, "sig.npy"))
    P = dg.PARAMS["config4"]
    rep = dg.config4(N, seed=9)
    assert np.array_equal(sig, oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], dg.DEFAULT_SEED64))
    want_p, want_raw, _ = oracle.lsh_sorted(sig, P["bands"], P["rows"], P["cap"])
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, want_p, P["max_d"])
    assert all(int(m[0]) == want_raw for m in metas)
    assert list(metas[0][1:]) == list(metas[1][1:]) == [p.shape[0] for p, _ in parts]
    assert sum(p.shape[0] for p, _ in parts) == want_p.shape[0]
    mp_, md_ = shard.merge_parts(parts, batch_rows)
    assert np.array_equal(mp_, want_p)
    assert np.array_equal(md_, want_d)
    share = [p.shape[0] / want_p.shape[0] for p, _ in parts]
    assert min(share) > 0.3                                            # block-cyclic ownership balances the ranks
