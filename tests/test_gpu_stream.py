"""sq_lsh_prepare / sq_lsh_emit_range / sq_candidates_stream_host:
the candidate list emitted piecewise -- by row range, out-of-core through a deliberately tiny device
block, and block-cyclic over two parts -- must reproduce the oracle's whole list and distances."""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_17330_b200 import datagen as dg
from paper_2602_17330_b200 import shard

pytestmark = pytest.mark.gpu
SEED = dg.DEFAULT_SEED64


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def _setup(cfg, n, seed, pair_capacity, extra=0):
    from paper_2602_17330_b200 import binding
    P = dict(dg.PARAMS[cfg])
    rep = dg.GENERATORS[cfg](n, seed=seed)
    sq = binding.SubQuad(0)
    max_len = int(rep.lengths.max())
    sq.set_workspace(sq.workspace_bytes(binding.OP_LSH, rep.n, int(rep.offsets[-1]), max_len, P["H"], P["bands"],
                                        P["cap"], pair_capacity) + extra)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    sig = sq.minhash(P["k"], P["H"], SEED)
    want_p, want_raw, _ = oracle.lsh_sorted(_u32(sig), P["bands"], P["rows"], P["cap"])
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, want_p, P["max_d"])
    return binding, sq, P, rep, sig, want_p, want_raw, want_d


@pytest.mark.parametrize("cfg,n", [("config2", 30_011), ("config4", 40_009)])
def test_emit_range_pieces_concatenate_to_the_whole_list(cfg, n):
    binding, sq, P, rep, sig, want_p, want_raw, want_d = _setup(cfg, n, 41, 200 * n)
    raw = sq.lsh_prepare(sig, P["bands"], P["rows"], P["cap"])
    assert raw == want_raw
    buf = torch.empty((want_p.shape[0] + 8, 2), dtype=torch.int32, device="cuda")
    rng = np.random.default_rng(1)
    cuts = np.unique(np.concatenate([[0, 1, 2, n - 1, n], rng.integers(0, n, 9)]))
    got = []
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        c = sq.lsh_emit_range(int(lo), int(hi), buf)
        p = _u32(buf[:c]).copy()
        assert ((p[:, 0] >= lo) & (p[:, 0] < hi)).all()
        # the schedule left by every emit call drives the DP of that piece (forced on)
        sq.set_option(binding.OPT_SCHED_MIN_BYTES, 0)
        d = sq.edit_distance(buf, c, P["max_d"])
        sel = (want_p[:, 0] >= lo) & (want_p[:, 0] < hi)
        assert np.array_equal(p, want_p[sel])
        assert np.array_equal(d[:c].cpu().numpy().view(np.uint16), want_d[sel])
        got.append(p)
    assert np.array_equal(np.concatenate(got), want_p)
    # ranges in any order, repeated, empty; the whole range equals sq_lsh_candidates
    assert sq.lsh_emit_range(5, 5, buf) == 0
    c = sq.lsh_emit_range(0, n, buf, flags=binding.LSH_UNORDERED)
    p = _u32(buf[:c])
    assert c == want_p.shape[0]
    key = np.sort(p[:, 0].astype(np.int64) << 32 | p[:, 1])
    assert np.array_equal(key, want_p[:, 0].astype(np.int64) << 32 | want_p[:, 1])
    with pytest.raises(binding.SubQuadError) as ei:               # capacity protocol per range
        sq.lsh_emit_range(0, n, buf[:10])
    assert ei.value.code == binding.SQ_ERR_CAPACITY and ei.value.required == want_p.shape[0]
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, int(rep.lengths.max()))
    with pytest.raises(binding.SubQuadError) as ei:               # the prepared state died with the re-pack
        sq.lsh_emit_range(0, n, buf)
    assert ei.value.code == binding.SQ_ERR_NOT_PACKED
    sq.close()


@pytest.mark.parametrize("block_capacity,batch_rows", [(20_000, 0), (3_000, 4_096), (150_000, 1_000)])
def test_streamed_candidates_through_a_tiny_device_block(block_capacity, batch_rows):
    """Config 2 at full size (2.4 M candidates) through a device block of a few thousand pairs: the
    host buffers end up holding exactly the oracle's list and distances."""
    n = 100_000
    binding, sq, P, rep, sig, want_p, want_raw, want_d = _setup("config2", n, 0, block_capacity,
                                                                 extra=20 * block_capacity + 4096)
    cap = want_p.shape[0] + 16
    ph = torch.zeros((cap, 2), dtype=torch.int32).pin_memory()
    dh = torch.zeros(cap, dtype=torch.int16).pin_memory()
    cnt, raw = sq.candidates_stream_host(sig, P["bands"], P["rows"], P["cap"], P["max_d"], ph, dh,
                                         block_capacity, batch_rows=batch_rows)
    assert cnt == want_p.shape[0] and raw == want_raw
    assert np.array_equal(ph.numpy().view(np.uint32)[:cnt], want_p)
    assert np.array_equal(dh.numpy().view(np.uint16)[:cnt], want_d)
    with pytest.raises(binding.SubQuadError) as ei:               # host capacity protocol
        sq.candidates_stream_host(sig, P["bands"], P["rows"], P["cap"], P["max_d"], ph[:1000], dh[:1000],
                                  block_capacity, batch_rows=batch_rows)
    assert ei.value.code == binding.SQ_ERR_CAPACITY and ei.value.required == cnt
    sq.close()


def test_a_single_row_larger_than_the_block_is_reported():
    rep = dg.from_list([[1, 2, 3, 4, 5, 6, 7, 8]] * 300)          # one bucket: row 0 has 299 partners
    from paper_2602_17330_b200 import binding
    sq = binding.SubQuad(0)
    sq.set_workspace(sq.workspace_bytes(binding.OP_LSH, rep.n, int(rep.offsets[-1]), 8, 32, 8, 1000, 100) + (1 << 20))
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, 8)
    sig = sq.minhash(3, 32, SEED)
    ph = torch.zeros((50_000, 2), dtype=torch.int32).pin_memory()
    dh = torch.zeros(50_000, dtype=torch.int16).pin_memory()
    with pytest.raises(binding.SubQuadError) as ei:
        sq.candidates_stream_host(sig, 8, 4, 1000, 1, ph, dh, 100, batch_rows=64)
    assert ei.value.code == binding.SQ_ERR_CAPACITY
    cnt, raw = sq.candidates_stream_host(sig, 8, 4, 1000, 1, ph, dh, 300, batch_rows=64)
    assert cnt == 300 * 299 // 2 and raw == 8 * cnt
    sq.close()


def test_two_parts_block_cyclic_merge_to_the_whole_list():
    """The sharding of ONE repertoire over G = 2 ranks, run here as two calls on one
    GPU: part g gets the batches b % 2 == g; merged by batch they are the oracle's list."""
    n = 60_013
    binding, sq, P, rep, sig, want_p, want_raw, want_d = _setup("config4", n, 3, 400_000, extra=20 * 400_000 + 4096)
    batch_rows = shard.default_batch_rows(n, 2, batches_per_rank=5)
    parts = []
    for g in range(2):
        ph = torch.zeros((want_p.shape[0] + 16, 2), dtype=torch.int32).pin_memory()
        dh = torch.zeros(want_p.shape[0] + 16, dtype=torch.int16).pin_memory()
        cnt, raw = sq.candidates_stream_host(sig, P["bands"], P["rows"], P["cap"], P["max_d"], ph, dh, 400_000,
                                             batch_rows=batch_rows, part=g, n_parts=2)
        assert raw == want_raw
        p = ph.numpy().view(np.uint32)[:cnt].copy()
        owner = (p[:, 0] // batch_rows) % 2
        assert (owner == g).all()
        parts.append((p, dh.numpy().view(np.uint16)[:cnt].copy()))
    assert sum(p.shape[0] for p, _ in parts) == want_p.shape[0]
    mp, md = shard.merge_parts(parts, batch_rows)
    assert np.array_equal(mp, want_p) and np.array_equal(md, want_d)
    sq.close()
