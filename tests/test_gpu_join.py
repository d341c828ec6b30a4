"""Parity of sq_join / sq_join_host against oracle.join_threshold.

Integer work: identical hit sets, order (ascending (i, j)) and distances.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_17330_b200 import datagen as dg

pytestmark = pytest.mark.gpu


def _two(rep_a, rep_b, capacity, max_len=None):
    """Two contexts, A and B packed with one max_len; A's workspace sized for the join."""
    from paper_2602_17330_b200 import binding
    if max_len is None:
        max_len = int(max(rep_a.lengths.max() if rep_a.n else 1, rep_b.lengths.max() if rep_b.n else 1))
    ctxs = []
    for rep, other in ((rep_a, rep_b), (rep_b, rep_a)):
        sq = binding.SubQuad(0)
        sq.set_workspace(sq.workspace_bytes(binding.OP_JOIN, rep.n, int(rep.offsets[-1]), max_len,
                                            pair_capacity=capacity, n_other=other.n))
        seqs = torch.from_numpy(rep.seqs if rep.seqs.size else np.zeros(1, np.uint8)).cuda()
        sq.pack(seqs, torch.from_numpy(rep.offsets).cuda(), alphabet=20, max_len=max_len)
        ctxs.append(sq)
    return binding, ctxs[0], ctxs[1]


def _run_join(sa, sb, max_d, capacity, **kw):
    pairs = torch.empty((capacity, 2), dtype=torch.int32, device="cuda")
    dist = torch.empty(capacity, dtype=torch.int16, device="cuda")
    cnt = sa.join(sb, max_d, pairs, dist, **kw)
    return pairs.cpu().numpy().view(np.uint32)[:cnt], dist.cpu().numpy().view(np.uint16)[:cnt]


def test_join_two_repertoires_cdr3():
    a, b = dg.split(dg.config2(3800, seed=11), 1500)
    want_p, want_d = oracle.join_threshold(a.seqs, a.offsets, b.seqs, b.offsets, 3)
    assert want_p.shape[0] > 1000
    binding, sa, sb = _two(a, b, want_p.shape[0] + 64)
    got_p, got_d = _run_join(sa, sb, 3, want_p.shape[0] + 64)
    assert np.array_equal(got_p, want_p) and np.array_equal(got_d, want_d)
    # the other orientation is the transpose (the contexts swap roles: B's scratch is used)
    tp, td = _run_join(sb, sa, 3, want_p.shape[0] + 64)
    order = np.lexsort((want_p[:, 0], want_p[:, 1]))
    assert np.array_equal(tp, want_p[order][:, ::-1]) and np.array_equal(td, want_d[order])
    # a row range
    sub_p, sub_d = _run_join(sa, sb, 3, want_p.shape[0] + 64, a_begin=377, a_end=1033)
    m = (want_p[:, 0] >= 377) & (want_p[:, 0] < 1033)
    assert np.array_equal(sub_p, want_p[m]) and np.array_equal(sub_d, want_d[m])
    sa.close(); sb.close()


def test_join_self_upper_equals_all_pairs():
    rep = dg.config2(2500, seed=4)
    want_p, want_d = oracle.all_pairs_threshold(rep.seqs, rep.offsets, 2)
    binding, sa, sb = _two(rep, rep, want_p.shape[0] * 2 + rep.n + 64)
    got_p, got_d = _run_join(sa, sa, 2, want_p.shape[0] + 64, flags=binding.JOIN_UPPER)   # b is a itself
    assert np.array_equal(got_p, want_p) and np.array_equal(got_d, want_d)
    got_p, got_d = _run_join(sa, sb, 2, want_p.shape[0] + 64, flags=binding.JOIN_UPPER)
    assert np.array_equal(got_p, want_p) and np.array_equal(got_d, want_d)
    # the whole rectangle: both orientations and the diagonal
    full_p, full_d = _run_join(sa, sb, 2, want_p.shape[0] * 2 + rep.n + 64)
    op, od = oracle.join_threshold(rep.seqs, rep.offsets, rep.seqs, rep.offsets, 2)
    assert np.array_equal(full_p, op) and np.array_equal(full_d, od)
    sa.close(); sb.close()


def test_join_long_sequences_multiword():
    a, b = dg.split(dg.config5(900, seed=2), 350)
    want_p, want_d = oracle.join_threshold(a.seqs, a.offsets, b.seqs, b.offsets, 15)
    assert want_p.shape[0] > 500
    binding, sa, sb = _two(a, b, want_p.shape[0] + 64)
    got_p, got_d = _run_join(sa, sb, 15, want_p.shape[0] + 64)
    assert np.array_equal(got_p, want_p) and np.array_equal(got_d, want_d)
    sa.close(); sb.close()


def test_join_survivor_overflow_splits_rows():
    # permutations of one residue multiset: bag distance 0 for every pair, so every cell survives
    # the filter (700 * 900 = 630,000 > 4 * capacity + 65,536) while few are within max_d
    rng = np.random.default_rng(9)
    base = rng.integers(0, 20, 18).astype(np.uint8)
    a = dg.from_list([rng.permutation(base) for _ in range(700)])
    b = dg.from_list([rng.permutation(base) for _ in range(900)])
    want_p, want_d = oracle.join_threshold(a.seqs, a.offsets, b.seqs, b.offsets, 8)
    cap = max(64, want_p.shape[0] + 8)
    assert 4 * cap + 65536 < 700 * 900
    binding, sa, sb = _two(a, b, cap)
    got_p, got_d = _run_join(sa, sb, 8, cap)
    assert np.array_equal(got_p, want_p) and np.array_equal(got_d, want_d)
    sa.close(); sb.close()


def test_join_edges_and_errors():
    from paper_2602_17330_b200.binding import SubQuadError, SQ_ERR_CAPACITY, SQ_ERR_INVALID_ARG
    a, b = dg.split(dg.config2(900, seed=1), 400)
    want_p, want_d = oracle.join_threshold(a.seqs, a.offsets, b.seqs, b.offsets, 3)
    binding, sa, sb = _two(a, b, want_p.shape[0] + 64)
    # capacity too small: the required count comes back
    with pytest.raises(SubQuadError) as e:
        _run_join(sa, sb, 3, 10)
    assert e.value.code == SQ_ERR_CAPACITY and e.value.required == want_p.shape[0]
    # empty row range, max_d = 0 (exact duplicates only), negative max_d rejected
    p, d = _run_join(sa, sb, 3, 16, a_begin=5, a_end=5)
    assert p.shape[0] == 0
    p0, d0 = _run_join(sa, sb, 0, want_p.shape[0] + 64)
    m = want_d == 0
    assert np.array_equal(p0, want_p[m]) and np.all(d0 == 0)
    with pytest.raises(SubQuadError) as e:
        _run_join(sa, sb, -1, 16)
    assert e.value.code == SQ_ERR_INVALID_ARG
    sa.close(); sb.close()
    # an empty B, and an A with empty sequences inside
    e_rep = dg.from_list([])
    binding, sa, sb = _two(a, e_rep, 64, max_len=int(a.lengths.max()))
    p, d = _run_join(sa, sb, 3, 64)
    assert p.shape[0] == 0
    sa.close(); sb.close()
    with_empty = dg.from_list([[], [1, 2, 3], [], [1, 2], [4] * 7])
    wp, wd = oracle.join_threshold(with_empty.seqs, with_empty.offsets, with_empty.seqs, with_empty.offsets, 2)
    binding, sa, sb = _two(with_empty, with_empty, 64)
    p, d = _run_join(sa, sb, 2, 64)
    assert np.array_equal(p, wp) and np.array_equal(d, wd)
    sa.close(); sb.close()


@pytest.mark.parametrize("batch_rows,block_cap", [(0, 1 << 20), (97, 1 << 20), (1000, 3000), (5000, 700)])
def test_join_host_blocks(batch_rows, block_cap):
    a, b = dg.split(dg.config2(5200, seed=21), 2100)
    want_p, want_d = oracle.join_threshold(a.seqs, a.offsets, b.seqs, b.offsets, 3)
    binding, sa, sb = _two(a, b, block_cap)
    cap = want_p.shape[0] + 16
    ph = torch.empty((cap, 2), dtype=torch.int32).pin_memory()
    dh = torch.empty(cap, dtype=torch.int16).pin_memory()
    cnt = sa.join_host(sb, 3, ph, dh, block_capacity=block_cap, batch_rows=batch_rows)
    assert cnt == want_p.shape[0]
    assert np.array_equal(ph.numpy().view(np.uint32)[:cnt], want_p)
    assert np.array_equal(dh.numpy().view(np.uint16)[:cnt], want_d)
    # host capacity too small: required total returned
    from paper_2602_17330_b200.binding import SubQuadError, SQ_ERR_CAPACITY
    with pytest.raises(SubQuadError) as e:
        sa.join_host(sb, 3, ph[:100], dh[:100], block_capacity=block_cap, batch_rows=batch_rows)
    assert e.value.code == SQ_ERR_CAPACITY and e.value.required == want_p.shape[0]
    sa.close(); sb.close()


def test_join_full_size_sampled_rows():
    """Cross-repertoire shape of PAPER.md L647 (a 1 M pool): 100,000 x 900,000 CDR3s, max_d = 2;
    sampled rows against the oracle's join of those rows with all of B."""
    a, b = dg.split(dg.config3(1_000_000, seed=0), 100_000)
    cap = 60_000_000
    binding, sa, sb = _two(a, b, cap)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
    dist = torch.empty(cap, dtype=torch.int16, device="cuda")
    cnt = sa.join(sb, 2, pairs, dist)
    assert cnt > 1_000_000
    P = pairs[:cnt].cpu().numpy().view(np.uint32)
    D = dist[:cnt].cpu().numpy().view(np.uint16)
    key = P[:, 0].astype(np.int64) * b.n + P[:, 1]
    assert np.all(np.diff(key) > 0)                       # ascending (i, j), no duplicate
    assert D.max() <= 2
    rows = np.random.default_rng(3).choice(a.n, 12, replace=False)
    sub = dg.from_list([a.seq(int(r)) for r in rows])
    wp, wd = oracle.join_threshold(sub.seqs, sub.offsets, b.seqs, b.offsets, 2)
    for t, r in enumerate(rows):
        lo, hi = np.searchsorted(P[:, 0], [r, r + 1])
        m = wp[:, 0] == t
        assert np.array_equal(P[lo:hi, 1], wp[m, 1]) and np.array_equal(D[lo:hi], wd[m])
    sa.close(); sb.close()


@pytest.mark.parametrize("cfg,n_total,n_a,max_d", [("config2", 7300, 1100, 3), ("config3", 9000, 1500, 2),
                                                   ("config5", 4400, 150, 15)])
def test_join_columns_sorted_by_length(cfg, n_total, n_a, max_d):
    """With >= 4,096 columns the filter walks B in order of length (blocks skip rows whose length is
    out of reach); the result must not change."""
    a, b = dg.split(dg.GENERATORS[cfg](n_total, seed=13), n_a)
    assert b.n >= 4096
    want_p, want_d = oracle.join_threshold(a.seqs, a.offsets, b.seqs, b.offsets, max_d)
    assert want_p.shape[0] > 200
    binding, sa, sb = _two(a, b, want_p.shape[0] + 64)
    got_p, got_d = _run_join(sa, sb, max_d, want_p.shape[0] + 64)
    assert np.array_equal(got_p, want_p) and np.array_equal(got_d, want_d)
    sa.close(); sb.close()
