"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

All work is integer: the bar is bit-exact signatures, identical candidate-pair sets (and
order, which the ABI fixes to ascending (i, j)) and identical distances.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_17330_b200 import datagen as dg

pytestmark = pytest.mark.gpu
SEED = dg.DEFAULT_SEED64


def _ctx():
    from paper_2602_17330_b200 import binding
    return binding, binding.SubQuad(0)


def _pack(sq, binding, rep, bands=0, cap=0, pair_capacity=0, max_len=None, op=None, H=0):
    max_len = int(rep.lengths.max()) if max_len is None and rep.n else (max_len or 0)
    op = binding.OP_LSH if op is None else op
    ws = sq.workspace_bytes(op, rep.n, int(rep.offsets[-1]), max_len, H, max(bands, 1), cap,
                            pair_capacity)
    sq.set_workspace(ws)
    seqs = torch.from_numpy(rep.seqs if rep.seqs.size else np.zeros(1, np.uint8)).cuda()
    offs = torch.from_numpy(rep.offsets).cuda()
    sq.pack(seqs, offs, alphabet=20, max_len=max_len)
    return seqs, offs


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def _u16(t):
    return t.cpu().numpy().view(np.uint16)


# ---------------------------------------------------------------------------------------------
# config 1: exhaustive all pairs + MinHash k=3 H=32
# ---------------------------------------------------------------------------------------------
def test_config1_minhash_and_all_pairs():
    binding, sq = _ctx()
    rep = dg.config1()
    n = rep.n
    npairs = n * (n - 1) // 2
    _pack(sq, binding, rep, op=binding.OP_ALL_PAIRS, pair_capacity=npairs)
    sig = sq.minhash(3, 32, SEED)
    want = oracle.minhash(rep.seqs, rep.offsets, 3, 32, SEED)
    assert np.array_equal(_u32(sig), want)
    dist = torch.empty(npairs, dtype=torch.int16, device="cuda")
    cnt = sq.all_pairs(-1, None, dist)
    assert cnt == npairs
    full = oracle.all_pairs_full(rep.seqs, rep.offsets)
    assert np.array_equal(_u16(dist), full)
    # thresholded tile path == filter of the full matrix (config-1 size)
    for md in (4, 7):
        sel = np.nonzero(full <= md)[0]
        pairs = torch.empty((sel.size + 16, 2), dtype=torch.int32, device="cuda")
        d2 = torch.empty(sel.size + 16, dtype=torch.int16, device="cuda")
        cnt = sq.all_pairs(md, pairs, d2)
        assert cnt == sel.size
        ii, jj = np.triu_indices(n, 1)
        got = _u32(pairs)[:cnt]
        assert np.array_equal(got[:, 0], ii[sel]) and np.array_equal(got[:, 1], jj[sel])
        assert np.array_equal(_u16(d2)[:cnt], full[sel])
    # explicit pair list == all-pairs
    ii, jj = np.triu_indices(n, 1)
    take = np.random.default_rng(0).choice(npairs, 200000, replace=False)
    pl = np.stack([ii[take], jj[take]], 1).astype(np.uint32)
    d = sq.edit_distance(torch.from_numpy(pl.view(np.int32)).cuda(), pl.shape[0], -1)
    assert np.array_equal(_u16(d)[:pl.shape[0]], full[take])
    sq.close()


@pytest.mark.parametrize("k,H", [(3, 32), (3, 64), (4, 128), (5, 256), (6, 96), (1, 32)])
def test_minhash_shapes(k, H):
    binding, sq = _ctx()
    rep = dg.config3(20011, seed=3)          # ragged tail: not a multiple of the block size
    _pack(sq, binding, rep, op=binding.OP_MINHASH)
    sig = sq.minhash(k, H, SEED ^ 0xABCDEF)
    want = oracle.minhash(rep.seqs, rep.offsets, k, H, SEED ^ 0xABCDEF)
    assert np.array_equal(_u32(sig), want)
    sq.close()


def test_minhash_long_slots_and_single_sequence():
    """Slots longer than one 32-byte sector (stride 144: the word pipeline of the sketch kernel
    walks 36 words) and a one-sequence input (every other thread of the block idles)."""
    binding, sq = _ctx()
    rep = dg.config5(1_003, seed=5)          # lengths 100-140
    _pack(sq, binding, rep, op=binding.OP_MINHASH)
    sig = sq.minhash(4, 64, SEED)
    assert np.array_equal(_u32(sig), oracle.minhash(rep.seqs, rep.offsets, 4, 64, SEED))
    sq.close()
    binding, sq = _ctx()
    one = dg.config2(1, seed=9)
    _pack(sq, binding, one, op=binding.OP_MINHASH)
    sig = sq.minhash(3, 64, SEED)
    assert np.array_equal(_u32(sig), oracle.minhash(one.seqs, one.offsets, 3, 64, SEED))
    sq.close()


# ---------------------------------------------------------------------------------------------
# configs 2-4 shapes: minhash -> lsh -> edit distance
# ---------------------------------------------------------------------------------------------
def _run_path(rep, P, capacity, flags=0, sort_key_bytes=None):
    binding, sq = _ctx()
    if sort_key_bytes is not None:
        sq.set_option(binding.OPT_SORT_KEY_BYTES, sort_key_bytes)
    _pack(sq, binding, rep, bands=P["bands"], cap=P["cap"], pair_capacity=capacity, H=P["H"])
    sig = sq.minhash(P["k"], P["H"], SEED)
    pairs = torch.empty((capacity, 2), dtype=torch.int32, device="cuda")
    cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs, flags=flags)
    dist = sq.edit_distance(pairs, cnt, P["max_d"])
    torch.cuda.synchronize()
    out = (_u32(sig), _u32(pairs)[:cnt].copy(), _u16(dist)[:cnt].copy(), sq.last_raw_pairs())
    sq.close()
    return out


@pytest.mark.parametrize("cfg,n,cap_override", [
    ("config2", 100_000, None),      # full config 2
    ("config2", 30_011, 7),          # cap binds
    ("config3", 60_007, None),
    ("config4", 50_003, None),
    ("config4", 50_003, 5),
])
def test_path_against_oracle(cfg, n, cap_override):
    P = dict(dg.PARAMS[cfg])
    if cap_override:
        P["cap"] = cap_override
    rep = dg.GENERATORS[cfg](n, seed=1)
    want_sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], SEED)
    want_pairs, want_raw, mism = oracle.lsh_sorted(want_sig, P["bands"], P["rows"], P["cap"])
    assert mism == 0
    sig, pairs, dist, raw = _run_path(rep, P, want_pairs.shape[0] + 1000)
    assert np.array_equal(sig, want_sig)
    assert pairs.shape == want_pairs.shape
    assert np.array_equal(pairs, want_pairs)          # same set AND ascending (i, j) order
    assert raw == want_raw
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, want_pairs, P["max_d"])
    assert np.array_equal(dist, want_d)


@pytest.mark.parametrize("kb", [1, 2, 3, 8])
def test_bucket_sort_prefix_bytes_do_not_change_buckets(kb):
    """The bucket sort orders by the top `kb` key bytes and repairs prefix runs that hold several
    full keys; with 1-2 bytes nearly every run is mixed, so the repair does the real work."""
    P = dict(dg.PARAMS["config2"])
    rep = dg.config2(40_009, seed=8)
    want_sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], SEED)
    want_pairs, want_raw, _ = oracle.lsh_sorted(want_sig, P["bands"], P["rows"], P["cap"])
    for flags in (0, 1):
        _, pairs, dist, raw = _run_path(rep, P, want_pairs.shape[0] + 10, flags=flags, sort_key_bytes=kb)
        assert raw == want_raw
        if flags == 0:
            assert np.array_equal(pairs, want_pairs)
        else:
            key = np.sort(pairs[:, 0].astype(np.int64) << 32 | pairs[:, 1])
            assert np.array_equal(key, want_pairs[:, 0].astype(np.int64) << 32 | want_pairs[:, 1])


def test_lsh_unordered_is_the_same_set_and_capacity_protocol():
    P = dict(dg.PARAMS["config2"])
    rep = dg.config2(20_000, seed=5)
    want_sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], SEED)
    want_pairs, _, _ = oracle.lsh_sorted(want_sig, P["bands"], P["rows"], P["cap"])
    from paper_2602_17330_b200 import binding
    _, pairs, _, _ = _run_path(rep, P, want_pairs.shape[0] + 10, flags=binding.LSH_UNORDERED)
    key = np.sort(pairs[:, 0].astype(np.int64) << 32 | pairs[:, 1])
    wkey = want_pairs[:, 0].astype(np.int64) << 32 | want_pairs[:, 1]
    assert np.array_equal(key, wkey)
    # the documented order of SQ_LSH_UNORDERED: i ascending; inside a row, grouped by the first
    # band in which the pair shares a bucket, j ascending inside a group.  The cap (512) does not
    # bind here (largest bucket of this input < 512), so "shares a bucket" == equal band tuples.
    B, r = P["bands"], P["rows"]
    tup = want_sig[:, :B * r].reshape(rep.n, B, r)
    eq = (tup[pairs[:, 0]] == tup[pairs[:, 1]]).all(axis=2)          # [P, B]
    assert eq.any(axis=1).all()
    first = eq.argmax(axis=1).astype(np.int64)
    order = (pairs[:, 0].astype(np.int64) << 40) | (first << 32) | pairs[:, 1]
    assert (np.diff(order) > 0).all()
    # too small an output: SQ_ERR_CAPACITY and the required count comes back
    with pytest.raises(binding.SubQuadError) as ei:
        _run_path(rep, P, want_pairs.shape[0] // 2)
    assert ei.value.code == binding.SQ_ERR_CAPACITY
    assert ei.value.required == want_pairs.shape[0]


def test_determinism_two_runs_identical():
    # "fixed seeds and deterministic kernels"
    P = dict(dg.PARAMS["config2"])
    rep = dg.config2(40_000, seed=9)
    a = _run_path(rep, P, 3_000_000)
    b = _run_path(rep, P, 3_000_000)
    for x, y in zip(a[:3], b[:3]):
        assert np.array_equal(x, y)


# ---------------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------------
def test_edit_distance_textbook_and_edge_cases():
    binding, sq = _ctx()
    enc = lambda s: [ord(c) - ord("a") for c in s]      # 26 letters < 32-symbol alphabet
    words = ["kitten", "sitting", "", "a", "saturday", "sunday", "flaw", "lawn", "abc", "abc",
             "intention", "execution", "a" * 31, "b" * 31, "ab" * 15, "ba" * 15]
    rep = dg.from_list([enc(w) for w in words])
    ws = sq.workspace_bytes(binding.OP_ALL_PAIRS, rep.n, int(rep.offsets[-1]), 31, 0, 1, 0, 1000)
    sq.set_workspace(ws)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(),
            alphabet=26, max_len=31)
    n = rep.n
    ii, jj = np.triu_indices(n, 1)
    pl = np.stack([ii, jj], 1).astype(np.uint32)
    pl = np.concatenate([pl, np.stack([np.arange(n), np.arange(n)], 1).astype(np.uint32)])  # i == j
    want = oracle.edit_distance_pairs(rep.seqs, rep.offsets, pl, -1)
    assert want[0] == 3                                   # kitten / sitting
    for md in (-1, 0, 2, 5):
        d = sq.edit_distance(torch.from_numpy(pl.view(np.int32)).cuda(), pl.shape[0], md)
        w = want if md < 0 else np.minimum(want, md + 1)
        assert np.array_equal(_u16(d)[:pl.shape[0]], w)
    full = torch.empty(n * (n - 1) // 2, dtype=torch.int16, device="cuda")
    sq.all_pairs(-1, None, full)
    assert np.array_equal(_u16(full), oracle.all_pairs_full(rep.seqs, rep.offsets))
    sq.close()


# ---------------------------------------------------------------------------------------------
# single-word DP, one-pattern chunks: 32 consecutive pairs that share i take the branch-free chain
# in which a lane whose text has ended keeps shifting its state through all-ones table words
# (sq_edit.cu).  Rows of >= 32 partners with every mix of text lengths: equal lengths, spreads that
# still fit m + Lmax - Lmin <= 32, spreads that do not (general path), empty patterns and texts,
# thresholds from "everything filtered" to none, both slot strides.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("max_len,alphabet", [(31, 20), (15, 20), (25, 4), (31, 2)])
def test_edit_distance_one_pattern_chunks(max_len, alphabet):
    binding, sq = _ctx()
    rng = np.random.default_rng(1234 + max_len + alphabet)
    seqs = []
    # group g: sequences whose lengths are drawn from a narrow or a wide window
    windows = [(0, 0), (0, 3), (1, 1), (max_len, max_len), (max_len - 2, max_len), (0, max_len),
               (5, 9), (8, min(25, max_len)), (max_len // 2, max_len), (3, 3)]
    group = []
    for g, (lo, hi) in enumerate(windows):
        for _ in range(70):
            L = int(rng.integers(lo, hi + 1))
            base = rng.integers(0, alphabet, size=L)
            seqs.append(base.tolist())
            group.append(g)
    rep = dg.from_list(seqs)
    n = rep.n
    group = np.array(group)
    # rows: the first 3 sequences of every group against all later members of the same group (67-69
    # partners: two full one-pattern chunks and a ragged tail shared with the next row), and against a
    # mixed window of other groups
    pl = []
    for g in range(len(windows)):
        idx = np.flatnonzero(group == g)
        for a in idx[:3]:
            for b in idx[idx > a]:
                pl.append((a, b))
        a = idx[3]
        for b in rng.permutation(n)[:96]:
            pl.append((a, int(b)))
    pl = np.array(pl, dtype=np.uint32)
    ws = sq.workspace_bytes(binding.OP_ALL_PAIRS, n, int(rep.offsets[-1]), max_len, 0, 1, 0, 1000)
    sq.set_workspace(ws)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(),
            alphabet=alphabet, max_len=max_len)
    want = oracle.edit_distance_pairs(rep.seqs, rep.offsets, pl, -1)
    pt = torch.from_numpy(pl.view(np.int32)).cuda()
    for md in (-1, 0, 1, 3, 7, 40):
        d = sq.edit_distance(pt, pl.shape[0], md)
        w = want if md < 0 else np.minimum(want, md + 1)
        assert np.array_equal(_u16(d)[:pl.shape[0]], w), md
    sq.close()


def test_empty_inputs_and_short_sequences():
    binding, sq = _ctx()
    # n = 0
    rep0 = dg.from_list([])
    sq.set_workspace(1 << 20)
    sq.pack(torch.zeros(1, dtype=torch.uint8, device="cuda"),
            torch.zeros(1, dtype=torch.int64, device="cuda"), alphabet=20, max_len=0)
    assert sq.minhash(3, 32, SEED).shape[0] == 0
    pairs = torch.empty((4, 2), dtype=torch.int32, device="cuda")
    assert sq.lsh_candidates(torch.empty((0, 32), dtype=torch.int32, device="cuda"), 8, 4, 10, pairs) == 0
    assert rep0.n == 0
    # sequences shorter than k get the sentinel and take no part in LSH
    seqs = [[1, 2]] * 5 + [[], [3]] + [[1, 2, 3, 4, 5]] * 3 + [[7, 8, 9, 10, 11, 12]]
    rep = dg.from_list(seqs)
    _pack(sq, binding, rep, bands=4, cap=100, pair_capacity=100, H=32)
    sig = sq.minhash(3, 32, SEED)
    want = oracle.minhash(rep.seqs, rep.offsets, 3, 32, SEED)
    assert np.array_equal(_u32(sig), want)
    assert (want[:7] == 0xFFFFFFFF).all()
    pairs = torch.empty((100, 2), dtype=torch.int32, device="cuda")
    cnt = sq.lsh_candidates(sig, 8, 4, 100, pairs)
    wp, _, _ = oracle.lsh_sorted(want, 8, 4, 100)
    assert cnt == wp.shape[0] == 3
    assert np.array_equal(_u32(pairs)[:cnt], wp)
    sq.close()


def test_closed_form_identical_sequences_and_caps():
    binding, sq = _ctx()
    s = [3, 7, 1, 19, 4, 4, 9, 12]
    rep = dg.from_list([s] * 700)
    _pack(sq, binding, rep, bands=16, cap=1024, pair_capacity=300_000, H=64)
    sig = sq.minhash(3, 64, SEED)
    pairs = torch.empty((300_000, 2), dtype=torch.int32, device="cuda")
    for cap in (1024, 700, 512, 33, 2, 1):
        m = min(700, cap)
        cnt = sq.lsh_candidates(sig, 16, 4, cap, pairs)
        assert cnt == m * (m - 1) // 2
        if cnt:
            got = _u32(pairs)[:cnt]
            assert got.max() == m - 1                     # the cap SMALLEST indices are kept
            ii, jj = np.triu_indices(m, 1)
            assert np.array_equal(got[:, 0], ii) and np.array_equal(got[:, 1], jj)
    sq.close()


def test_error_codes():
    binding, sq = _ctx()
    sq.set_workspace(1 << 22)
    seqs = torch.tensor([1, 2, 25, 3], dtype=torch.uint8, device="cuda")     # 25 >= alphabet 20
    offs = torch.tensor([0, 2, 4], dtype=torch.int64, device="cuda")
    with pytest.raises(binding.SubQuadError) as ei:
        sq.pack(seqs, offs, alphabet=20, max_len=8)
    assert ei.value.code == binding.SQ_ERR_BAD_RESIDUE
    with pytest.raises(binding.SubQuadError) as ei:              # nothing packed after a failure
        sq.minhash(3, 32, SEED)
    assert ei.value.code == binding.SQ_ERR_NOT_PACKED
    with pytest.raises(binding.SubQuadError) as ei:              # longer than the declared bound
        sq.pack(torch.zeros(40, dtype=torch.uint8, device="cuda"),
                torch.tensor([0, 40], dtype=torch.int64, device="cuda"), alphabet=20, max_len=8)
    assert ei.value.code == binding.SQ_ERR_UNSUPPORTED
    for bad_offs in ([0, 3, 2], [-1, 2, 4], [0, 9, 4]):          # decreasing, negative, beyond offsets[n]
        with pytest.raises(binding.SubQuadError) as ei:
            sq.pack(seqs, torch.tensor(bad_offs, dtype=torch.int64, device="cuda"), alphabet=20, max_len=8)
        assert ei.value.code == binding.SQ_ERR_INVALID_ARG
    with pytest.raises(binding.SubQuadError) as ei:
        sq.pack(seqs, offs, alphabet=20, max_len=1000)
    assert ei.value.code == binding.SQ_ERR_UNSUPPORTED
    sq.pack(torch.tensor([1, 2, 5, 3], dtype=torch.uint8, device="cuda"), offs, alphabet=20, max_len=8)
    with pytest.raises(binding.SubQuadError) as ei:
        sq.minhash(7, 32, SEED)                                  # 5k > 32
    assert ei.value.code == binding.SQ_ERR_INVALID_ARG
    buf = torch.empty(2 * 32 + 4, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.SubQuadError) as ei:              # signature rows are written by
        sq.minhash(2, 32, SEED, sig_out=buf[4:].view(2, 32))     # 32-byte stores: 16-byte offset
    assert ei.value.code == binding.SQ_ERR_INVALID_ARG
    sig = sq.minhash(2, 32, SEED)
    pairs = torch.empty((8, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.SubQuadError) as ei:
        sq.lsh_candidates(sig, 16, 4, 10, pairs)                 # bands*rows > H
    assert ei.value.code == binding.SQ_ERR_INVALID_ARG
    small = binding.SubQuad(0)
    small.set_workspace(8192)
    with pytest.raises(binding.SubQuadError) as ei:
        small.pack(torch.zeros(10_000, dtype=torch.uint8, device="cuda"),
                   torch.arange(0, 10_001, 10, dtype=torch.int64, device="cuda"), 20, 10)
    assert ei.value.code == binding.SQ_ERR_WORKSPACE
    small.close()
    sq.close()


def test_all_pairs_bag_filter_and_its_fallback():
    """Thresholded all-pairs: (a) the bag-distance filter never drops a hit; (b) when more pairs
    survive the filter than its scratch holds (anagrams: equal histograms, large distances), the
    fused kernel takes over and the result is the same."""
    binding, sq = _ctx()
    rng = np.random.default_rng(11)
    base = rng.integers(0, 20, 40).astype(np.uint8)
    seqs = [rng.permutation(base) for _ in range(700)]            # 244,650 pairs, all with bag distance 0
    seqs += [base.copy(), np.concatenate([base[:20], base[21:]]), np.concatenate([base, [3]])]   # a few true hits
    rep = dg.from_list(seqs)
    want_p, want_d = oracle.all_pairs_threshold(rep.seqs, rep.offsets, 3, use_cutoff=True)
    assert 0 < want_p.shape[0] < 1000
    for cap in (1000, 100_000):                                   # 69,536 < survivors < 465,536
        ws = sq.workspace_bytes(binding.OP_ALL_PAIRS, rep.n, int(rep.offsets[-1]), 41, 0, 1, 0, cap)
        sq.set_workspace(ws)
        sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, 41)
        pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
        dist = torch.empty(cap, dtype=torch.int16, device="cuda")
        cnt = sq.all_pairs(3, pairs, dist)
        assert cnt == want_p.shape[0]
        assert np.array_equal(_u32(pairs)[:cnt], want_p)
        assert np.array_equal(_u16(dist)[:cnt], want_d)
    sq.close()


# ---------------------------------------------------------------------------------------------
# next-1: weighted edit distance (substitution table + indel cost)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("table,indel", [("class", 1), ("class3", 2), ("random", 3), ("unit", 1)])
def test_weighted_edit_distance_short_sequences(table, indel):
    binding, sq = _ctx()
    rep = dg.config2(20_011, seed=6)                      # lengths 5..28, one 32-byte slot
    _pack(sq, binding, rep, op=binding.OP_EDIT_DISTANCE)
    rng = np.random.default_rng(7)
    # pairs grouped by i (like LSH output) plus fully random ones (many runs per warp)
    ii = np.repeat(rng.integers(0, rep.n, 3000), rng.integers(1, 90, 3000))
    grouped = np.stack([ii, rng.integers(0, rep.n, ii.size)], 1)
    pl = np.concatenate([grouped, rng.integers(0, rep.n, (40_003, 2))]).astype(np.uint32)
    cost = {"class": dg.class_substitution_costs(), "class3": dg.class_substitution_costs(2, 3),
            "random": dg.random_substitution_costs(20, 1, 9, 5),
            "unit": (1 - np.eye(20)).astype(np.uint8)}[table]
    sub = torch.from_numpy(cost).cuda()
    pt = torch.from_numpy(pl.view(np.int32)).cuda()
    for md in (-1, 3, 10):
        want = oracle.edit_distance_weighted_pairs(rep.seqs, rep.offsets, pl, cost, indel, md)
        d = sq.edit_distance_weighted(pt, pl.shape[0], sub, indel, md)
        assert np.array_equal(_u16(d)[:pl.shape[0]], want)
    if table == "unit":                                   # reduces to the bit-parallel kernel
        d1 = sq.edit_distance(pt, pl.shape[0], -1)
        d2 = sq.edit_distance_weighted(pt, pl.shape[0], sub, 1, -1)
        assert torch.equal(d1[:pl.shape[0]], d2[:pl.shape[0]])
    sq.close()


def test_weighted_edit_distance_long_and_tiny_sequences():
    binding, sq = _ctx()
    rng = np.random.default_rng(8)
    rep = dg.config5(1_000, seed=3)                       # lengths 100..140: the general kernel
    _pack(sq, binding, rep, op=binding.OP_EDIT_DISTANCE)
    pl = rng.integers(0, rep.n, (6_001, 2)).astype(np.uint32)
    cost = dg.class_substitution_costs()
    want = oracle.edit_distance_weighted_pairs(rep.seqs, rep.offsets, pl, cost, 1, 40)
    d = sq.edit_distance_weighted(torch.from_numpy(pl.view(np.int32)).cuda(), pl.shape[0],
                                  torch.from_numpy(cost).cuda(), 1, 40)
    assert np.array_equal(_u16(d)[:pl.shape[0]], want)
    # tiny and empty sequences, 16-byte slots
    seqs = [[], [3], [3, 4], [4, 3], [1, 2, 3, 4, 5, 6, 7], [7, 6, 5, 4, 3, 2, 1], [0] * 15, [19] * 15]
    rep2 = dg.from_list(seqs)
    _pack(sq, binding, rep2, op=binding.OP_EDIT_DISTANCE, max_len=15)
    n = rep2.n
    pl2 = np.array([(i, j) for i in range(n) for j in range(n)], np.uint32)
    cost2 = dg.random_substitution_costs(20, 1, 200, 9)
    for indel in (1, 7, 255):
        want = oracle.edit_distance_weighted_pairs(rep2.seqs, rep2.offsets, pl2, cost2, indel, -1)
        d = sq.edit_distance_weighted(torch.from_numpy(pl2.view(np.int32)).cuda(), pl2.shape[0],
                                      torch.from_numpy(cost2).cuda(), indel, -1)
        assert np.array_equal(_u16(d)[:pl2.shape[0]], want)
    sq.close()


def test_weighted_table_diagonal_is_never_used():
    """PAPER.md L754 Eq. 46: the cost is multiplied by I(a != b) -- a table with a NON-ZERO diagonal
    gives the distances of the same table with a zero diagonal (reading 22b); short
    (profile kernel) and long (general kernel) sequences."""
    binding, sq = _ctx()
    rng = np.random.default_rng(17)
    cost = rng.integers(1, 9, (20, 20)).astype(np.uint8)          # diagonal 1..8
    for rep in (dg.config2(6_007, seed=9), dg.config5(400, seed=4)):
        _pack(sq, binding, rep, op=binding.OP_EDIT_DISTANCE)
        ii = np.repeat(rng.integers(0, rep.n, 500), rng.integers(1, 40, 500))
        pl = np.stack([ii, rng.integers(0, rep.n, ii.size)], 1).astype(np.uint32)
        pl[::7, 1] = pl[::7, 0]                                   # i == j: all matches, distance 0
        pt = torch.from_numpy(pl.view(np.int32)).cuda()
        for indel, md in ((1, -1), (2, 6)):
            want = oracle.edit_distance_weighted_pairs(rep.seqs, rep.offsets, pl, cost, indel, md)
            d = sq.edit_distance_weighted(pt, pl.shape[0], torch.from_numpy(cost).cuda(), indel, md)
            assert np.array_equal(_u16(d)[:pl.shape[0]], want)
            assert (want[::7] == 0).all()
    sq.close()


# ---------------------------------------------------------------------------------------------
# the family-ordered schedule of the DP stages, forced on small inputs (SQ_OPT_SCHED_MIN_BYTES = 0)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("by_label", [1, 0])
@pytest.mark.parametrize("cfg,n,flags", [("config2", 30_011, 0), ("config2", 30_011, 1), ("config4", 60_013, 0),
                                         ("config3", 40_009, 0)])
def test_schedule_forced_edit_weighted_graph(cfg, n, flags, by_label):
    """With the schedule forced, sq_edit_distance / sq_edit_distance_weighted / sq_affinity_graph walk
    the pairs in the schedule's order -- rows by family label (SQ_OPT_SCHED_BY_LABEL = 1, the default)
    or in band 0's bucket order (0); chunk schedule, rows of every size, empty rows, chunks that cross
    rows: every distance and the whole graph still equal the oracle, bit for bit."""
    binding, sq = _ctx()
    P = dict(dg.PARAMS[cfg])
    rep = dg.GENERATORS[cfg](n, seed=31)
    cap = (160 if cfg == "config4" else 90) * n
    max_len = int(rep.lengths.max())
    ws = max(sq.workspace_bytes(binding.OP_LSH, rep.n, int(rep.offsets[-1]), max_len, P["H"], P["bands"], P["cap"], cap),
             sq.workspace_bytes(binding.OP_GRAPH, rep.n, 0, max_len, 0, 0, 0, cap)) + 4 * cap + 8 * n
    sq.set_workspace(ws)
    sq.set_option(binding.OPT_SCHED_MIN_BYTES, 0)
    sq.set_option(binding.OPT_SCHED_BY_LABEL, by_label)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    sig = sq.minhash(P["k"], P["H"], SEED)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
    cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs, flags=flags)
    hp = _u32(pairs)[:cnt].copy()
    dist = torch.full((cnt,), 0x5A5A, dtype=torch.int16, device="cuda")      # an unwritten slot would show
    sq.edit_distance(pairs, cnt, P["max_d"], dist)
    want = oracle.edit_distance_pairs(rep.seqs, rep.offsets, hp, P["max_d"])
    assert np.array_equal(_u16(dist), want)
    cost = dg.class_substitution_costs()
    wd = torch.full((cnt,), 0x5A5A, dtype=torch.int16, device="cuda")
    sq.edit_distance_weighted(pairs, cnt, torch.from_numpy(cost).cuda(), 1, 5, wd)
    assert np.array_equal(_u16(wd), oracle.edit_distance_weighted_pairs(rep.seqs, rep.offsets, hp, cost, 1, 5))
    if flags == 0:
        mm = int(np.ceil(0.7 * P["H"]))
        row_ptr = torch.empty(rep.n + 1, dtype=torch.int64, device="cuda")
        col = torch.empty(cnt, dtype=torch.int32, device="cuda")
        wgt = torch.empty(cnt, dtype=torch.float32, device="cuda")
        e = sq.affinity_graph(pairs, dist, cnt, P["max_d"], sig, mm, row_ptr, col, wgt)
        rp, wc, ww = oracle.affinity_graph(hp, want, P["max_d"], _u32(sig), mm, rep.lengths, rep.n)
        assert e == rp[-1] and np.array_equal(row_ptr.cpu().numpy(), rp)
        assert np.array_equal(_u32(col)[:e], wc)
        assert np.allclose(wgt.cpu().numpy()[:e], ww, rtol=0, atol=1.5e-7)
    sq.close()


def test_schedule_hint_survives_an_in_place_rewrite_of_the_pair_buffer():
    """The schedule hint is keyed on the pair buffer's address and count.  It only permutes the ORDER
    in which pairs are visited -- every pair is read from the caller's buffer -- so after the caller
    overwrites that very buffer (same pointer, same count) with arbitrary pairs, the distances are
    those of the NEW pairs."""
    binding, sq = _ctx()
    P = dict(dg.PARAMS["config2"])
    rep = dg.config2(40_009, seed=33)
    cap = 60 * rep.n
    _pack(sq, binding, rep, bands=P["bands"], cap=P["cap"], pair_capacity=cap, H=P["H"])
    sq.set_option(binding.OPT_SCHED_MIN_BYTES, 0)
    sig = sq.minhash(P["k"], P["H"], SEED)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
    cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs)
    rng = np.random.default_rng(34)
    newp = rng.integers(0, rep.n, (cnt, 2)).astype(np.uint32)
    newp[::11, 0] = rep.n + 5                                      # out-of-range index -> 0xFFFF
    pairs[:cnt].copy_(torch.from_numpy(newp.view(np.int32)).cuda())
    dist = torch.full((cnt,), 0x5A5A, dtype=torch.int16, device="cuda")
    sq.edit_distance(pairs, cnt, P["max_d"], dist)
    ok = newp[:, 0] < rep.n
    want = np.full(cnt, 0xFFFF, np.uint16)
    want[ok] = oracle.edit_distance_pairs(rep.seqs, rep.offsets, newp[ok], P["max_d"])
    assert np.array_equal(_u16(dist), want)
    sq.close()


# ---------------------------------------------------------------------------------------------
# next-2: verified candidates -> sparse similarity graph
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("flags", [0, 1])
def test_affinity_graph_against_oracle(flags):
    binding, sq = _ctx()
    P = dict(dg.PARAMS["config2"])
    rep = dg.config2(30_011, seed=12)
    cap = 1_200_000
    max_len = int(rep.lengths.max())
    ws = max(sq.workspace_bytes(binding.OP_LSH, rep.n, int(rep.offsets[-1]), max_len, P["H"], P["bands"],
                                P["cap"], cap),
             sq.workspace_bytes(binding.OP_GRAPH, rep.n, 0, max_len, 0, 0, 0, cap))
    sq.set_workspace(ws)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    sig = sq.minhash(P["k"], P["H"], SEED)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
    cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs, flags=flags)
    dist = sq.edit_distance(pairs, cnt, P["max_d"])
    hp, hd, hs = _u32(pairs)[:cnt].copy(), _u16(dist)[:cnt].copy(), _u32(sig)
    row_ptr = torch.empty(rep.n + 1, dtype=torch.int64, device="cuda")
    col = torch.empty(cnt, dtype=torch.int32, device="cuda")
    wgt = torch.empty(cnt, dtype=torch.float32, device="cuda")
    for mm in (0, 20, 45, 64):
        e = sq.affinity_graph(pairs, dist, cnt, P["max_d"], sig, mm, row_ptr, col, wgt)
        rp, wc, ww = oracle.affinity_graph(hp, hd, P["max_d"], hs, mm, rep.lengths, rep.n)
        assert e == rp[-1]
        assert np.array_equal(row_ptr.cpu().numpy(), rp)
        assert np.array_equal(_u32(col)[:e], wc)
        # fp32 (1 - d/L, correctly rounded ops) against the fp64 oracle: half an ulp per op
        assert np.allclose(wgt.cpu().numpy()[:e], ww, rtol=0, atol=1.5e-7)
    with pytest.raises(binding.SubQuadError) as ei:           # capacity protocol
        sq.affinity_graph(pairs, dist, cnt, P["max_d"], sig, 0, row_ptr, col[:10], wgt[:10])
    assert ei.value.code == binding.SQ_ERR_CAPACITY and ei.value.required == (hd <= P["max_d"]).sum()
    sq.close()


@pytest.mark.parametrize("lo,hi", [(33, 64), (65, 128), (129, 160), (200, 240)])
def test_multiword_dp_every_word_count(lo, hi):
    """2, 4, 5 and 8 32-bit words per DP column (up to SQ_MAX_LEN = 240 residues): pair lists,
    the fused tile kernel (unthresholded) and the filtered thresholded path against the oracle."""
    binding, sq = _ctx()
    rng = np.random.default_rng(hi)
    seeds = [rng.integers(0, 20, rng.integers(lo, hi + 1)).astype(np.uint8) for _ in range(12)]
    seqs = []
    for s in seeds:
        for _ in range(25):
            t = s.copy()
            for _e in range(rng.integers(0, 9)):                  # substitutions keep the length in range
                t[rng.integers(0, t.size)] = rng.integers(0, 20)
            seqs.append(t)
    seqs.append(np.zeros(0, np.uint8))                            # an empty sequence among long ones
    rep = dg.from_list(seqs)
    n = rep.n
    npairs = n * (n - 1) // 2
    ws = sq.workspace_bytes(binding.OP_ALL_PAIRS, n, int(rep.offsets[-1]), hi, 0, 1, 0, npairs)
    sq.set_workspace(ws)
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, hi)
    full = torch.empty(npairs, dtype=torch.int16, device="cuda")
    assert sq.all_pairs(-1, None, full) == npairs
    want = oracle.all_pairs_full(rep.seqs, rep.offsets)
    assert np.array_equal(_u16(full), want)
    ii, jj = np.triu_indices(n, 1)
    for md in (0, 8, 30):
        sel = np.nonzero(want <= md)[0]
        pairs = torch.empty((sel.size + 8, 2), dtype=torch.int32, device="cuda")
        d2 = torch.empty(sel.size + 8, dtype=torch.int16, device="cuda")
        cnt = sq.all_pairs(md, pairs, d2)
        assert cnt == sel.size
        got = _u32(pairs)[:cnt]
        assert np.array_equal(got[:, 0], ii[sel]) and np.array_equal(got[:, 1], jj[sel])
        assert np.array_equal(_u16(d2)[:cnt], want[sel])
    take = rng.choice(npairs, 20_000, replace=False)
    pl = np.stack([jj[take], ii[take]], 1).astype(np.uint32)      # (j, i): i > j is allowed in a pair list
    for md in (-1, 12):
        d = sq.edit_distance(torch.from_numpy(pl.view(np.int32)).cuda(), pl.shape[0], md)
        w = want[take] if md < 0 else np.minimum(want[take], md + 1)
        assert np.array_equal(_u16(d)[:pl.shape[0]], w)
    sq.close()


# ---------------------------------------------------------------------------------------------
# the whole path from host buffers (the e2e entry points)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n", [("config2", 30_011), ("config4", 50_003)])
def test_pipeline_host_pairs_and_csr(cfg, n):
    binding, sq = _ctx()
    P = dict(dg.PARAMS[cfg])
    rep = dg.GENERATORS[cfg](n, seed=6)
    want_sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], SEED)
    want_pairs, _, _ = oracle.lsh_sorted(want_sig, P["bands"], P["rows"], P["cap"])
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, want_pairs, P["max_d"])
    cap = want_pairs.shape[0] + 100
    max_len = int(rep.lengths.max())
    sq.set_workspace(sq.workspace_bytes(binding.OP_PIPELINE_HOST, rep.n, int(rep.offsets[-1]), max_len,
                                        P["H"], P["bands"], P["cap"], cap))
    seqs_h = torch.from_numpy(rep.seqs).pin_memory()
    offs_h = torch.from_numpy(rep.offsets).pin_memory()
    pairs_h = torch.empty((cap, 2), dtype=torch.int32).pin_memory()
    dist_h = torch.empty(cap, dtype=torch.int16).pin_memory()
    cnt = sq.pipeline_host(seqs_h, offs_h, 20, max_len, P["k"], P["H"], SEED, P["bands"], P["rows"],
                           P["cap"], P["max_d"], pairs_h, dist_h)
    assert cnt == want_pairs.shape[0]
    assert np.array_equal(pairs_h.numpy().view(np.uint32)[:cnt], want_pairs)
    assert np.array_equal(dist_h.numpy().view(np.uint16)[:cnt], want_d)
    # CSR form: same content, 5 bytes per candidate
    row_ptr = torch.full((rep.n + 1,), -1, dtype=torch.int64).pin_memory()
    col = torch.empty(cap, dtype=torch.int32).pin_memory()
    d8 = torch.empty(cap, dtype=torch.uint8).pin_memory()
    cnt2 = sq.pipeline_host_csr(seqs_h, offs_h, 20, max_len, P["k"], P["H"], SEED, P["bands"], P["rows"],
                                P["cap"], P["max_d"], row_ptr, col, d8)
    assert cnt2 == cnt
    want_rp = np.searchsorted(want_pairs[:, 0], np.arange(rep.n + 1), side="left")
    assert np.array_equal(row_ptr.numpy(), want_rp)
    assert np.array_equal(col.numpy().view(np.uint32)[:cnt], want_pairs[:, 1])
    assert np.array_equal(d8.numpy()[:cnt], want_d.astype(np.uint8))
    sq.close()


def test_pipeline_host_csr_no_candidates_and_limits():
    from paper_2602_17330_b200.binding import SubQuadError, SQ_ERR_UNSUPPORTED
    binding, sq = _ctx()
    rep = dg.config1(300, seed=2)                  # iid random sequences: k=5 sketches share no band
    max_len = int(rep.lengths.max())
    sq.set_workspace(sq.workspace_bytes(binding.OP_PIPELINE_HOST, rep.n, int(rep.offsets[-1]), max_len,
                                        64, 16, 8, 1000))
    seqs_h = torch.from_numpy(rep.seqs).pin_memory()
    offs_h = torch.from_numpy(rep.offsets).pin_memory()
    row_ptr = torch.full((rep.n + 1,), -1, dtype=torch.int64).pin_memory()
    col = torch.empty(1000, dtype=torch.int32).pin_memory()
    d8 = torch.empty(1000, dtype=torch.uint8).pin_memory()
    sig = oracle.minhash(rep.seqs, rep.offsets, 5, 64, SEED)
    want_pairs, _, _ = oracle.lsh_sorted(sig, 16, 4, 8)
    cnt = sq.pipeline_host_csr(seqs_h, offs_h, 20, max_len, 5, 64, SEED, 16, 4, 8, 3, row_ptr, col, d8)
    assert cnt == want_pairs.shape[0]
    want_rp = np.searchsorted(want_pairs[:, 0], np.arange(rep.n + 1), side="left")
    assert np.array_equal(row_ptr.numpy(), want_rp)
    with pytest.raises(SubQuadError) as e:
        sq.pipeline_host_csr(seqs_h, offs_h, 20, max_len, 5, 64, SEED, 16, 4, 8, 255, row_ptr, col, d8)
    assert e.value.code == SQ_ERR_UNSUPPORTED
    sq.close()


# ---------------------------------------------------------------------------------------------
# long sequences under a threshold: look-ahead filter + banded multi-word column
# ---------------------------------------------------------------------------------------------
def _edited_families(rng, n_fam, members, L_lo, L_hi, max_edits):
    seqs = []
    for _ in range(n_fam):
        base = rng.integers(0, 20, rng.integers(L_lo, L_hi + 1)).astype(np.uint8)
        for _ in range(members):
            s = list(base)
            for _ in range(rng.integers(0, max_edits + 1)):
                op = rng.integers(0, 3)
                pos = rng.integers(0, len(s) + (op == 1))
                if op == 0 and len(s):
                    s[min(pos, len(s) - 1)] = rng.integers(0, 20)
                elif op == 1:
                    s.insert(pos, rng.integers(0, 20))
                elif len(s) > 1:
                    del s[min(pos, len(s) - 1)]
            seqs.append(np.asarray(s, np.uint8))
    order = rng.permutation(len(seqs))
    return dg.from_list([seqs[q] for q in order])


@pytest.mark.parametrize("L_lo,L_hi,max_edits,max_d", [
    (66, 80, 6, 3), (66, 80, 12, 8), (100, 130, 20, 15), (100, 130, 40, 31), (100, 130, 40, 32),
    (150, 160, 24, 20), (200, 225, 30, 25), (33, 70, 10, 7), (120, 125, 3, 0), (100, 130, 50, 40), (70, 96, 20, 16),
    (70, 96, 20, 17)])
def test_all_pairs_long_thresholded_band(L_lo, L_hi, max_edits, max_d):
    """Distances straddle max_d (edits up to ~1.3 max_d per member), lengths span 2-8 words."""
    rng = np.random.default_rng(L_lo * 1000 + max_d)
    rep = _edited_families(rng, 12, 40, L_lo, L_hi, max_edits)
    want_p, want_d = oracle.all_pairs_threshold(rep.seqs, rep.offsets, max_d)
    assert want_p.shape[0] > 100
    binding, sq = _ctx()
    cap = want_p.shape[0] + 64
    _pack(sq, binding, rep, op=binding.OP_ALL_PAIRS, pair_capacity=cap)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
    dist = torch.empty(cap, dtype=torch.int16, device="cuda")
    cnt = sq.all_pairs(max_d, pairs, dist)
    assert cnt == want_p.shape[0]
    assert np.array_equal(_u32(pairs)[:cnt], want_p)
    assert np.array_equal(_u16(dist)[:cnt], want_d)
    sq.close()


def test_roofline_probes_are_consistent():
    """The denominators bench.py quotes: the column chain alone cannot beat the plain LOP3 stream, and
    two pipes fed with fresh register operands stay below the sum of the pipes' own peaks."""
    binding, sq = _ctx()
    sq.set_workspace(1 << 20)
    lop3 = sq.int_peak(0, 1024)
    imad = sq.int_peak(3, 1024)
    both_fresh = sq.int_peak(8, 1024)
    mix = sq.int_peak(9, 1024)
    chain = sq.dp_chain_peak(20, 500) * 7
    assert lop3 > 1e12 and imad > 1e12
    assert lop3 * 0.9 < both_fresh < (lop3 + imad) * 1.02
    assert lop3 * 0.9 < mix < (lop3 + imad) * 1.02
    assert 0.3 * lop3 < chain < 1.02 * lop3
    with pytest.raises(binding.SubQuadError):
        sq.dp_chain_peak(0, 10)
    with pytest.raises(binding.SubQuadError):
        sq.dp_chain_peak(32, 10)
    sq.close()
