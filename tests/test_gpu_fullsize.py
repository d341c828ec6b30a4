"""Full-size parity checks, in the launch configuration bench.py times (BASELINE.json configs 3-5).

At these sizes the oracle cannot produce the whole output in seconds, so the CUDA path is
checked (a) on sampled outputs the oracle computes one by one -- whole signatures, whole
candidate rows from the definition (oracle.lsh_row), distances by Wagner-Fischer -- and (b) via
properties that hold at any size: strictly ascending duplicate-free (i, j), i < j, the raw-pair
count, the generator's bound d(i, j) <= e_i + e_j inside a family, determinism of the count.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_17330_b200 import datagen as dg

pytestmark = pytest.mark.gpu
SEED = dg.DEFAULT_SEED64


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def _run_full(cfg, n=None, flags=0):
    from paper_2602_17330_b200 import binding
    P = dg.PARAMS[cfg]
    rep = dg.GENERATORS[cfg](n, seed=0) if n else dg.GENERATORS[cfg](seed=0)
    sq = binding.SubQuad(0)
    max_len = int(rep.lengths.max())
    total_len = int(rep.offsets[-1])
    cap = {"config3": 60, "config4": 200}[cfg] * rep.n
    seqs = torch.from_numpy(rep.seqs).cuda()
    offs = torch.from_numpy(rep.offsets).cuda()
    while True:
        sq.workspace = None
        torch.cuda.empty_cache()
        sq.set_workspace(sq.workspace_bytes(binding.OP_LSH, rep.n, total_len, max_len, P["H"],
                                            P["bands"], P["cap"], cap))
        sq.pack(seqs, offs, 20, max_len)
        sig = sq.minhash(P["k"], P["H"], SEED)
        pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
        try:
            cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs, flags=flags)
            break
        except binding.SubQuadError as ex:
            assert ex.code == binding.SQ_ERR_CAPACITY
            cap = int(ex.required) + 1024
            del pairs
    dist = sq.edit_distance(pairs, cnt, P["max_d"])
    torch.cuda.synchronize()
    raw = sq.last_raw_pairs()
    sq.close()
    return rep, P, sig, pairs, cnt, dist, raw


def _check_sampled(rep, P, sig, pairs, cnt, dist, n_rows, n_sigs, n_dist, rng):
    n = rep.n
    # (b) properties over the WHOLE output, on the device
    pi = pairs[:cnt, 0].long() & 0xFFFFFFFF
    pj = pairs[:cnt, 1].long() & 0xFFFFFFFF
    assert bool((pi < pj).all()) and bool((pj < n).all())
    key = pi * (1 << 32) + pj
    assert bool((key[1:] > key[:-1]).all()), "pairs not strictly ascending in (i, j)"
    d = dist[:cnt].to(torch.int32) & 0xFFFF
    assert int(d.max()) <= P["max_d"] + 1
    fam = torch.from_numpy(rep.family.astype(np.int64)).cuda()
    ne = torch.from_numpy(rep.n_edits.astype(np.int32)).cuda()
    same = fam[pi] == fam[pj]
    bound = torch.clamp(ne[pi] + ne[pj], max=P["max_d"] + 1)
    assert bool((d[same] <= bound[same]).all()), "d(i,j) > e_i + e_j inside a family"
    # (a) sampled signatures: whole rows, bit exact
    ids = np.sort(rng.choice(n, n_sigs, replace=False))
    sub = dg.from_list([rep.seq(int(i)) for i in ids])
    want = oracle.minhash(sub.seqs, sub.offsets, P["k"], P["H"], SEED)
    got = _u32(sig[torch.from_numpy(ids).cuda()])
    assert np.array_equal(got, want)
    # (a) sampled candidate rows from the definition (needs every signature on the host)
    sig_h = _u32(sig)
    row_start = torch.searchsorted(key, torch.arange(n + 1, device="cuda", dtype=torch.int64) << 32)
    counts = (row_start[1:] - row_start[:-1]).cpu().numpy()
    heavy = np.argsort(-counts)[:4]                         # the largest rows, where the cap binds
    rows = np.unique(np.concatenate([rng.choice(n, n_rows, replace=False), heavy]))
    rs = row_start.cpu().numpy()
    for i in rows:
        part = oracle.lsh_row(sig_h, P["bands"], P["rows"], P["cap"], int(i))
        want_j = part[part > i]
        got_j = _u32(pairs[rs[i]:rs[i + 1], 1])
        assert np.array_equal(got_j, want_j), f"candidate row {i} differs"
    # (a) sampled distances by Wagner-Fischer
    take = np.sort(rng.choice(cnt, n_dist, replace=False))
    tk = torch.from_numpy(take).cuda()
    pl = _u32(pairs[tk])
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, pl, P["max_d"])
    assert np.array_equal(dist[tk].cpu().numpy().view(np.uint16), want_d)


def test_config3_full_size_sampled():
    rep, P, sig, pairs, cnt, dist, raw = _run_full("config3")
    assert rep.n == 1_000_000 and cnt > 0 and raw >= cnt
    _check_sampled(rep, P, sig, pairs, cnt, dist, n_rows=40, n_sigs=20_000, n_dist=500_000,
                   rng=np.random.default_rng(3))


def test_config4_full_size_sampled():
    rep, P, sig, pairs, cnt, dist, raw = _run_full("config4")
    assert rep.n == 10_000_000 and cnt > 0 and raw >= cnt
    _check_sampled(rep, P, sig, pairs, cnt, dist, n_rows=24, n_sigs=20_000, n_dist=1_000_000,
                   rng=np.random.default_rng(4))


def _digest128(pairs_u32):
    """order-independent 128-bit digest of a pair set (two 64-bit sums of mixed keys, mod 2^64)"""
    k = (pairs_u32[:, 0].astype(np.uint64) << np.uint64(32)) | pairs_u32[:, 1].astype(np.uint64)
    with np.errstate(over="ignore"):
        a = k * np.uint64(0x9E3779B97F4A7C15)
        a ^= a >> np.uint64(29)
        b = (k ^ np.uint64(0x6A09E667F3BCC908)) * np.uint64(0xD1B54A32D192ED03)
        b ^= b >> np.uint64(31)
        return int(a.sum(dtype=np.uint64)), int(b.sum(dtype=np.uint64))


def test_config3_whole_candidate_set_and_every_distance_against_the_oracle():
    """at config 3 the oracle's sort-based tier (validated against the brute force in
    tests/test_oracle_lsh.py) still fits: count, raw count, a 128-bit order-independent digest of
    the pair set, the pair list element by element, and ALL distances."""
    rep, P, sig, pairs, cnt, dist, raw = _run_full("config3")
    sig_h = _u32(sig)
    want_p, want_raw, mism = oracle.lsh_sorted(sig_h, P["bands"], P["rows"], P["cap"])
    assert mism == 0
    assert cnt == want_p.shape[0] and raw == want_raw
    got_p = _u32(pairs[:cnt])
    assert _digest128(got_p) == _digest128(want_p)
    assert np.array_equal(got_p, want_p)
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, want_p, P["max_d"])
    assert np.array_equal(dist[:cnt].cpu().numpy().view(np.uint16), want_d)


def test_config4_one_million_prefix_whole_set_against_the_oracle():
    """Config 4's generator (power-law families, caps that bind) at the largest n whose raw pair list
    the oracle sorts in about a minute: count, raw count, digest, pair list and all distances."""
    rep, P, sig, pairs, cnt, dist, raw = _run_full("config4", n=1_000_000)
    want_p, want_raw, mism = oracle.lsh_sorted(_u32(sig), P["bands"], P["rows"], P["cap"])
    assert mism == 0
    assert cnt == want_p.shape[0] and raw == want_raw
    got_p = _u32(pairs[:cnt])
    assert _digest128(got_p) == _digest128(want_p)
    assert np.array_equal(got_p, want_p)
    want_d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, want_p, P["max_d"])
    assert np.array_equal(dist[:cnt].cpu().numpy().view(np.uint16), want_d)


def test_config4_full_size_rewritten_pair_buffer():
    """At full size the packed sequences exceed the L2 and sq_edit_distance follows the schedule
    left by sq_lsh_candidates (keyed on the buffer's address and count).  The buffer is overwritten
    in place with random pairs: the distances must be those of the new pairs (sampled oracle)."""
    from paper_2602_17330_b200 import binding
    P = dg.PARAMS["config4"]
    rep = dg.config4(seed=0)
    sq = binding.SubQuad(0)
    max_len, total_len = int(rep.lengths.max()), int(rep.offsets[-1])
    cap = 165 * rep.n
    sq.set_workspace(sq.workspace_bytes(binding.OP_LSH, rep.n, total_len, max_len, P["H"], P["bands"], P["cap"], cap))
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    sig = sq.minhash(P["k"], P["H"], SEED)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device="cuda")
    cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs)
    del sig
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    pairs[:cnt] = torch.randint(0, rep.n, (cnt, 2), device="cuda", dtype=torch.int32, generator=g)
    dist = torch.full((cnt,), 0x5A5A, dtype=torch.int16, device="cuda")
    sq.edit_distance(pairs, cnt, P["max_d"], dist)
    torch.cuda.synchronize()
    assert int((dist.to(torch.int32) & 0xFFFF).max()) <= P["max_d"] + 1       # no slot left unwritten
    rng = np.random.default_rng(6)
    take = np.sort(rng.choice(cnt, 1_000_000, replace=False))
    tk = torch.from_numpy(take).cuda()
    pl = _u32(pairs[tk])
    assert np.array_equal(dist[tk].cpu().numpy().view(np.uint16),
                          oracle.edit_distance_pairs(rep.seqs, rep.offsets, pl, P["max_d"]))
    sq.close()


def test_config4_unordered_has_the_same_count_and_set_digest():
    # SQ_LSH_UNORDERED must give the same SET: compare the count and an order-independent digest
    rep, P, sig, pairs, cnt, dist, raw = _run_full("config4", n=2_000_000)
    rep2, _, _, pairs2, cnt2, dist2, raw2 = _run_full("config4", n=2_000_000, flags=1)
    assert cnt == cnt2 and raw == raw2

    def digest(p, c):
        k = (p[:c, 0].long() & 0xFFFFFFFF) * 1_000_003 + (p[:c, 1].long() & 0xFFFFFFFF) * 998_244_353
        return int(k.sum().item()), int((k ^ (k >> 17)).sum().item())

    assert digest(pairs, cnt) == digest(pairs2, cnt2)
    # distances follow their pairs: the multiset of (pair, distance) is the same
    def digest_d(p, d, c):
        k = (p[:c, 0].long() & 0xFFFFFFFF) * 7 + (p[:c, 1].long() & 0xFFFFFFFF) * 13
        return int((k * ((d[:c].long() & 0xFFFF) + 1)).sum().item())

    assert digest_d(pairs, dist, cnt) == digest_d(pairs2, dist2, cnt2)


# ---------------------------------------------------------------------------------------------
# config 5: long sequences, multi-word bit-parallel DP, thresholded all-pairs tile path
# ---------------------------------------------------------------------------------------------
def _all_pairs(rep, max_d, capacity):
    from paper_2602_17330_b200 import binding
    sq = binding.SubQuad(0)
    max_len = int(rep.lengths.max())
    sq.set_workspace(sq.workspace_bytes(binding.OP_ALL_PAIRS, rep.n, int(rep.offsets[-1]), max_len,
                                        0, 1, 0, capacity))
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    pairs = torch.empty((capacity, 2), dtype=torch.int32, device="cuda")
    dist = torch.empty(capacity, dtype=torch.int16, device="cuda")
    cnt = sq.all_pairs(max_d, pairs, dist)
    out = _u32(pairs)[:cnt].copy(), dist.cpu().numpy().view(np.uint16)[:cnt].copy()
    sq.close()
    return out


def test_config5_reduced_against_oracle():
    rep = dg.config5(2_000, seed=2)                       # 20 families of 100, lengths 100-140
    assert int(rep.lengths.max()) > 128                   # three 64-bit words / five 32-bit words
    want_p, want_d = oracle.all_pairs_threshold(rep.seqs, rep.offsets, 15, use_cutoff=True)
    got_p, got_d = _all_pairs(rep, 15, want_p.shape[0] + 100)
    assert np.array_equal(got_p, want_p)
    assert np.array_equal(got_d, want_d)
    # Tier A (full Wagner-Fischer) on a sample of the hits and of the non-hits
    rng = np.random.default_rng(0)
    hit = got_p[rng.choice(got_p.shape[0], 2000, replace=False)]
    assert np.array_equal(oracle.edit_distance_pairs(rep.seqs, rep.offsets, hit, -1),
                          got_d[np.searchsorted(got_p[:, 0].astype(np.int64) << 32 | got_p[:, 1],
                                                hit[:, 0].astype(np.int64) << 32 | hit[:, 1])])


def test_config5_full_size_sampled():
    rep = dg.config5()
    n = rep.n
    assert n == 50_000
    got_p, got_d = _all_pairs(rep, 15, 8_000_000)
    assert got_p.shape[0] > 0
    key = got_p[:, 0].astype(np.int64) << 32 | got_p[:, 1]
    assert (np.diff(key) > 0).all() and (got_p[:, 0] < got_p[:, 1]).all() and got_d.max() <= 15
    # every hit re-computed by the oracle (Wagner-Fischer, no cut-off) on a sample
    rng = np.random.default_rng(5)
    take = np.sort(rng.choice(got_p.shape[0], 20_000, replace=False))
    assert np.array_equal(oracle.edit_distance_pairs(rep.seqs, rep.offsets, got_p[take], -1),
                          got_d[take])
    # whole rows: row i against every j > i by the oracle (full Wagner-Fischer), for sampled i
    starts = np.searchsorted(key, np.arange(n + 1, dtype=np.int64) << 32)
    for i in rng.choice(n - 1, 12, replace=False):
        js = np.arange(i + 1, n, dtype=np.uint32)
        pl = np.stack([np.full(js.shape, i, np.uint32), js], 1)
        d = oracle.edit_distance_pairs(rep.seqs, rep.offsets, pl, 15)
        sel = d <= 15
        assert np.array_equal(got_p[starts[i]:starts[i + 1], 1], js[sel]), f"row {i}"
        assert np.array_equal(got_d[starts[i]:starts[i + 1]], d[sel])
