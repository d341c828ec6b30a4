"""Pins for the oracle's LSH candidate generation (spec C3).

Banding is not in the paper (BASELINE.json configs fix bands x rows and the cap), so
pins are: the set definition executed by brute force (Tier A) vs the sort-based
Tier B, key equality == tuple equality, closed-form counts, the cap semantics on
hand-built signatures, and the textbook S-curve 1-(1-J^r)^B.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2602_17330_b200 import datagen as dg

SEED = dg.DEFAULT_SEED64


def _naive_python(sig, bands, rows, cap):
    """Literal restatement with dicts of tuples (no 64-bit key at all)."""
    n = sig.shape[0]
    out = set()
    for b in range(bands):
        buckets = {}
        for i in range(n):
            if (sig[i] == 0xFFFFFFFF).all():
                continue
            buckets.setdefault(tuple(sig[i, b * rows:(b + 1) * rows].tolist()), []).append(i)
        for members in buckets.values():
            kept = members[:cap]
            for u in range(len(kept)):
                for v in range(u + 1, len(kept)):
                    out.add((kept[u], kept[v]))
    return np.array(sorted(out), np.uint32).reshape(-1, 2)


def test_band_key_constants_and_sensitivity():
    # 0x6A09E667F3BCC908 = frac(sqrt 2) * 2^64; 0x9E3779B97F4A7C15 = 2^64 / golden ratio (odd)
    assert math.isqrt(2 << 128) - (1 << 64) == 0x6A09E667F3BCC908
    phi_inv = (math.isqrt(5 << 128) - (1 << 64)) // 2          # (sqrt5 - 1)/2 * 2^64
    assert phi_inv | 1 == 0x9E3779B97F4A7C15
    # empty tuple -> the initial accumulator
    assert oracle.band_key(np.zeros(0, np.uint32)) == 0x6A09E667F3BCC908
    # one value: ((init ^ v) * mult) ^ (that >> 29)
    v = 0x12345678
    acc = ((0x6A09E667F3BCC908 ^ v) * 0x9E3779B97F4A7C15) & ((1 << 64) - 1)
    acc ^= acc >> 29
    assert oracle.band_key([v]) == acc
    # order matters, every position matters
    assert oracle.band_key([1, 2, 3, 4]) != oracle.band_key([2, 1, 3, 4])
    base = oracle.band_key([5, 6, 7, 8])
    for p in range(4):
        t = [5, 6, 7, 8]
        t[p] ^= 1
        flipped = bin(base ^ oracle.band_key(t)).count("1")
        assert 12 <= flipped <= 52


@pytest.mark.parametrize("gen,k,H,bands,rows,cap", [
    ("config2", 3, 64, 16, 4, 512),
    ("config2", 3, 64, 16, 4, 6),        # cap binds
    ("config3", 4, 128, 32, 4, 1024),
    ("config4", 3, 64, 16, 4, 3),
])
def test_bruteforce_equals_sorted(gen, k, H, bands, rows, cap):
    r = dg.GENERATORS[gen](3000, seed=4)
    sig = oracle.minhash(r.seqs, r.offsets, k, H, SEED)
    A, mismA = oracle.lsh_bruteforce(sig, bands, rows, cap)
    B, raw, mismB = oracle.lsh_sorted(sig, bands, rows, cap)
    assert mismA == 0 and mismB == 0            # key equality == tuple equality
    assert A.shape == B.shape and (A == B).all()
    assert raw >= A.shape[0] > 0
    # strictly ascending, i < j
    key = A[:, 0].astype(np.int64) << 32 | A[:, 1]
    assert (np.diff(key) > 0).all() and (A[:, 0] < A[:, 1]).all()


def test_matches_literal_python_on_small_input():
    r = dg.config2(600, seed=8)
    sig = oracle.minhash(r.seqs, r.offsets, 3, 32, SEED)
    for cap in (2, 4, 1000):
        want = _naive_python(sig, 8, 4, cap)
        A, _ = oracle.lsh_bruteforce(sig, 8, 4, cap)
        B, _, _ = oracle.lsh_sorted(sig, 8, 4, cap)
        assert (A == want).all() and (B == want).all()


def test_closed_form_counts_identical_sequences():
    s = [3, 7, 1, 19, 4, 4, 9, 12]
    for n, cap in ((40, 1000), (40, 16), (40, 2), (40, 1), (1, 5)):
        rep = dg.from_list([s] * n)
        sig = oracle.minhash(rep.seqs, rep.offsets, 3, 32, SEED)
        m = min(n, cap)
        for fn in (lambda: oracle.lsh_bruteforce(sig, 8, 4, cap)[0],
                   lambda: oracle.lsh_sorted(sig, 8, 4, cap)[0]):
            P = fn()
            assert P.shape[0] == m * (m - 1) // 2
            if P.size:
                assert P.max() == m - 1            # the `cap` SMALLEST indices are kept


def test_cap_semantics_on_handbuilt_signatures():
    # 2 bands x 1 row.  band 0: {0,1,2,3} share a tuple; band 1: {2,3,4} share a tuple.
    sig = np.array([[10, 100], [10, 101], [10, 200], [10, 200], [11, 200], [12, 102]], np.uint32)
    full = {(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3), (2, 4), (3, 4)}
    P, _ = oracle.lsh_bruteforce(sig, 2, 1, 10)
    assert set(map(tuple, P.tolist())) == full
    # cap 2: band 0 keeps {0,1}; band 1 keeps {2,3}  (not a dropped bucket, reading 8)
    for fn in (oracle.lsh_bruteforce, oracle.lsh_sorted):
        P = fn(sig, 2, 1, 2)[0]
        assert set(map(tuple, P.tolist())) == {(0, 1), (2, 3)}
        P = fn(sig, 2, 1, 3)[0]
        assert set(map(tuple, P.tolist())) == {(0, 1), (0, 2), (1, 2), (2, 3), (2, 4), (3, 4)}
        assert fn(sig, 2, 1, 1)[0].shape[0] == 0
    # keys are compared only within the same band: value 200 in band 0 vs band 1 never collide
    sig2 = np.array([[200, 1], [2, 200]], np.uint32)
    assert oracle.lsh_bruteforce(sig2, 2, 1, 10)[0].shape[0] == 0
    assert oracle.lsh_sorted(sig2, 2, 1, 10)[0].shape[0] == 0


def test_rows_beyond_bands_ignored_and_empty_signatures_excluded():
    r = dg.config2(800, seed=2)
    sig = oracle.minhash(r.seqs, r.offsets, 3, 64, SEED)
    P1, _, _ = oracle.lsh_sorted(sig, 4, 4, 100)
    sig2 = sig.copy()
    sig2[:, 16:] = 7                      # columns >= bands*rows must not matter
    P2, _, _ = oracle.lsh_sorted(sig2, 4, 4, 100)
    assert (P1 == P2).all()
    # sequences shorter than k have the all-ones signature and take no part
    rep = dg.from_list([[1, 2]] * 5 + [[1, 2, 3]] * 3)
    s = oracle.minhash(rep.seqs, rep.offsets, 3, 16, SEED)
    for fn in (oracle.lsh_bruteforce, oracle.lsh_sorted):
        P = fn(s, 4, 4, 100)[0]
        assert set(map(tuple, P.tolist())) == {(5, 6), (5, 7), (6, 7)}


def test_row_oracle_matches_full_set():
    r = dg.config2(2500, seed=6)
    sig = oracle.minhash(r.seqs, r.offsets, 3, 64, SEED)
    for cap in (5, 512):
        P, _, _ = oracle.lsh_sorted(sig, 16, 4, cap)
        for i in range(0, r.n, 131):
            want = np.sort(np.concatenate([P[P[:, 0] == i, 1], P[P[:, 1] == i, 0]]))
            got = oracle.lsh_row(sig, 16, 4, cap, i)
            assert (got == want).all()


def test_s_curve():
    """Textbook banding: P(candidate | J) = 1 - (1 - J^r)^B, checked per exact-J bin."""
    k, H, B, rws = 3, 64, 16, 4
    r = dg.config2(8000, seed=13)
    sig = oracle.minhash(r.seqs, r.offsets, k, H, SEED)
    P, _, _ = oracle.lsh_sorted(sig, B, rws, 10 ** 9)
    cand = set((P[:, 0].astype(np.int64) << 32 | P[:, 1]).tolist())
    rng = np.random.default_rng(1)
    order = np.argsort(r.family, kind="stable")
    bins = {}
    for _ in range(30000):
        q = rng.integers(0, r.n - 3)
        i, j = order[q], order[q + rng.integers(1, 4)]
        if r.family[i] != r.family[j] or i == j:
            continue
        i, j = (i, j) if i < j else (j, i)
        num, den = oracle.kmer_jaccard(r.seq(i), r.seq(j), k)
        J = num / den
        hit = ((int(i) << 32) | int(j)) in cand
        b = bins.setdefault(round(J * 10), [0, 0, 0.0])
        b[0] += 1
        b[1] += hit
        b[2] += 1 - (1 - J ** rws) ** B
    tested = 0
    for _, (cnt, hits, psum) in bins.items():
        if cnt < 300:
            continue
        p = psum / cnt
        se = math.sqrt(max(p * (1 - p), 1e-4) / cnt)
        # MinHash rows are exchangeable but not independent across a fixed pair's bands only
        # through J itself; allow 5 s.e. + 0.02 model slack
        assert abs(hits / cnt - p) < 5 * se + 0.02, (cnt, hits / cnt, p)
        tested += 1
    assert tested >= 4
