"""Pins for the oracle's cross-repertoire join and Eq. 12 batch size.

join_threshold is pinned by what the mathematics fixes: closed-form distances on constructed
sequences, the planted-copy structure, symmetry under swapping the two sets, and the reduction of
the self-join's upper triangle to the independent C routine orc_all_pairs_threshold.
batch_size is pinned by hand-worked values of PAPER.md Eq. (12).
"""
import numpy as np
import pytest

import oracle
from paper_2602_17330_b200 import datagen


def _pack(lst):
    off = np.zeros(len(lst) + 1, np.int64)
    np.cumsum([len(s) for s in lst], out=off[1:])
    seqs = np.concatenate([np.asarray(s, np.uint8) for s in lst]) if off[-1] else np.zeros(0, np.uint8)
    return seqs, off


def test_batch_size_eq12_worked_values():
    # PAPER.md L141 Eq. (12), worked by hand:
    # M = 1e9, c = 4, l_max = 25: sqrt(1e9 / 100) = sqrt(1e7) = 3162.27.. -> 3162
    assert oracle.batch_size(10**7, 10**9, 4, 25) == 3162
    # the floor of 32: M = 1e5, c = 8, l_max = 130 -> sqrt(96.15) = 9.8 -> max(32, 9) = 32
    assert oracle.batch_size(10**7, 10**5, 8, 130) == 32
    # |S| caps it: 20 sequences only
    assert oracle.batch_size(20, 10**9, 4, 25) == 20
    # an exact square: M = 64 * 100 * 100, c * l_max = 64 -> exactly 100; one byte less -> 99
    assert oracle.batch_size(10**6, 64 * 10000, 2, 32) == 100
    assert oracle.batch_size(10**6, 64 * 10000 - 1, 2, 32) == 99
    # monotone in memory, never above |S|, never below min(|S|, 32)
    prev = 0
    for m in [0, 10, 10**3, 10**6, 10**9, 10**12, 10**15]:
        b = oracle.batch_size(5000, m, 3, 31)
        assert prev <= b <= 5000 and b >= 32
        prev = b
    assert oracle.batch_size(5000, 10**15, 3, 31) == 5000


def test_join_closed_forms():
    # A_i = residue 0 repeated i times; B_j = residue 0 repeated j times: d = |i - j|
    # A_i against a sequence over a disjoint residue: d = max(len)
    A = [[0] * i for i in range(0, 9)]
    B = [[0] * j for j in range(0, 12)] + [[1] * 5]
    sa, oa = _pack(A)
    sb, ob = _pack(B)
    p, d = oracle.join_threshold(sa, oa, sb, ob, 3)
    want = [(i, j, abs(i - j)) for i in range(9) for j in range(12) if abs(i - j) <= 3]
    want += [(i, 12, 5) for i in range(9) if max(i, 5) <= 3]        # none: max(i, 5) >= 5
    want.sort()
    assert [(int(a), int(b), int(c)) for (a, b), c in zip(p, d)] == want
    p5, d5 = oracle.join_threshold(sa, oa, sb, ob, 5)
    got = {(int(a), int(b)): int(c) for (a, b), c in zip(p5, d5)}
    for i in range(9):
        assert (got.get((i, 12)) == max(i, 5)) == (max(i, 5) <= 5)
        if max(i, 5) > 5:
            assert (i, 12) not in got


def test_join_planted_copies_and_symmetry():
    rng = np.random.default_rng(5)
    A = [rng.integers(0, 20, rng.integers(8, 21)).astype(np.uint8) for _ in range(60)]
    # B: for every A_i one exact copy and one copy with a single substitution, shuffled, plus noise
    B, src, edits = [], [], []
    for i, s in enumerate(A):
        B.append(s.copy()); src.append(i); edits.append(0)
        t = s.copy(); pos = rng.integers(0, len(t)); t[pos] = (t[pos] + 1 + rng.integers(0, 19)) % 20
        B.append(t); src.append(i); edits.append(1)
    for _ in range(40):
        B.append(rng.integers(0, 20, rng.integers(8, 21)).astype(np.uint8)); src.append(-1); edits.append(-1)
    perm = rng.permutation(len(B))
    B = [B[q] for q in perm]; src = [src[q] for q in perm]; edits = [edits[q] for q in perm]
    sa, oa = _pack(A)
    sb, ob = _pack(B)
    p, d = oracle.join_threshold(sa, oa, sb, ob, 2)
    got = {(int(a), int(b)): int(c) for (a, b), c in zip(p, d)}
    for j, (i, e) in enumerate(zip(src, edits)):
        if i >= 0:
            assert (i, j) in got and got[(i, j)] == e       # a substitution of a different residue: d = 1
    # ascending (i, j)
    key = p[:, 0].astype(np.int64) * len(B) + p[:, 1]
    assert np.all(np.diff(key) > 0)
    # symmetry: join(B, A) is the transpose
    pt, dt = oracle.join_threshold(sb, ob, sa, oa, 2)
    assert {(int(b), int(a)): int(c) for (a, b), c in zip(pt, dt)} == got


def test_self_join_upper_equals_all_pairs_routine():
    rep = datagen.config2(700, seed=3)
    seqs, off = rep.seqs, rep.offsets
    max_d = 3
    p, d = oracle.join_threshold(seqs, off, seqs, off, max_d, upper=True)
    p2, d2 = oracle.all_pairs_threshold(seqs, off, max_d)
    assert np.array_equal(p, p2) and np.array_equal(d, d2)
    # without `upper` the rectangle holds the diagonal (d = 0) and both orientations
    pf, df = oracle.join_threshold(seqs, off, seqs, off, max_d, upper=False)
    n = off.shape[0] - 1
    assert pf.shape[0] == 2 * p.shape[0] + n
    diag = pf[:, 0] == pf[:, 1]
    assert diag.sum() == n and np.all(df[diag] == 0)


def test_join_empty_sides():
    sa, oa = _pack([[1, 2, 3]])
    se, oe = _pack([])
    p, d = oracle.join_threshold(sa, oa, se, oe, 2)
    assert p.shape == (0, 2) and d.shape == (0,)
    p, d = oracle.join_threshold(se, oe, sa, oa, 2)
    assert p.shape == (0, 2) and d.shape == (0,)
