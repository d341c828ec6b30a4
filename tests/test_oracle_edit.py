"""Pins for the oracle's edit distance (spec C1; Eq. 46).

The paper prints no worked example, so the oracle is pinned to textbook values,
an independent definition (BFS over single edit operations), the metric
invariants, and closed-form special cases.  None of these retypes the recurrence.
"""
import itertools
import os
from collections import deque

import numpy as np
import pytest

import oracle
from paper_2602_17330_b200 import datagen as dg

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "edit_distance_textbook.txt")


def _codes(s):
    return np.array([ord(c) - ord("a") + 1 for c in s], dtype=np.uint8)


def test_textbook_values():
    n = 0
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        a, b, d = line.split()
        a = "" if a == "-" else a
        b = "" if b == "-" else b
        assert oracle.edit_distance(_codes(a), _codes(b)) == int(d), (a, b)
        n += 1
    assert n >= 15


def test_kitten_sitting_is_3():
    # named in BASELINE.json north_star
    assert oracle.edit_distance(_codes("kitten"), _codes("sitting")) == 3


def _bfs_distances(src, alphabet, max_len):
    """Shortest number of single-symbol insertions/deletions/substitutions from `src` to every
    string over `alphabet` with length <= max_len (an independent definition of Levenshtein
    distance: shortest path in the edit graph; intermediate strings of an optimal script never
    need to be longer than max(len(src), len(dst)))."""
    dist = {src: 0}
    q = deque([src])
    while q:
        s = q.popleft()
        d = dist[s]
        nxt = []
        for p in range(len(s)):
            nxt.append(s[:p] + s[p + 1:])
            for c in alphabet:
                if c != s[p]:
                    nxt.append(s[:p] + (c,) + s[p + 1:])
        if len(s) < max_len:
            for p in range(len(s) + 1):
                for c in alphabet:
                    nxt.append(s[:p] + (c,) + s[p:])
        for t in nxt:
            if t not in dist:
                dist[t] = d + 1
                q.append(t)
    return dist


@pytest.mark.parametrize("alphabet,max_len", [((0, 1), 5), ((0, 1, 2), 4)])
def test_exhaustive_vs_bfs(alphabet, max_len):
    strings = [()]
    for L in range(1, max_len + 1):
        strings += list(itertools.product(alphabet, repeat=L))
    checked = 0
    for a in strings:
        dist = _bfs_distances(a, alphabet, max_len)
        for b in strings:
            assert oracle.edit_distance(list(a), list(b)) == dist[b], (a, b)
            checked += 1
    assert checked == len(strings) ** 2


def test_metric_invariants_random():
    rng = np.random.default_rng(1)
    seqs = [rng.integers(0, 20, rng.integers(0, 30)).astype(np.uint8) for _ in range(60)]
    D = np.zeros((60, 60), int)
    for i in range(60):
        for j in range(60):
            D[i, j] = oracle.edit_distance(seqs[i], seqs[j])
    for i in range(60):
        assert D[i, i] == 0
        for j in range(60):
            la, lb = len(seqs[i]), len(seqs[j])
            assert D[i, j] == D[j, i]
            assert abs(la - lb) <= D[i, j] <= max(la, lb)
            if la == lb:
                assert D[i, j] <= int((seqs[i] != seqs[j]).sum())      # <= Hamming
            if D[i, j] == 0:
                assert la == lb and (seqs[i] == seqs[j]).all()
    # triangle inequality on all triples
    for i in range(60):
        # D[i,k] <= D[i,j] + D[j,k] for all j, k
        assert (D[i][None, :] > (D[i][:, None] + D)).sum() == 0


def test_distance_bounded_by_generator_edits():
    # a family member is its seed with e edits  =>  d(i, j) <= e_i + e_j inside a family
    r = dg.config2(3000, seed=3)
    order = np.argsort(r.family, kind="stable")
    fam = r.family[order]
    pairs = []
    for a, b in zip(order[:-1], order[1:]):
        if r.family[a] == r.family[b]:
            pairs.append((a, b))
    pairs = np.array(pairs, np.uint32)
    d = oracle.edit_distance_pairs(r.seqs, r.offsets, pairs, -1)
    bound = r.n_edits[pairs[:, 0]].astype(int) + r.n_edits[pairs[:, 1]].astype(int)
    assert (d <= bound).all()
    assert fam.size == r.n


def test_saturation_and_pair_list():
    r = dg.config1(300, seed=5)
    rng = np.random.default_rng(0)
    pairs = rng.integers(0, 300, (2000, 2)).astype(np.uint32)
    exact = oracle.edit_distance_pairs(r.seqs, r.offsets, pairs, -1)
    for md in (0, 3, 7):
        sat = oracle.edit_distance_pairs(r.seqs, r.offsets, pairs, md)
        assert (sat == np.minimum(exact, md + 1)).all()
    # single calls agree with the batched entry point
    for p in range(0, 2000, 97):
        i, j = pairs[p]
        assert exact[p] == oracle.edit_distance(r.seq(i), r.seq(j))


def test_cutoff_equals_full_dp():
    # Tier B (Ukkonen cut-off) == Tier A whenever d <= max_d, and > max_d otherwise
    rng = np.random.default_rng(7)
    r = dg.config2(4000, seed=11)
    n_checked = 0
    for _ in range(20000):
        i, j = rng.integers(0, r.n, 2)
        if rng.random() < 0.5:     # bias towards related pairs
            same = np.nonzero(r.family == r.family[i])[0]
            j = same[rng.integers(0, same.size)]
        a, b = r.seq(i), r.seq(j)
        full = oracle.edit_distance(a, b)
        for md in (0, 2, 3, 6):
            c = oracle.edit_distance_cutoff(a, b, md)
            assert c == min(full, md + 1)
        n_checked += 1
    assert n_checked == 20000


def test_all_pairs_full_layout_and_threshold_filter():
    r = dg.config1(120, seed=9)
    full = oracle.all_pairs_full(r.seqs, r.offsets)
    n = r.n
    assert full.size == n * (n - 1) // 2
    k = 0
    ii, jj = [], []
    for i in range(n):
        for j in range(i + 1, n):
            ii.append(i); jj.append(j)
            if (i * 7 + j) % 53 == 0:
                assert full[k] == oracle.edit_distance(r.seq(i), r.seq(j))
            k += 1
    ii, jj = np.array(ii), np.array(jj)
    for md, cut in ((6, False), (6, True), (9, True)):
        pairs, dist = oracle.all_pairs_threshold(r.seqs, r.offsets, md, use_cutoff=cut)
        sel = full <= md
        assert (pairs[:, 0] == ii[sel]).all() and (pairs[:, 1] == jj[sel]).all()
        assert (dist == full[sel]).all()


def test_empty_sequences():
    assert oracle.edit_distance([], []) == 0
    assert oracle.edit_distance([], [1, 2, 3]) == 3
    rep = dg.from_list([[], [1, 2], [], [1, 3, 2]])
    full = oracle.all_pairs_full(rep.seqs, rep.offsets)
    assert full.tolist() == [2, 0, 3, 2, 1, 3]
