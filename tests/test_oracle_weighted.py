"""Pins of the oracle's weighted edit distance (Eq. 46 with a
substitution table).  The paper prints no matrix and no worked example: the pins are the
reduction to the pinned unit-cost oracle, scaling, bounds, closed forms, and an independent
definition (Dijkstra over STRINGS under single edit operations) on tiny inputs."""
import heapq
import itertools

import numpy as np

import oracle
from paper_2602_17330_b200 import datagen as dg


def _unit(sigma):
    c = np.ones((sigma, sigma), np.uint8)
    np.fill_diagonal(c, 0)
    return c


def test_unit_table_is_levenshtein():
    rng = np.random.default_rng(0)
    u = _unit(20)
    for _ in range(3000):
        a = rng.integers(0, 20, rng.integers(0, 30))
        b = rng.integers(0, 20, rng.integers(0, 30))
        assert oracle.edit_distance_weighted(a, b, u, 1) == oracle.edit_distance(a, b)


def test_scaling_and_bounds():
    rng = np.random.default_rng(1)
    c = dg.class_substitution_costs()
    for _ in range(2000):
        a = rng.integers(0, 20, rng.integers(0, 25))
        b = rng.integers(0, 20, rng.integers(0, 25))
        d = oracle.edit_distance_weighted(a, b, c, 1)
        lev = oracle.edit_distance(a, b)
        assert lev <= d <= 2 * lev                       # every operation costs between 1 and 2
        assert oracle.edit_distance_weighted(a, b, (3 * c).astype(np.uint8), 3) == 3 * d
        assert d == oracle.edit_distance_weighted(b, a, c, 1)          # symmetric table
        assert abs(len(a) - len(b)) <= d


def test_closed_forms():
    c = dg.class_substitution_costs()
    A, G, I, K = (dg.ALPHABET.index(x) for x in "AGIK")
    s = [A, I, K, K, G, A]
    assert oracle.edit_distance_weighted(s, s, c, 1) == 0
    assert oracle.edit_distance_weighted([], s, c, 2) == 2 * len(s)
    t = list(s); t[1] = dg.ALPHABET.index("L")            # I -> L: same class
    assert oracle.edit_distance_weighted(s, t, c, 1) == 1
    t = list(s); t[1] = K                                  # I -> K: other class
    assert oracle.edit_distance_weighted(s, t, c, 1) == 2
    # an expensive substitution is replaced by delete + insert when 2*indel is cheaper
    big = _unit(20) * 9
    assert oracle.edit_distance_weighted([A], [K], big.astype(np.uint8), 2) == 4
    # asymmetric table: row = residue of the first argument
    asym = _unit(4).astype(np.uint8); asym[0, 1] = 3; asym[1, 0] = 1
    assert oracle.edit_distance_weighted([0], [1], asym, 5) == 3
    assert oracle.edit_distance_weighted([1], [0], asym, 5) == 1


def _dijkstra_strings(a, b, cost, indel, sigma, max_len):
    """Cheapest sequence of single edit operations turning string a into b (strings as tuples)."""
    a, b = tuple(a), tuple(b)
    dist = {a: 0}
    pq = [(0, a)]
    while pq:
        d, s = heapq.heappop(pq)
        if s == b:
            return d
        if d > dist.get(s, 1 << 30):
            continue
        nxt = []
        for p in range(len(s)):
            nxt.append((indel, s[:p] + s[p + 1:]))
            for ch in range(sigma):
                if ch != s[p]:
                    nxt.append((int(cost[s[p], ch]), s[:p] + (ch,) + s[p + 1:]))
        if len(s) < max_len:
            for p in range(len(s) + 1):
                for ch in range(sigma):
                    nxt.append((indel, s[:p] + (ch,) + s[p:]))
        for w, t in nxt:
            if d + w < dist.get(t, 1 << 30):
                dist[t] = d + w
                heapq.heappush(pq, (d + w, t))
    raise AssertionError("unreachable")


def test_independent_definition_on_tiny_strings():
    # metric tables only: with a metric, the cheapest operation sequence is an alignment
    sigma = 3
    tables = [(np.array([[0, 1, 2], [1, 0, 1], [2, 1, 0]], np.uint8), 1),
              (np.array([[0, 2, 3], [2, 0, 2], [3, 2, 0]], np.uint8), 2),
              (np.array([[0, 1, 1], [1, 0, 2], [1, 2, 0]], np.uint8), 1)]
    strings = [s for L in range(0, 4) for s in itertools.product(range(sigma), repeat=L)]
    rng = np.random.default_rng(2)
    for cost, indel in tables:
        for _ in range(120):
            a = strings[rng.integers(len(strings))]
            b = strings[rng.integers(len(strings))]
            want = _dijkstra_strings(a, b, cost, indel, sigma, 4)
            got = oracle.edit_distance_weighted(np.array(a, np.uint8), np.array(b, np.uint8), cost, indel)
            assert got == want, (a, b, cost.tolist(), indel)


def test_pairs_entry_point_saturates_like_the_unit_cost_one():
    rep = dg.config2(3000, seed=4)
    rng = np.random.default_rng(3)
    pairs = rng.integers(0, rep.n, (5000, 2)).astype(np.uint32)
    c = dg.class_substitution_costs()
    exact = oracle.edit_distance_weighted_pairs(rep.seqs, rep.offsets, pairs, c, 1, -1)
    for md in (0, 4, 9):
        got = oracle.edit_distance_weighted_pairs(rep.seqs, rep.offsets, pairs, c, 1, md)
        assert np.array_equal(got, np.minimum(exact, md + 1))
    one = oracle.edit_distance_weighted(rep.seq(int(pairs[7, 0])), rep.seq(int(pairs[7, 1])), c, 1)
    assert exact[7] == one


def test_equal_residues_cost_nothing_whatever_the_diagonal_says():
    """PAPER.md L754 Eq. 46 prints  d[x-1][y-1] + I(s_i[x] != s_j[y]) * substitution_cost : the
    indicator makes a match free, so the table's DIAGONAL is never used (reading 22b)."""
    rng = np.random.default_rng(7)
    sigma = 5
    for _ in range(300):
        cost = rng.integers(1, 6, (sigma, sigma)).astype(np.uint8)         # non-zero diagonal
        zero = cost.copy()
        np.fill_diagonal(zero, 0)
        a = rng.integers(0, sigma, rng.integers(0, 9))
        b = rng.integers(0, sigma, rng.integers(0, 9))
        indel = int(rng.integers(1, 4))
        assert oracle.edit_distance_weighted(a, b, cost, indel) == oracle.edit_distance_weighted(a, b, zero, indel)
        assert oracle.edit_distance_weighted(a, a, cost, indel) == 0       # d(s, s) = 0: every step a match
    # hand-worked: a = [0, 1], b = [0, 2], cost[1][2] = 4, indel = 3, diagonal = 5 everywhere.
    # Align 0-0 (match: 0, not cost[0][0] = 5) and 1-2 (substitution: 4)  =>  4; the alternative
    # delete + insert costs 6.
    cost = np.full((3, 3), 5, np.uint8)
    cost[1, 2] = 4
    assert oracle.edit_distance_weighted([0, 1], [0, 2], cost, 3) == 4
