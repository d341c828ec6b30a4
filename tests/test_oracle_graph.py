"""Pins of the oracle's graph step: a hand-worked example, closed forms and
the link between the integer match count and the (already pinned) MinHash Jaccard estimate."""
import numpy as np

import oracle
from paper_2602_17330_b200 import datagen as dg


def test_hand_worked_example():
    # 4 sequences of lengths 7, 5, 7, 0; sketches of H = 4 columns
    sig = np.array([[1, 2, 3, 4], [1, 2, 3, 9], [1, 8, 8, 8], [1, 2, 3, 4]], np.uint32)
    lengths = np.array([7, 5, 7, 0])
    pairs = np.array([[0, 1], [0, 2], [0, 3], [1, 2], [2, 3]], np.uint32)
    dist = np.array([2, 1, 0, 5, 3], np.uint16)
    # max_d = 3 drops (1,2); min_matches = 3 drops (0,2) [1 match] and (2,3) [1 match]
    rp, col, w = oracle.affinity_graph(pairs, dist, 3, sig, 3, lengths, 4)
    assert rp.tolist() == [0, 2, 2, 2, 2]
    assert col.tolist() == [1, 3]
    assert np.allclose(w, [1 - 2 / 7, 1 - 0 / 7])
    # no sketch filter: (0,1), (0,2), (0,3), (2,3) stay
    rp, col, w = oracle.affinity_graph(pairs, dist, 3, None, 0, lengths, 4)
    assert rp.tolist() == [0, 3, 3, 4, 4] and col.tolist() == [1, 2, 3, 3]
    assert np.allclose(w, [1 - 2 / 7, 1 - 1 / 7, 1.0, 1 - 3 / 7])


def test_closed_forms_and_link_to_the_jaccard_estimate():
    rep = dg.config2(3000, seed=2)
    P = dg.PARAMS["config2"]
    sig = oracle.minhash(rep.seqs, rep.offsets, P["k"], P["H"], dg.DEFAULT_SEED64)
    pairs, _, _ = oracle.lsh_sorted(sig, P["bands"], P["rows"], P["cap"])
    dist = oracle.edit_distance_pairs(rep.seqs, rep.offsets, pairs, P["max_d"])
    H = P["H"]
    rp0, col0, w0 = oracle.affinity_graph(pairs, dist, P["max_d"], sig, 0, rep.lengths, rep.n)
    assert rp0[-1] == (dist <= P["max_d"]).sum() == col0.size
    assert (np.diff(rp0) >= 0).all() and (w0 >= 0).all() and (w0 <= 1).all()
    # monotone in the threshold; min_matches = H keeps only identical sketches
    prev = rp0[-1]
    for mm in (16, 32, 48, 64):
        rp, col, w = oracle.affinity_graph(pairs, dist, P["max_d"], sig, mm, rep.lengths, rep.n)
        assert rp[-1] <= prev
        prev = rp[-1]
    same = (sig[pairs[:, 0]] == sig[pairs[:, 1]]).all(axis=1) & (dist <= P["max_d"])
    assert prev == same.sum()
    # matches / H is the MinHash estimate of the exact k-mer Jaccard (pinned in test_oracle_minhash):
    # on the kept edges at tau = 0.5 the exact Jaccard averages well above the dropped ones
    mm = H // 2
    m = (sig[pairs[:, 0]] == sig[pairs[:, 1]]).sum(axis=1)
    take = np.random.default_rng(0).choice(pairs.shape[0], 400, replace=False)
    J = []
    for t in take:
        num, den = oracle.kmer_jaccard(rep.seq(int(pairs[t, 0])), rep.seq(int(pairs[t, 1])), P["k"])
        J.append(num / den if den else 1.0)
    J = np.array(J)
    assert abs((m[take] / H - J).mean()) < 3 * 0.5 / np.sqrt(H) / np.sqrt(take.size) + 0.01
    assert J[m[take] >= mm].mean() > J[m[take] < mm].mean()
