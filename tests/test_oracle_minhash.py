"""Pins for the oracle's MinHash (spec C2; Eq. 30).

The paper gives no hash family, so there is no printed value.  Pins: constants
against their mathematical definition, bijectivity of the mixer via its inverse,
closed forms of the sketch, set-level invariants, and the statistical statement
the paper does make -- the Jaccard estimate's error is within 1/sqrt(M).
"""
import math

import numpy as np
import pytest

import oracle
from paper_2602_17330_b200 import datagen as dg

SEED = dg.DEFAULT_SEED64
M32 = 0xFFFFFFFF


def test_constants_are_the_stated_irrationals():
    # 0x6A09E667 = floor(frac(sqrt 2) * 2^32), 0xBB67AE85 = floor(frac(sqrt 3) * 2^32)
    c2 = math.isqrt(2 << 64) - (1 << 32)
    c3 = math.isqrt(3 << 64) - (1 << 32)
    assert c2 == 0x6A09E667 and c3 == 0xBB67AE85
    # g(1) only touches the two multipliers and the shifts: x=1 -> 1*c2, ^>>15, *c3, ^>>16
    x = c2
    x ^= x >> 15
    x = (x * c3) & M32
    x ^= x >> 16
    assert oracle.mix32(1) == x
    assert oracle.mix32(0) == 0


def _unxorshift(x, s):
    y = x
    for _ in range(32 // s + 1):
        y = x ^ (y >> s)
    return y


def test_mixer_is_a_bijection():
    inv2 = pow(0x6A09E667, -1, 1 << 32)
    inv3 = pow(0xBB67AE85, -1, 1 << 32)
    rng = np.random.default_rng(0)
    xs = [0, 1, M32, 0x80000000] + [int(v) for v in rng.integers(0, 1 << 32, 3000)]
    for x in xs:
        y = oracle.mix32(x)
        y = _unxorshift(y, 16)
        y = (y * inv3) & M32
        y = _unxorshift(y, 15)
        y = (y * inv2) & M32
        y = _unxorshift(y, 16)
        assert y == x
    # injective on the whole 15-bit k=3 k-mer space
    assert len({oracle.mix32(x) for x in range(1 << 15)}) == 1 << 15


def test_hash_params_odd_multipliers_and_seed_dependence():
    a, b = oracle.hash_params(SEED, 256)
    assert (a & 1).all()
    assert len(set(a.tolist())) == 256 and len(set(b.tolist())) == 256
    a2, b2 = oracle.hash_params(SEED ^ 1, 256)               # lo half feeds a only
    assert (a2 != a).mean() > 0.99 and (b2 == b).all()
    a3, b3 = oracle.hash_params(SEED ^ (1 << 32), 256)       # hi half feeds b only
    assert (a3 == a).all() and (b3 != b).mean() > 0.99
    # prefix property: parameters of hash j do not depend on H
    a64, b64 = oracle.hash_params(SEED, 64)
    assert (a64 == a[:64]).all() and (b64 == b[:64]).all()


def test_hash_params_hand_worked_values():
    """a_j = g(lo ^ g(2j+1)) | 1, b_j = g(hi ^ g(2j+2)) with lo / hi the low /
    high 32 bits of the seed.  Three (seed, j) cases worked step by step from the text of C2 --
    every intermediate of the mixer is a literal below, so the chain can be checked with a hex
    calculator; nothing here calls the oracle except the final comparison.  A wrong index
    (2j for 2j+1), swapped seed halves or a dropped `| 1` changes the literals."""
    def g_steps(x):                      # C2's mixer, one line per statement
        s = [x]
        x ^= x >> 16; s.append(x)
        x = (x * 0x6A09E667) & M32; s.append(x)
        x ^= x >> 15; s.append(x)
        x = (x * 0xBB67AE85) & M32; s.append(x)
        x ^= x >> 16; s.append(x)
        return s
    # g(1) and g(2): the inner values of j = 0
    assert g_steps(1) == [0x1, 0x1, 0x6A09E667, 0x6A093274, 0x5FBE0E44, 0x5FBE51FA]
    assert g_steps(2) == [0x2, 0x2, 0xD413CCCE, 0xD41264E9, 0x7AE3CB0D, 0x7AE3B1EE]
    # seed = 0, j = 0: a_0 = g(0 ^ g(1)) | 1 (the mixer ends on an even value here, so the `| 1`
    # is visible), b_0 = g(0 ^ g(2))
    assert g_steps(0x5FBE51FA) == [0x5FBE51FA, 0x5FBE0E44, 0xEEACD55C, 0xEEAD0805, 0x7C5B9099, 0x7C5BECC2]
    assert g_steps(0x7AE3B1EE) == [0x7AE3B1EE, 0x7AE3CB0D, 0x9F89603B, 0x9F885F29, 0xCF064E4D, 0xCF06814B]
    a, b = oracle.hash_params(0, 1)
    assert (int(a[0]), int(b[0])) == (0x7C5BECC3, 0xCF06814B)
    # the default seed 0x5EED5EED12345678: lo = 0x12345678 feeds a, hi = 0x5EED5EED feeds b
    assert 0x12345678 ^ 0x5FBE51FA == 0x4D8A0782 and 0x5EED5EED ^ 0x7AE3B1EE == 0x240EEF03
    assert g_steps(0x4D8A0782) == [0x4D8A0782, 0x4D8A4A08, 0x5B6EF938, 0x5B6E4FE5, 0xE6C027F9, 0xE6C0C139]
    assert g_steps(0x240EEF03) == [0x240EEF03, 0x240ECB0D, 0x51D6603B, 0x51D6C397, 0x7C453F73, 0x7C454336]
    a, b = oracle.hash_params(SEED, 8)
    assert SEED == 0x5EED5EED12345678
    assert (int(a[0]), int(b[0])) == (0xE6C0C139, 0x7C454336)
    # j = 5: inner arguments 2j+1 = 11 and 2j+2 = 12
    assert g_steps(11)[-1] == 0x19F58E71 and g_steps(12)[-1] == 0xFED0F94D
    assert g_steps(0x12345678 ^ 0x19F58E71)[-1] | 1 == 0x93F264E5
    assert g_steps(0x5EED5EED ^ 0xFED0F94D)[-1] == 0x55392642
    assert (int(a[5]), int(b[5])) == (0x93F264E5, 0x55392642)
    # lo = 0, hi = 1, j = 3: only b sees the seed
    a, b = oracle.hash_params(1 << 32, 4)
    assert g_steps(7)[-1] == 0x4E71C736 and g_steps(8)[-1] == 0x797CF042
    assert (int(a[3]), int(b[3])) == (g_steps(0x4E71C736)[-1] | 1, g_steps(1 ^ 0x797CF042)[-1])
    assert (int(a[3]), int(b[3])) == (0x6DDCADAF, 0xB0C239BA)


def test_closed_form_single_kmer():
    # poly-A: the only k-mer is x = 0 and g(0) = 0, so sig[j] = a_j*0 + b_j = b_j
    _, b = oracle.hash_params(SEED, 64)
    for L in (3, 4, 9):
        rep = dg.from_list([[0] * L])
        sig = oracle.minhash(rep.seqs, rep.offsets, 3, 64, SEED)
        assert (sig[0] == b).all()
    # a single general k-mer x: sig[j] = a_j*g(x) + b_j
    a, b = oracle.hash_params(SEED, 64)
    rep = dg.from_list([[7, 19, 3]])
    x = 7 * 32 * 32 + 19 * 32 + 3                          # x_p = sum code * 32^(k-1-t)
    want = (a.astype(np.uint64) * np.uint64(oracle.mix32(x)) + b.astype(np.uint64)) & np.uint64(M32)
    sig = oracle.minhash(rep.seqs, rep.offsets, 3, 64, SEED)
    assert (sig[0] == want.astype(np.uint32)).all()


def test_short_sequences_get_the_sentinel():
    rep = dg.from_list([[], [1], [1, 2], [1, 2, 3]])
    sig = oracle.minhash(rep.seqs, rep.offsets, 3, 32, SEED)
    assert (sig[:3] == M32).all()
    assert (sig[3] != M32).any()


def test_set_semantics_union_and_order_invariance():
    rng = np.random.default_rng(2)
    k, H = 3, 64
    for _ in range(50):
        A = rng.integers(0, 20, rng.integers(5, 20)).astype(np.uint8)
        B = rng.integers(0, 20, rng.integers(5, 20)).astype(np.uint8)
        # "A then separator-free join" would create new k-mers; instead build sequences whose
        # k-mer SETS are known: repeat A twice (same set as A plus the junction k-mers).
        rep = dg.from_list([A, B])
        sA, sB = oracle.minhash(rep.seqs, rep.offsets, k, H, SEED)
        # one sequence per k-mer of A and of B: sketch of a union = elementwise min
        kms = [A[p:p + k] for p in range(len(A) - k + 1)] + [B[p:p + k] for p in range(len(B) - k + 1)]
        rep2 = dg.from_list(kms)
        sk = oracle.minhash(rep2.seqs, rep2.offsets, k, H, SEED)
        nA = len(A) - k + 1
        assert (sk[:nA].min(axis=0) == sA).all()
        assert (sk[nA:].min(axis=0) == sB).all()
        # duplicates do not matter: A+A has set(A) plus junction k-mers >= as a set
        AA = np.concatenate([A, A])
        rep3 = dg.from_list([AA])
        sAA = oracle.minhash(rep3.seqs, rep3.offsets, k, H, SEED)[0]
        assert (sAA <= sA).all()
    # identical sequences -> identical signatures; reversed periodic sequence same set
    rep = dg.from_list([[1, 2, 1, 2, 1, 2, 1], [2, 1, 2, 1, 2, 1, 2, 1, 2]])
    s = oracle.minhash(rep.seqs, rep.offsets, 3, 32, SEED)
    assert (s[0] == s[1]).all()          # both have k-mer set {121, 212}


def test_kmer_jaccard_tiny_sets():
    # {ABC, BCD} vs {BCD, CDE}: J = 1/3
    assert oracle.kmer_jaccard([0, 1, 2, 3], [1, 2, 3, 4], 3) == (1, 3)
    assert oracle.kmer_jaccard([0, 1, 2, 3], [0, 1, 2, 3], 3) == (2, 2)
    assert oracle.kmer_jaccard([0, 1, 2], [5, 6, 7], 3) == (0, 2)
    assert oracle.kmer_jaccard([0, 0, 0, 0, 0], [0, 0, 0], 3) == (1, 1)


@pytest.mark.parametrize("k,H", [(3, 64), (4, 128), (3, 256)])
def test_collision_rate_converges_to_jaccard(k, H):
    """PAPER.md L495-497 Eq. (30): s.e. of the Jaccard estimate <= 1/sqrt(M).
    Mean error within 4 s.e. of 0 (unbiased) and RMS error <= 1/sqrt(H); the RMS must
    also match the binomial prediction sqrt(J(1-J)/H) within 15 %."""
    r = dg.config2(6000, seed=21) if k == 3 else dg.config3(6000, seed=21)
    sig = oracle.minhash(r.seqs, r.offsets, k, H, SEED)
    rng = np.random.default_rng(5)
    order = np.argsort(r.family, kind="stable")
    errs, preds = [], []
    for _ in range(3000):
        q = rng.integers(0, r.n - 1)
        i, j = order[q], order[q + 1]
        if r.family[i] != r.family[j]:
            continue
        num, den = oracle.kmer_jaccard(r.seq(i), r.seq(j), k)
        J = num / den
        Jhat = float((sig[i] == sig[j]).mean())
        errs.append(Jhat - J)
        preds.append(J * (1 - J) / H)
    errs = np.array(errs)
    assert errs.size > 2000
    rms = float(np.sqrt((errs ** 2).mean()))
    pred = float(np.sqrt(np.mean(preds)))
    assert abs(errs.mean()) < 4 * rms / math.sqrt(errs.size)
    assert rms <= 1.0 / math.sqrt(H)
    assert 0.85 * pred <= rms <= 1.15 * pred


def test_tiny_set_collision_rate_many_hashes():
    # north_star: "MinHash collision rate converging to the exact k-mer Jaccard on tiny sets"
    H = 4096
    cases = [([0, 1, 2, 3], [1, 2, 3, 4]),           # J = 1/3
             ([0, 1, 2, 3, 4], [0, 1, 2, 3, 5]),     # {012,123,234} vs {012,123,235}: J = 2/4
             ([3, 4, 5], [3, 4, 5, 6, 7, 8])]        # J = 1/4
    for s, t in cases:
        num, den = oracle.kmer_jaccard(s, t, 3)
        rep = dg.from_list([s, t])
        sig = oracle.minhash(rep.seqs, rep.offsets, 3, H, SEED)
        rate = float((sig[0] == sig[1]).mean())
        J = num / den
        assert abs(rate - J) < 4 * math.sqrt(J * (1 - J) / H)
