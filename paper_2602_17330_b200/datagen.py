"""Seeded synthetic CDR3-like repertoires (numpy only).

This module holds NONE of the method's arithmetic (no hashing, no banding, no
edit distance): it only draws the inputs.  The CPU oracle (`oracle/`) and the CUDA
path both receive the arrays it returns; neither of them imports the other.

The generators stand in for the paper's VDJdb / McPAS-TCR / NEPdb CDR3-beta
repertoires at 10^4..10^7 sequences, which are
not available here.  Shapes, sizes and value distributions follow BASELINE.json
`configs[0..4]`; the exact recipe is restated in DESIGN.md ("Input recipe").

Every generator returns a `Repertoire`:
    seqs    uint8[total]   residue codes 0..19 (A C D E F G H I K L M N P Q R S T V W Y)
    offsets int64[n+1]     sequence i is seqs[offsets[i]:offsets[i+1]]
    family  int32[n]       family id of each sequence (-1: no family structure)
    n_edits uint8[n]       number of edits applied to the family seed
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SIGMA = 20
ALPHABET = "ACDEFGHIKLMNPQRSTVWY"


@dataclass
class Repertoire:
    seqs: np.ndarray
    offsets: np.ndarray
    family: np.ndarray
    n_edits: np.ndarray
    name: str = ""

    @property
    def n(self) -> int:
        return int(self.offsets.shape[0] - 1)

    @property
    def lengths(self) -> np.ndarray:
        return np.diff(self.offsets)

    def seq(self, i: int) -> np.ndarray:
        return self.seqs[self.offsets[i]:self.offsets[i + 1]]

    def as_str(self, i: int) -> str:
        return "".join(ALPHABET[c] for c in self.seq(i))


def encode(s: str) -> np.ndarray:
    """One-letter amino-acid string -> uint8 codes (alphabetical order)."""
    return np.array([ALPHABET.index(c) for c in s], dtype=np.uint8)


def from_list(seqs) -> Repertoire:
    """Build a Repertoire from a list of uint8 arrays / lists of codes."""
    arrs = [np.asarray(s, dtype=np.uint8).reshape(-1) for s in seqs]
    lens = np.array([a.shape[0] for a in arrs], dtype=np.int64)
    offsets = np.zeros(len(arrs) + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    flat = np.concatenate(arrs) if arrs and offsets[-1] > 0 else np.zeros(0, np.uint8)
    n = len(arrs)
    return Repertoire(flat.astype(np.uint8), offsets, np.full(n, -1, np.int32),
                      np.zeros(n, np.uint8), "list")


# ---------------------------------------------------------------------------
# helpers
# ---------------------------------------------------------------------------

def _residue_probs(kind: str) -> np.ndarray:
    if kind == "uniform":
        return np.full(SIGMA, 1.0 / SIGMA)
    if kind == "zipf1.1":
        w = 1.0 / np.arange(1, SIGMA + 1, dtype=np.float64) ** 1.1
        return w / w.sum()
    raise ValueError(kind)


def _draw_residues(rng, probs, size):
    cdf = np.cumsum(probs)
    cdf[-1] = 1.0
    return np.searchsorted(cdf, rng.random(size), side="right").astype(np.uint8)


def _draw_other_residue(rng, probs, old):
    """Residue drawn from `probs` conditioned on != old (vectorised rejection)."""
    new = _draw_residues(rng, probs, old.shape[0])
    bad = np.nonzero(new == old)[0]
    while bad.size:
        new[bad] = _draw_residues(rng, probs, bad.size)
        bad = bad[new[bad] == old[bad]]
    return new


def _flatten(mat, lens):
    """Padded [n, W] matrix + lengths -> (flat uint8, offsets int64)."""
    n, W = mat.shape
    offsets = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    mask = np.arange(W, dtype=np.int32)[None, :] < lens[:, None]
    return np.ascontiguousarray(mat[mask]), offsets


def _mutate_block(rng, mat, lens, n_edits, probs, max_edits):
    """Apply n_edits[i] edits to row i of the padded matrix, in place.

    Each edit is a substitution / insertion / deletion with probability 1/3 each
    at a uniform position; a substitution draws from `probs` conditioned on
    != old residue (common rules).
    """
    n, W = mat.shape
    cols = np.arange(W, dtype=np.int32)[None, :]
    for r in range(max_edits):
        act = np.nonzero(n_edits > r)[0]
        if act.size == 0:
            break
        op = rng.integers(0, 3, act.size)            # 0 sub, 1 ins, 2 del
        u = rng.random(act.size)
        L = lens[act].astype(np.int64)
        op = np.where((op == 2) & (L <= 1), 0, op)   # never delete the last residue
        op = np.where((op == 1) & (L >= W), 0, op)   # never overflow the pad width
        # substitution
        s = act[op == 0]
        if s.size:
            pos = np.minimum((u[op == 0] * L[op == 0]).astype(np.int64), L[op == 0] - 1)
            old = mat[s, pos]
            mat[s, pos] = _draw_other_residue(rng, probs, old)
        # insertion before position pos in [0, L]
        s = act[op == 1]
        if s.size:
            Ls = L[op == 1]
            pos = np.minimum((u[op == 1] * (Ls + 1)).astype(np.int64), Ls)
            src = cols - (cols > pos[:, None])
            rows = np.take_along_axis(mat[s], src.astype(np.int64), axis=1)
            rows[np.arange(s.size), pos] = _draw_residues(rng, probs, s.size)
            mat[s] = rows
            lens[s] += 1
        # deletion of position pos in [0, L)
        s = act[op == 2]
        if s.size:
            Ls = L[op == 2]
            pos = np.minimum((u[op == 2] * Ls).astype(np.int64), Ls - 1)
            src = np.minimum(cols + (cols >= pos[:, None]), W - 1)
            mat[s] = np.take_along_axis(mat[s], src.astype(np.int64), axis=1)
            lens[s] -= 1


def _expand_families(rng, seed_mat, seed_lens, fam_of_member, probs, max_edits, pad_w,
                     block=1 << 20):
    """Members = family seed + U{0..max_edits} random edits; returns padded matrix."""
    n = fam_of_member.shape[0]
    n_edits = rng.integers(0, max_edits + 1, n).astype(np.uint8)
    mat = np.zeros((n, pad_w), dtype=np.uint8)
    lens = np.zeros(n, dtype=np.int32)
    n_seeds = seed_mat.shape[0]
    for lo in range(0, n, block):
        hi = min(n, lo + block)
        sid = fam_of_member[lo:hi] % n_seeds
        sub = np.zeros((hi - lo, pad_w), dtype=np.uint8)
        sub[:, :seed_mat.shape[1]] = seed_mat[sid]
        sl = seed_lens[sid].astype(np.int32)
        _mutate_block(rng, sub, sl, n_edits[lo:hi], probs, max_edits)
        mat[lo:hi] = sub
        lens[lo:hi] = sl
    return mat, lens, n_edits


def _geometric_sizes(rng, n_fam, mean, n_total):
    """Geometric(p=1/mean) sizes adjusted to sum exactly to n_total.

    Members are added to / removed from the largest families round-robin
    (SURVEY.md section 8(d), G2)."""
    sizes = rng.geometric(1.0 / mean, n_fam).astype(np.int64)
    diff = int(n_total - sizes.sum())
    order = np.argsort(-sizes, kind="stable")
    k = 0
    while diff != 0:
        f = order[k % n_fam]
        if diff > 0:
            sizes[f] += 1
            diff -= 1
        elif sizes[f] > 1:
            sizes[f] -= 1
            diff += 1
        k += 1
    return sizes


def _powerlaw_sizes(rng, alpha, cap, n_total):
    """Sizes with P(s) ~ s^-alpha on {1..cap}, drawn until n_total is reached;
    the last family is truncated (SURVEY.md section 8(c) reading 20 / G4)."""
    w = 1.0 / np.arange(1, cap + 1, dtype=np.float64) ** alpha
    cdf = np.cumsum(w / w.sum())
    cdf[-1] = 1.0
    out = []
    total = 0
    mean = float((np.arange(1, cap + 1) * w).sum() / w.sum())
    while total < n_total:
        m = max(1024, int((n_total - total) / mean * 1.05) + 16)
        s = np.searchsorted(cdf, rng.random(m), side="right").astype(np.int64) + 1
        cs = np.cumsum(s) + total
        k = int(np.searchsorted(cs, n_total, side="left"))
        if k < m:                       # reached n_total inside this batch
            s = s[:k + 1].copy()
            s[-1] -= int(cs[k] - n_total)
            out.append(s)
            total = n_total
        else:
            out.append(s)
            total = int(cs[-1])
    return np.concatenate(out)


def _seed_sequences(rng, n_seeds, len_kind, probs):
    if len_kind == "normal15_3":
        lens = np.clip(np.rint(rng.normal(15.0, 3.0, n_seeds)), 8, 25).astype(np.int32)
    elif len_kind == "uniform8_25":
        lens = rng.integers(8, 26, n_seeds).astype(np.int32)
    elif len_kind == "uniform110_130":
        lens = rng.integers(110, 131, n_seeds).astype(np.int32)
    else:
        raise ValueError(len_kind)
    W = int(lens.max())
    mat = _draw_residues(rng, probs, n_seeds * W).reshape(n_seeds, W)
    return mat, lens


def families(n, n_seeds, size_law, len_kind, residues, max_edits, seed, name=""):
    """Generic family-mutation generator behind configs 2-5."""
    rng = np.random.default_rng(seed)
    probs = _residue_probs(residues)
    seed_mat, seed_lens = _seed_sequences(rng, n_seeds, len_kind, probs)
    if size_law == "geometric50":
        sizes = _geometric_sizes(rng, n_seeds, 50.0, n)
    elif size_law == "powerlaw2_cap1e4":
        sizes = _powerlaw_sizes(rng, 2.0, 10_000, n)
    elif size_law == "equal":
        sizes = np.full(n_seeds, n // n_seeds, dtype=np.int64)
        sizes[: n - int(sizes.sum())] += 1
    else:
        raise ValueError(size_law)
    fam = np.repeat(np.arange(sizes.shape[0], dtype=np.int32), sizes)
    pad_w = int(seed_lens.max()) + max_edits
    mat, lens, n_edits = _expand_families(rng, seed_mat, seed_lens, fam, probs, max_edits, pad_w)
    perm = rng.permutation(n)                       # families are not contiguous
    mat, lens, fam, n_edits = mat[perm], lens[perm], fam[perm], n_edits[perm]
    flat, offsets = _flatten(mat, lens)
    return Repertoire(flat, offsets, fam, n_edits, name)


# ---------------------------------------------------------------------------
# the five BASELINE.json configs (+ scaled-down variants via `n`)
# ---------------------------------------------------------------------------

def config1(n=2000, seed=0):
    """G1: lengths U{8..20}, iid uniform residues, no families."""
    rng = np.random.default_rng(seed)
    lens = rng.integers(8, 21, n).astype(np.int64)
    offsets = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(lens, out=offsets[1:])
    flat = rng.integers(0, SIGMA, int(offsets[-1])).astype(np.uint8)
    return Repertoire(flat, offsets, np.full(n, -1, np.int32), np.zeros(n, np.uint8), "config1")


def config2(n=100_000, seed=0):
    """G2: n/50 seeds, len ~N(15,3) clipped 8-25, uniform residues, geometric(50) families."""
    return families(n, max(1, n // 50), "geometric50", "normal15_3", "uniform", 3, seed, "config2")


def config3(n=1_000_000, seed=0):
    """G3: n/50 seeds, Zipf(1.1) residues, geometric(50) families."""
    return families(n, max(1, n // 50), "geometric50", "normal15_3", "zipf1.1", 3, seed, "config3")


def config4(n=10_000_000, seed=0):
    """G4: n/100 distinct seed sequences, family sizes ~ s^-2 on {1..10^4} drawn until n."""
    return families(n, max(1, n // 100), "powerlaw2_cap1e4", "uniform8_25", "uniform", 3, seed,
                    "config4")


def config5(n=50_000, seed=0):
    """G5: n/100 seeds of length U{110..130}, 100 members each, 0-10 edits."""
    return families(n, max(1, n // 100), "equal", "uniform110_130", "uniform", 10, seed, "config5")


# parameters of the path for each config (BASELINE.json `configs`)
PARAMS = {
    "config1": dict(k=3, H=32, bands=0, rows=0, cap=0, max_d=-1),
    "config2": dict(k=3, H=64, bands=16, rows=4, cap=512, max_d=3),
    "config3": dict(k=4, H=128, bands=32, rows=4, cap=1024, max_d=2),
    "config4": dict(k=3, H=64, bands=16, rows=4, cap=1024, max_d=3),
    "config5": dict(k=0, H=0, bands=0, rows=0, cap=0, max_d=15),
}
GENERATORS = {"config1": config1, "config2": config2, "config3": config3,
              "config4": config4, "config5": config5}
DEFAULT_SEED64 = 0x5EED5EED12345678  # MinHash seed used by tests and bench


# ---------------------------------------------------------------------------
# substitution-cost tables for the weighted edit distance (an INPUT of the path;
# the paper prints no matrix: "typically based on biochemical similarity", L760)
# ---------------------------------------------------------------------------
RESIDUE_CLASSES = ("AGSTP", "ILVMC", "FWYH", "DENQ", "KR")   # small / aliphatic / aromatic / acid+amide / basic


def class_substitution_costs(same_class: int = 1, other_class: int = 2) -> np.ndarray:
    """uint8[20][20]: 0 on the diagonal, `same_class` inside a physico-chemical class,
    `other_class` across classes.  With 1 <= same <= other <= 2*same it is a metric."""
    cls = np.zeros(SIGMA, np.int32)
    for k, members in enumerate(RESIDUE_CLASSES):
        for ch in members:
            cls[ALPHABET.index(ch)] = k
    cost = np.where(cls[:, None] == cls[None, :], same_class, other_class).astype(np.uint8)
    np.fill_diagonal(cost, 0)
    return cost


def random_substitution_costs(sigma: int, lo: int, hi: int, seed: int) -> np.ndarray:
    """uint8[sigma][sigma], zero diagonal, symmetric, off-diagonal uniform in [lo, hi]."""
    rng = np.random.default_rng(seed)
    c = rng.integers(lo, hi + 1, (sigma, sigma)).astype(np.uint8)
    c = np.triu(c, 1)
    c = c + c.T
    return c.astype(np.uint8)


def split(rep: Repertoire, n_a: int):
    """Two repertoires out of one: the first n_a sequences and the rest.  The generators above end
    with a random permutation, so every family has members on both sides -- the shape of a
    cross-repertoire (multi-donor) comparison where clonotype families are shared between donors
    ("pooled CDR3 sequences from ten unrelated individuals")."""
    n_a = int(n_a)
    cut = int(rep.offsets[n_a])
    a = Repertoire(rep.seqs[:cut].copy(), rep.offsets[:n_a + 1].copy(), rep.family[:n_a].copy(),
                   rep.n_edits[:n_a].copy(), rep.name + "/A")
    b = Repertoire(rep.seqs[cut:].copy(), (rep.offsets[n_a:] - cut).copy(), rep.family[n_a:].copy(),
                   rep.n_edits[n_a:].copy(), rep.name + "/B")
    return a, b
