"""ctypes wrapper over oracle/sq_oracle.c -- the CPU oracle of the SubQuad hot path.

TEST INFRASTRUCTURE ONLY.  May be imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs; never by paper_2602_17330_b200/.
It imports nothing from the CUDA path and takes plain numpy arrays.

Functions mirror the C file one to one; see its header for the cited passages
(Eq. 46; L157-158 Alg. 1; L495-497 Eq. 30) and the spec readings.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _declare(_lib)
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def _declare(L):
    u8p, i64p, u32p, u16p = (C.POINTER(C.c_uint8), C.POINTER(C.c_int64), C.POINTER(C.c_uint32),
                             C.POINTER(C.c_uint16))
    L.orc_num_threads.restype = C.c_int
    L.orc_set_num_threads.argtypes = [C.c_int]
    L.orc_wagner_fischer.restype = C.c_int
    L.orc_wagner_fischer.argtypes = [u8p, C.c_int, u8p, C.c_int]
    L.orc_wagner_fischer_cutoff.restype = C.c_int
    L.orc_wagner_fischer_cutoff.argtypes = [u8p, C.c_int, u8p, C.c_int, C.c_int]
    L.orc_edit_distance_pairs.restype = None
    L.orc_edit_distance_pairs.argtypes = [u8p, i64p, u32p, C.c_int64, C.c_int, u16p]
    L.orc_wagner_fischer_weighted.restype = C.c_int
    L.orc_wagner_fischer_weighted.argtypes = [u8p, C.c_int, u8p, C.c_int, u8p, C.c_int, C.c_int]
    L.orc_edit_distance_weighted_pairs.restype = None
    L.orc_edit_distance_weighted_pairs.argtypes = [u8p, i64p, u32p, C.c_int64, u8p, C.c_int, C.c_int,
                                                   C.c_int, u16p]
    L.orc_all_pairs_full.restype = None
    L.orc_all_pairs_full.argtypes = [u8p, i64p, C.c_int64, u16p]
    L.orc_all_pairs_threshold.restype = C.c_int64
    L.orc_all_pairs_threshold.argtypes = [u8p, i64p, C.c_int64, C.c_int, C.c_int, u32p, u16p,
                                          C.c_int64]
    L.orc_mix32.restype = C.c_uint32
    L.orc_mix32.argtypes = [C.c_uint32]
    L.orc_hash_params.restype = None
    L.orc_hash_params.argtypes = [C.c_uint64, C.c_int, u32p, u32p]
    L.orc_minhash.restype = None
    L.orc_minhash.argtypes = [u8p, i64p, C.c_int64, C.c_int, C.c_int, C.c_uint64, u32p]
    L.orc_kmer_jaccard.restype = None
    L.orc_kmer_jaccard.argtypes = [u8p, C.c_int, u8p, C.c_int, C.c_int, C.POINTER(C.c_int),
                                   C.POINTER(C.c_int)]
    L.orc_band_key.restype = C.c_uint64
    L.orc_band_key.argtypes = [u32p, C.c_int]
    L.orc_lsh_bruteforce.restype = C.c_int64
    L.orc_lsh_bruteforce.argtypes = [u32p, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, u32p,
                                     C.c_int64, i64p]
    L.orc_lsh_sorted.restype = C.c_int64
    L.orc_lsh_sorted.argtypes = [u32p, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, u32p,
                                 C.c_int64, i64p, i64p]
    L.orc_lsh_row.restype = C.c_int64
    L.orc_lsh_row.argtypes = [u32p, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int64,
                              u32p, C.c_int64]


def _u8(a):
    a = np.ascontiguousarray(a, dtype=np.uint8)
    return a if a.size else np.zeros(1, np.uint8)   # never hand C a NULL base pointer


def _off(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(t: int) -> None:
    lib().orc_set_num_threads(int(t))


# ---- C1 edit distance ------------------------------------------------------

def wagner_fischer(a, b) -> int:
    a, b = _u8(np.asarray(a, np.uint8)), _u8(np.asarray(b, np.uint8))
    la, lb = int(np.asarray(a).size if len(a) else 0), int(np.asarray(b).size if len(b) else 0)
    return int(lib().orc_wagner_fischer(_p(a, C.c_uint8), la, _p(b, C.c_uint8), lb))


def _wf_len(a, b, la, lb):
    return int(lib().orc_wagner_fischer(_p(a, C.c_uint8), la, _p(b, C.c_uint8), lb))


def edit_distance(a, b) -> int:
    """Levenshtein distance of two code sequences (lists / arrays / bytes)."""
    aa = np.frombuffer(a, np.uint8) if isinstance(a, (bytes, bytearray)) else np.asarray(a, np.uint8)
    bb = np.frombuffer(b, np.uint8) if isinstance(b, (bytes, bytearray)) else np.asarray(b, np.uint8)
    return _wf_len(_u8(aa), _u8(bb), int(aa.size), int(bb.size))


def edit_distance_cutoff(a, b, max_d: int) -> int:
    aa, bb = np.asarray(a, np.uint8), np.asarray(b, np.uint8)
    return int(lib().orc_wagner_fischer_cutoff(_p(_u8(aa), C.c_uint8), int(aa.size),
                                               _p(_u8(bb), C.c_uint8), int(bb.size), int(max_d)))


def edit_distance_pairs(seqs, offsets, pairs, max_d: int) -> np.ndarray:
    seqs, offsets = _u8(seqs), _off(offsets)
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros(pairs.shape[0], np.uint16)
    if pairs.shape[0]:
        lib().orc_edit_distance_pairs(_p(seqs, C.c_uint8), _p(offsets, C.c_int64),
                                      _p(pairs, C.c_uint32), pairs.shape[0], int(max_d),
                                      _p(out, C.c_uint16))
    return out


def edit_distance_weighted(a, b, sub, indel: int) -> int:
    """Weighted edit distance (Eq. 46 with a substitution table)."""
    aa, bb = np.asarray(a, np.uint8), np.asarray(b, np.uint8)
    sub = np.ascontiguousarray(sub, dtype=np.uint8)
    assert sub.ndim == 2 and sub.shape[0] == sub.shape[1]
    return int(lib().orc_wagner_fischer_weighted(_p(_u8(aa), C.c_uint8), int(aa.size),
                                                 _p(_u8(bb), C.c_uint8), int(bb.size),
                                                 _p(sub, C.c_uint8), int(sub.shape[0]), int(indel)))


def edit_distance_weighted_pairs(seqs, offsets, pairs, sub, indel: int, max_d: int) -> np.ndarray:
    seqs, offsets = _u8(seqs), _off(offsets)
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1, 2)
    sub = np.ascontiguousarray(sub, dtype=np.uint8)
    out = np.zeros(pairs.shape[0], np.uint16)
    if pairs.shape[0]:
        lib().orc_edit_distance_weighted_pairs(_p(seqs, C.c_uint8), _p(offsets, C.c_int64),
                                               _p(pairs, C.c_uint32), pairs.shape[0],
                                               _p(sub, C.c_uint8), int(sub.shape[0]), int(indel),
                                               int(max_d), _p(out, C.c_uint16))
    return out


def all_pairs_full(seqs, offsets) -> np.ndarray:
    seqs, offsets = _u8(seqs), _off(offsets)
    n = offsets.shape[0] - 1
    out = np.zeros(max(0, n * (n - 1) // 2), np.uint16)
    if out.size:
        lib().orc_all_pairs_full(_p(seqs, C.c_uint8), _p(offsets, C.c_int64), n, _p(out, C.c_uint16))
    return out


def all_pairs_threshold(seqs, offsets, max_d: int, use_cutoff: bool = False):
    seqs, offsets = _u8(seqs), _off(offsets)
    n = offsets.shape[0] - 1
    cap = 1 << 16
    while True:
        pairs = np.zeros((cap, 2), np.uint32)
        dist = np.zeros(cap, np.uint16)
        tot = int(lib().orc_all_pairs_threshold(_p(seqs, C.c_uint8), _p(offsets, C.c_int64), n,
                                                int(max_d), int(use_cutoff), _p(pairs, C.c_uint32),
                                                _p(dist, C.c_uint16), cap))
        if tot <= cap:
            return pairs[:tot].copy(), dist[:tot].copy()
        cap = tot


# ---- C2 MinHash ---------------------------------------------------------------

def mix32(x: int) -> int:
    return int(lib().orc_mix32(C.c_uint32(x & 0xFFFFFFFF)))


def hash_params(seed: int, H: int):
    a, b = np.zeros(H, np.uint32), np.zeros(H, np.uint32)
    lib().orc_hash_params(C.c_uint64(seed), H, _p(a, C.c_uint32), _p(b, C.c_uint32))
    return a, b


def minhash(seqs, offsets, k: int, H: int, seed: int) -> np.ndarray:
    seqs, offsets = _u8(seqs), _off(offsets)
    n = offsets.shape[0] - 1
    sig = np.zeros((n, H), np.uint32)
    if n:
        lib().orc_minhash(_p(seqs, C.c_uint8), _p(offsets, C.c_int64), n, int(k), int(H),
                          C.c_uint64(seed), _p(sig, C.c_uint32))
    return sig


def kmer_jaccard(s, t, k: int):
    s, t = np.asarray(s, np.uint8), np.asarray(t, np.uint8)
    num, den = C.c_int(0), C.c_int(0)
    lib().orc_kmer_jaccard(_p(_u8(s), C.c_uint8), int(s.size), _p(_u8(t), C.c_uint8), int(t.size),
                           int(k), C.byref(num), C.byref(den))
    return num.value, den.value


# ---- C3 LSH -----------------------------------------------------------------------

def band_key(tuple_vals) -> int:
    t = np.ascontiguousarray(tuple_vals, dtype=np.uint32)
    return int(lib().orc_band_key(_p(t, C.c_uint32), int(t.size)))


def lsh_bruteforce(sig, bands: int, rows: int, cap: int):
    """Tier A.  Returns (pairs[P,2] ascending, key/tuple mismatch count)."""
    sig = np.ascontiguousarray(sig, dtype=np.uint32)
    n, H = sig.shape
    capy = max(1024, 64 * n)
    mism = np.zeros(1, np.int64)
    while True:
        out = np.zeros((capy, 2), np.uint32)
        tot = int(lib().orc_lsh_bruteforce(_p(sig, C.c_uint32), n, H, bands, rows, cap,
                                           _p(out, C.c_uint32), capy, _p(mism, C.c_int64)))
        if tot <= capy:
            return out[:tot].copy(), int(mism[0])
        capy = tot


def lsh_sorted(sig, bands: int, rows: int, cap: int):
    """Tier B.  Returns (pairs[P,2] ascending, n_raw, key/tuple mismatch count)."""
    sig = np.ascontiguousarray(sig, dtype=np.uint32)
    n, H = sig.shape
    capy = max(1024, 64 * n)
    raw, mism = np.zeros(1, np.int64), np.zeros(1, np.int64)
    while True:
        out = np.zeros((capy, 2), np.uint32)
        tot = int(lib().orc_lsh_sorted(_p(sig, C.c_uint32), n, H, bands, rows, cap,
                                       _p(out, C.c_uint32), capy, _p(raw, C.c_int64),
                                       _p(mism, C.c_int64)))
        if tot <= capy:
            return out[:tot].copy(), int(raw[0]), int(mism[0])
        capy = tot


def lsh_row(sig, bands: int, rows: int, cap: int, i: int) -> np.ndarray:
    """All candidate partners of sequence i, straight from the definition (spot checks)."""
    sig = np.ascontiguousarray(sig, dtype=np.uint32)
    n, H = sig.shape
    out = np.zeros(max(16, bands * cap), np.uint32)
    tot = int(lib().orc_lsh_row(_p(sig, C.c_uint32), n, H, bands, rows, cap, int(i),
                                _p(out, C.c_uint32), out.size))
    return out[:tot].copy()


# ---- next-2: verified candidates -> sparse similarity graph (plain numpy, fp64) ----------------

def affinity_graph(pairs, dist, max_d: int, sig, min_matches: int, lengths, n: int):
    """Upper-triangular CSR of the similarity graph (Eq. 1; L185; Jaccard estimate
    from the sketches L495-497 Eq. 30 thresholded as an integer count of equal columns).
    Edge (i, j) kept iff dist <= max_d and #{c: sig[i][c] == sig[j][c]} >= min_matches;
    weight = 1 - d / max(len_i, len_j) in fp64 (1 for two empty sequences).
    Returns (row_ptr int64[n+1], col uint32[E], weight float64[E]) in the order of `pairs`."""
    pairs = np.asarray(pairs, dtype=np.uint32).reshape(-1, 2)
    dist = np.asarray(dist, dtype=np.uint16)
    keep = dist.astype(np.int64) <= max_d
    if min_matches > 0:
        sig = np.asarray(sig, dtype=np.uint32)
        matches = np.zeros(pairs.shape[0], np.int64)
        for s in range(0, pairs.shape[0], 1 << 18):               # bounded memory
            e = min(pairs.shape[0], s + (1 << 18))
            matches[s:e] = (sig[pairs[s:e, 0]] == sig[pairs[s:e, 1]]).sum(axis=1)
        keep &= matches >= min_matches
    kp = pairs[keep]
    kd = dist[keep].astype(np.float64)
    L = np.maximum(np.asarray(lengths)[kp[:, 0]], np.asarray(lengths)[kp[:, 1]]).astype(np.float64)
    weight = np.where(L > 0, 1.0 - kd / np.where(L > 0, L, 1.0), 1.0)
    row_ptr = np.zeros(n + 1, np.int64)
    np.cumsum(np.bincount(kp[:, 0], minlength=n), out=row_ptr[1:])
    return row_ptr, kp[:, 1].copy(), weight


# ---- next-3 / next-4: Eq. 12 batch size and the cross-repertoire join (plain definitions) -------

def batch_size(n_seqs: int, avail_bytes: int, c: int, l_max: int) -> int:
    """PAPER.md L139-143 Eq. (12): B = min(#S, max(32, floor(sqrt(M_avail / (c * l_max))))).
    Integer arithmetic throughout (math.isqrt of the integer quotient floor(M_avail / (c*l_max));
    floor(sqrt(x)) == isqrt(floor(x)) for real x >= 0), so no floating-point rounding decides B.
    c = the per-sequence memory overhead constant (bytes per sequence per unit of length); the
    paper leaves its value open (reading 23)."""
    import math
    if n_seqs < 0 or avail_bytes < 0 or c < 1 or l_max < 1:
        raise ValueError("batch_size: bad argument")
    return min(int(n_seqs), max(32, math.isqrt(int(avail_bytes) // (int(c) * int(l_max)))))


def join_threshold(seqs_a, offsets_a, seqs_b, offsets_b, max_d: int, upper: bool = False):
    """Cross-repertoire join (Eq. 45: "N and M represent the sizes of the two
    sequence batches being compared"): every (i, j), i in A, j in B, with Levenshtein distance
    d(A_i, B_j) <= max_d, ascending by (i, j), and the distances.  `upper` keeps j > i only (the
    self-join's upper triangle when B is A).  The definition written out: the full rectangle is
    enumerated and every distance comes from the plain Wagner-Fischer routine."""
    seqs_a, offsets_a = _u8(seqs_a), _off(offsets_a)
    seqs_b, offsets_b = _u8(seqs_b), _off(offsets_b)
    na, nb = offsets_a.shape[0] - 1, offsets_b.shape[0] - 1
    both = np.concatenate([seqs_a, seqs_b])
    off = np.concatenate([offsets_a, offsets_b[1:] + offsets_a[-1]])
    out_p, out_d = [], []
    rows_per = max(1, (1 << 22) // max(1, nb))
    jj = np.arange(nb, dtype=np.uint32)
    for i0 in range(0, na, rows_per):
        i1 = min(na, i0 + rows_per)
        ii = np.repeat(np.arange(i0, i1, dtype=np.uint32), nb)
        jt = np.tile(jj, i1 - i0)
        pr = np.stack([ii, jt + np.uint32(na)], axis=1)
        d = edit_distance_pairs(both, off, pr, -1)
        keep = d.astype(np.int64) <= max_d
        if upper:
            keep &= jt > ii
        out_p.append(np.stack([ii[keep], jt[keep]], axis=1))
        out_d.append(d[keep])
    if not out_p:
        return np.zeros((0, 2), np.uint32), np.zeros(0, np.uint16)
    return np.concatenate(out_p).astype(np.uint32), np.concatenate(out_d).astype(np.uint16)
