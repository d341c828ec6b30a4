"""Thin Python binding over libsubquad.so (C ABI: include/subquad.h).

Argument marshalling only -- every step of the path runs in the library's CUDA kernels.
torch is used for device memory, pinned host memory and the stream handle; nothing here
computes.  There is NO CPU fallback: if the library or a CUDA device is missing, importing
works but constructing `SubQuad` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsubquad.so")

SQ_OK = 0
SQ_ERR_INVALID_ARG, SQ_ERR_BAD_RESIDUE, SQ_ERR_NOT_PACKED, SQ_ERR_CAPACITY = -1, -2, -3, -4
SQ_ERR_WORKSPACE, SQ_ERR_UNSUPPORTED, SQ_ERR_CUDA = -5, -6, -7
SQ_MAX_LEN, SQ_MAX_H, SQ_MAX_BANDS = 240, 256, 32
SQ_HITS_STATIC_MAX_PAIRS = 1 << 27
OP_PACK, OP_MINHASH, OP_LSH, OP_EDIT_DISTANCE, OP_ALL_PAIRS, OP_PIPELINE_HOST, OP_GRAPH, OP_JOIN = range(8)
LSH_SORTED, LSH_UNORDERED = 0, 1
JOIN_UPPER = 1
OPT_SORT_KEY_BYTES, OPT_SCHED_MIN_BYTES, OPT_SCHED_BY_LABEL = 1, 2, 3

EXPORTS = ["sq_create", "sq_destroy", "sq_workspace_bytes", "sq_set_workspace", "sq_pack",
           "sq_minhash", "sq_lsh_candidates", "sq_lsh_prepare", "sq_lsh_emit_range", "sq_candidates_stream_host", "sq_edit_distance", "sq_edit_distance_hits", "sq_edit_distance_hits_static", "sq_edit_distance_weighted", "sq_affinity_graph", "sq_all_pairs",
           "sq_join", "sq_join_host", "sq_batch_size", "sq_set_option", "sq_pipeline_host", "sq_pipeline_host_csr", "sq_packed_n", "sq_packed_stride", "sq_last_raw_pairs",
           "sq_kernel_launches", "sq_last_cuda_error", "sq_strerror", "sq_int_peak", "sq_dp_chain_peak",
           "sq_profile_enable", "sq_profile_reset", "sq_profile_read", "sq_profile_name"]


class SqSizes(C.Structure):
    _fields_ = [("n", C.c_int64), ("total_len", C.c_int64), ("max_len", C.c_int32),
                ("H", C.c_int32), ("bands", C.c_int32), ("bucket_cap", C.c_int32),
                ("pair_capacity", C.c_int64), ("n_other", C.c_int64)]


class SubQuadError(RuntimeError):
    def __init__(self, code, msg, required=None):
        super().__init__(f"libsubquad error {code}: {msg}")
        self.code = code
        self.required = required


_lib = None


def load_library():
    """dlopen libsubquad.so and declare the prototypes.  Fails loudly when it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: run `python -m paper_2602_17330_b200.build` "
            "(or __graft_entry__.build()).  There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int
    L.sq_create.restype = i32
    L.sq_create.argtypes = [C.POINTER(vp), i32, vp]
    L.sq_destroy.restype = None
    L.sq_destroy.argtypes = [vp]
    L.sq_workspace_bytes.restype = C.c_size_t
    L.sq_workspace_bytes.argtypes = [vp, i32, C.POINTER(SqSizes)]
    L.sq_set_workspace.restype = i32
    L.sq_set_workspace.argtypes = [vp, vp, C.c_size_t]
    L.sq_pack.restype = i32
    L.sq_pack.argtypes = [vp, vp, vp, i64, i32, i32]
    L.sq_minhash.restype = i32
    L.sq_minhash.argtypes = [vp, i32, i32, C.c_uint64, vp]
    L.sq_lsh_candidates.restype = i32
    L.sq_lsh_candidates.argtypes = [vp, vp, i32, i32, i32, i32, i32, vp, i64, C.POINTER(i64)]
    L.sq_lsh_prepare.restype = i32
    L.sq_lsh_prepare.argtypes = [vp, vp, i32, i32, i32, i32, C.POINTER(i64)]
    L.sq_lsh_emit_range.restype = i32
    L.sq_lsh_emit_range.argtypes = [vp, i64, i64, i32, vp, i64, C.POINTER(i64)]
    L.sq_candidates_stream_host.restype = i32
    L.sq_candidates_stream_host.argtypes = [vp, vp, i32, i32, i32, i32, i32, i64, i64, i32, i32, vp, vp, i64,
                                            C.POINTER(i64), C.POINTER(i64)]
    L.sq_edit_distance.restype = i32
    L.sq_edit_distance.argtypes = [vp, vp, i64, i32, vp]
    for fn in (L.sq_edit_distance_hits, L.sq_edit_distance_hits_static):
        fn.restype = i32
        fn.argtypes = [vp, vp, i64, i32, vp, vp, vp, i64, C.POINTER(i64)]
    L.sq_edit_distance_weighted.restype = i32
    L.sq_edit_distance_weighted.argtypes = [vp, vp, i64, vp, i32, i32, vp]
    L.sq_affinity_graph.restype = i32
    L.sq_affinity_graph.argtypes = [vp, vp, vp, i64, i32, vp, i32, i32, vp, vp, vp, i64, C.POINTER(i64)]
    L.sq_all_pairs.restype = i32
    L.sq_all_pairs.argtypes = [vp, i32, vp, vp, i64, C.POINTER(i64)]
    L.sq_join.restype = i32
    L.sq_join.argtypes = [vp, vp, i64, i64, i32, i32, vp, vp, i64, C.POINTER(i64)]
    L.sq_join_host.restype = i32
    L.sq_join_host.argtypes = [vp, vp, i32, i32, i64, i64, vp, vp, i64, C.POINTER(i64)]
    L.sq_set_option.restype = i32
    L.sq_set_option.argtypes = [vp, i32, i64]
    L.sq_batch_size.restype = i64
    L.sq_batch_size.argtypes = [i64, C.c_uint64, C.c_uint32, C.c_uint32]
    L.sq_pipeline_host.restype = i32
    L.sq_pipeline_host.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, C.c_uint64, i32, i32, i32,
                                   i32, vp, vp, i64, C.POINTER(i64)]
    L.sq_pipeline_host_csr.restype = i32
    L.sq_pipeline_host_csr.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, C.c_uint64, i32, i32, i32,
                                       i32, vp, vp, vp, i64, C.POINTER(i64)]
    L.sq_packed_n.restype = i64
    L.sq_packed_n.argtypes = [vp]
    L.sq_packed_stride.restype = i32
    L.sq_packed_stride.argtypes = [vp]
    L.sq_last_raw_pairs.restype = i64
    L.sq_last_raw_pairs.argtypes = [vp]
    L.sq_kernel_launches.restype = i64
    L.sq_kernel_launches.argtypes = [vp]
    L.sq_last_cuda_error.restype = C.c_char_p
    L.sq_last_cuda_error.argtypes = [vp]
    L.sq_strerror.restype = C.c_char_p
    L.sq_strerror.argtypes = [i32]
    L.sq_int_peak.restype = i32
    L.sq_int_peak.argtypes = [vp, i32, i32, C.POINTER(C.c_double)]
    L.sq_dp_chain_peak.restype = i32
    L.sq_dp_chain_peak.argtypes = [vp, i32, i32, C.POINTER(C.c_double)]
    L.sq_profile_enable.restype = i32
    L.sq_profile_enable.argtypes = [vp, i32]
    L.sq_profile_reset.restype = i32
    L.sq_profile_reset.argtypes = [vp]
    L.sq_profile_read.restype = i32
    L.sq_profile_read.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(i64)]
    L.sq_profile_name.restype = C.c_char_p
    L.sq_profile_name.argtypes = [i32]
    _lib = L
    return L


def batch_size(n_seqs: int, avail_bytes: int, c: int, l_max: int) -> int:
    """PAPER.md Eq. (12) through the library (host arithmetic in C)."""
    return int(load_library().sq_batch_size(n_seqs, avail_bytes, c, l_max))


def strerror(code: int) -> str:
    return load_library().sq_strerror(code).decode()


def _dev_ptr(t, dtype, name):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    return C.c_void_p(t.data_ptr())


class SubQuad:
    """One context = one device + one stream + one workspace (a torch uint8 tensor it keeps alive).

    Methods have the names and arguments of the C entry points; tensors are torch CUDA tensors.
    """

    def __init__(self, device: int = 0, stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("SubQuad needs a CUDA device: there is no CPU fallback")
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        self._check(self.lib.sq_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream)))
        self.h = h
        self.workspace = None

    def close(self):
        if getattr(self, "h", None):
            self.lib.sq_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers ---------------------------------------------------------------------------
    def _check(self, rc, required=None):
        if rc != SQ_OK:
            msg = self.lib.sq_strerror(rc).decode()
            if rc == SQ_ERR_CUDA and getattr(self, "h", None):
                msg += ": " + self.lib.sq_last_cuda_error(self.h).decode()
            raise SubQuadError(rc, msg, required)

    def workspace_bytes(self, op, n, total_len=0, max_len=0, H=0, bands=0, bucket_cap=0,
                        pair_capacity=0, n_other=0) -> int:
        s = SqSizes(n, total_len, max_len, H, bands, bucket_cap, pair_capacity, n_other)
        return int(self.lib.sq_workspace_bytes(self.h, op, C.byref(s)))

    def set_workspace(self, nbytes: int):
        """Allocate (through torch) and hand over a workspace of `nbytes`."""
        nbytes = (int(nbytes) + 255) // 256 * 256
        if self.workspace is None or self.workspace.numel() < nbytes:
            self.workspace = None
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._check(self.lib.sq_set_workspace(self.h, C.c_void_p(self.workspace.data_ptr()),
                                              self.workspace.numel()))

    def ensure_workspace(self, nbytes: int):
        if self.workspace is None or self.workspace.numel() < nbytes:
            self.set_workspace(nbytes)

    # -- the path --------------------------------------------------------------------------
    def pack(self, seqs, offsets, alphabet=20, max_len=None):
        n = offsets.numel() - 1
        if max_len is None:
            raise ValueError("max_len (an upper bound on the sequence length) is required")
        self._check(self.lib.sq_pack(self.h, _dev_ptr(seqs, torch.uint8, "seqs"),
                                     _dev_ptr(offsets, torch.int64, "offsets"), n, alphabet,
                                     max_len))
        self.n = n

    def minhash(self, k, H, seed, sig_out=None):
        n = int(self.lib.sq_packed_n(self.h))
        if sig_out is None:
            sig_out = torch.empty((max(n, 0), H), dtype=torch.int32, device=self.device)
        self._check(self.lib.sq_minhash(self.h, k, H, C.c_uint64(seed),
                                        _dev_ptr(sig_out, torch.int32, "sig_out")))
        return sig_out

    def lsh_candidates(self, sig, bands, rows, bucket_cap, pairs_out, flags=LSH_SORTED):
        """pairs_out: int32 CUDA tensor [capacity, 2] (bit pattern = uint32).  Returns the count;
        raises SubQuadError(code=SQ_ERR_CAPACITY, required=count) when it does not fit."""
        H = sig.shape[1] if sig.dim() == 2 else 0
        cnt = C.c_int64(0)
        rc = self.lib.sq_lsh_candidates(self.h, _dev_ptr(sig, torch.int32, "sig"), H, bands, rows,
                                        bucket_cap, flags,
                                        _dev_ptr(pairs_out, torch.int32, "pairs_out"),
                                        pairs_out.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def lsh_prepare(self, sig, bands, rows, bucket_cap) -> int:
        """Band keys, bucket sort and bucket scan, kept in the workspace; returns the raw pair count."""
        H = sig.shape[1] if sig.dim() == 2 else 0
        raw = C.c_int64(0)
        self._check(self.lib.sq_lsh_prepare(self.h, _dev_ptr(sig, torch.int32, "sig"), H, bands, rows,
                                            bucket_cap, C.byref(raw)))
        return raw.value

    def lsh_emit_range(self, row_lo, row_hi, pairs_out, flags=LSH_SORTED) -> int:
        """Candidates of the rows [row_lo, row_hi) after lsh_prepare; returns their number."""
        cnt = C.c_int64(0)
        rc = self.lib.sq_lsh_emit_range(self.h, row_lo, row_hi, flags,
                                        _dev_ptr(pairs_out, torch.int32, "pairs_out"), pairs_out.shape[0],
                                        C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def candidates_stream_host(self, sig, bands, rows, bucket_cap, max_d, pairs_out_host, dist_out_host,
                               block_capacity, batch_rows=0, part=0, n_parts=1):
        """Out-of-core / sharded candidates + distances into (pinned) HOST tensors.  Returns
        (pairs of this part, raw pairs over all rows)."""
        for t in (pairs_out_host, dist_out_host):
            if t.is_cuda or not t.is_contiguous():
                raise TypeError("candidates_stream_host takes contiguous host tensors")
        H = sig.shape[1] if sig.dim() == 2 else 0
        cnt, raw = C.c_int64(0), C.c_int64(0)
        rc = self.lib.sq_candidates_stream_host(
            self.h, _dev_ptr(sig, torch.int32, "sig"), H, bands, rows, bucket_cap, max_d, batch_rows,
            block_capacity, part, n_parts, C.c_void_p(pairs_out_host.data_ptr()),
            C.c_void_p(dist_out_host.data_ptr()), dist_out_host.shape[0], C.byref(cnt), C.byref(raw))
        self._check(rc, required=cnt.value)
        return cnt.value, raw.value

    def edit_distance(self, pairs, n_pairs, max_d, dist_out=None):
        if dist_out is None:
            dist_out = torch.empty(max(n_pairs, 1), dtype=torch.int16, device=self.device)
        self._check(self.lib.sq_edit_distance(self.h, _dev_ptr(pairs, torch.int32, "pairs"),
                                              n_pairs, max_d,
                                              _dev_ptr(dist_out, torch.int16, "dist_out")))
        return dist_out

    def edit_distance_hits(self, pairs, n_pairs, max_d, dist_out, hit_pairs_out, hit_dist_out, static=False):
        """Distances + the pairs with d <= max_d compacted in input order; returns the hit count.
        static=True: the entry point whose scratch is a static device array (allocates nothing)."""
        fn = self.lib.sq_edit_distance_hits_static if static else self.lib.sq_edit_distance_hits
        cnt = C.c_int64(0)
        rc = fn(self.h, _dev_ptr(pairs, torch.int32, "pairs"), n_pairs, max_d,
                _dev_ptr(dist_out, torch.int16, "dist_out"), _dev_ptr(hit_pairs_out, torch.int32, "hit_pairs_out"),
                _dev_ptr(hit_dist_out, torch.int16, "hit_dist_out"), hit_dist_out.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def edit_distance_weighted(self, pairs, n_pairs, sub_cost, indel, max_d, dist_out=None):
        """sub_cost: uint8 CUDA tensor [alphabet, alphabet]."""
        if dist_out is None:
            dist_out = torch.empty(max(n_pairs, 1), dtype=torch.int16, device=self.device)
        self._check(self.lib.sq_edit_distance_weighted(
            self.h, _dev_ptr(pairs, torch.int32, "pairs"), n_pairs,
            _dev_ptr(sub_cost, torch.uint8, "sub_cost"), indel, max_d,
            _dev_ptr(dist_out, torch.int16, "dist_out")))
        return dist_out

    def affinity_graph(self, pairs, dist, n_pairs, max_d, sig, min_matches, row_ptr, col, weight):
        """row_ptr int64[n+1], col int32[cap], weight float32[cap] (CUDA).  Returns the edge count."""
        H = sig.shape[1] if sig is not None else 0
        cnt = C.c_int64(0)
        rc = self.lib.sq_affinity_graph(
            self.h, _dev_ptr(pairs, torch.int32, "pairs"), _dev_ptr(dist, torch.int16, "dist"), n_pairs,
            max_d, _dev_ptr(sig, torch.int32, "sig"), H, min_matches,
            _dev_ptr(row_ptr, torch.int64, "row_ptr"), _dev_ptr(col, torch.int32, "col"),
            _dev_ptr(weight, torch.float32, "weight"), col.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def all_pairs(self, max_d, pairs_out, dist_out):
        cnt = C.c_int64(0)
        rc = self.lib.sq_all_pairs(self.h, max_d, _dev_ptr(pairs_out, torch.int32, "pairs_out"),
                                   _dev_ptr(dist_out, torch.int16, "dist_out"),
                                   dist_out.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def join(self, other, max_d, pairs_out, dist_out, a_begin=0, a_end=None, flags=0):
        """Hits (i in self, j in other, d <= max_d) of rows [a_begin, a_end) into CUDA tensors."""
        if a_end is None:
            a_end = int(self.lib.sq_packed_n(self.h))
        cnt = C.c_int64(0)
        rc = self.lib.sq_join(self.h, other.h, a_begin, a_end, max_d, flags,
                              _dev_ptr(pairs_out, torch.int32, "pairs_out"),
                              _dev_ptr(dist_out, torch.int16, "dist_out"), dist_out.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def join_host(self, other, max_d, pairs_out_host, dist_out_host, block_capacity, batch_rows=0,
                  flags=0):
        """Out-of-core join into (pinned) HOST tensors, block by block; returns the hit count."""
        for t in (pairs_out_host, dist_out_host):
            if t.is_cuda or not t.is_contiguous():
                raise TypeError("join_host takes contiguous host tensors")
        cnt = C.c_int64(0)
        rc = self.lib.sq_join_host(self.h, other.h, max_d, flags, batch_rows, block_capacity,
                                   C.c_void_p(pairs_out_host.data_ptr()),
                                   C.c_void_p(dist_out_host.data_ptr()), dist_out_host.shape[0],
                                   C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def pipeline_host(self, seqs_host, offsets_host, alphabet, max_len, k, H, seed, bands, rows,
                      bucket_cap, max_d, pairs_out_host, dist_out_host):
        """Whole path from (pinned) HOST tensors; returns the number of candidate pairs."""
        for t in (seqs_host, offsets_host, pairs_out_host, dist_out_host):
            if t.is_cuda or not t.is_contiguous():
                raise TypeError("pipeline_host takes contiguous host tensors")
        n = offsets_host.numel() - 1
        cnt = C.c_int64(0)
        rc = self.lib.sq_pipeline_host(
            self.h, C.c_void_p(seqs_host.data_ptr()), C.c_void_p(offsets_host.data_ptr()), n,
            alphabet, max_len, k, H, C.c_uint64(seed), bands, rows, bucket_cap, max_d,
            C.c_void_p(pairs_out_host.data_ptr()), C.c_void_p(dist_out_host.data_ptr()),
            pairs_out_host.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def pipeline_host_csr(self, seqs_host, offsets_host, alphabet, max_len, k, H, seed, bands, rows,
                          bucket_cap, max_d, row_ptr_host, col_host, dist_host):
        """Whole path from (pinned) HOST tensors, CSR results (int64 row_ptr[n+1], int32 col,
        uint8 dist); returns the number of candidate pairs."""
        for t in (seqs_host, offsets_host, row_ptr_host, col_host, dist_host):
            if t.is_cuda or not t.is_contiguous():
                raise TypeError("pipeline_host_csr takes contiguous host tensors")
        n = offsets_host.numel() - 1
        cnt = C.c_int64(0)
        rc = self.lib.sq_pipeline_host_csr(
            self.h, C.c_void_p(seqs_host.data_ptr()), C.c_void_p(offsets_host.data_ptr()), n,
            alphabet, max_len, k, H, C.c_uint64(seed), bands, rows, bucket_cap, max_d,
            C.c_void_p(row_ptr_host.data_ptr()), C.c_void_p(col_host.data_ptr()),
            C.c_void_p(dist_host.data_ptr()), col_host.shape[0], C.byref(cnt))
        self._check(rc, required=cnt.value)
        return cnt.value

    def set_option(self, option: int, value: int):
        self._check(self.lib.sq_set_option(self.h, option, value))

    # -- introspection -----------------------------------------------------------------------
    def packed_stride(self) -> int:
        return int(self.lib.sq_packed_stride(self.h))

    def last_raw_pairs(self) -> int:
        return int(self.lib.sq_last_raw_pairs(self.h))

    def kernel_launches(self) -> int:
        return int(self.lib.sq_kernel_launches(self.h))

    def profile_enable(self, on: bool = True):
        self._check(self.lib.sq_profile_enable(self.h, 1 if on else 0))

    def profile_reset(self):
        self._check(self.lib.sq_profile_reset(self.h))

    def profile_read(self) -> dict:
        """{kernel class: (milliseconds, launches)} accumulated since the last reset."""
        out = {}
        k = 0
        while True:
            name = self.lib.sq_profile_name(k)
            if not name:
                break
            ms, ln = C.c_double(0.0), C.c_int64(0)
            self._check(self.lib.sq_profile_read(self.h, k, C.byref(ms), C.byref(ln)))
            out[name.decode()] = (ms.value, ln.value)
            k += 1
        return out

    def int_peak(self, kind: int, iters: int = 4096) -> float:
        out = C.c_double(0.0)
        self._check(self.lib.sq_int_peak(self.h, kind, iters, C.byref(out)))
        return out.value

    def dp_chain_peak(self, text_len: int = 20, iters: int = 2000) -> float:
        """(lane, text column) steps per second of the single-word DP column chain alone"""
        out = C.c_double(0.0)
        self._check(self.lib.sq_dp_chain_peak(self.h, text_len, iters, C.byref(out)))
        return out.value
