/*
 * subquad.h -- C ABI of the B200-native SubQuad candidate-pair affinity path
 * (arxiv/paper_2602_17330).  One shared library, libsubquad.so, hand-written CUDA for
 * sm_100a.  No torch types, no exceptions, no printing, NO CPU FALLBACK: every entry point
 * runs CUDA kernels or returns an error code.
 *
 * The path (Alg. 1 steps 1-2 and 7-8, L157-158 and L177-178):
 *     S  --sq_pack-->  packed residues  --sq_minhash-->  signatures
 *        --sq_lsh_candidates-->  CAND (unique pairs i<j)  --sq_edit_distance-->  d(s_i, s_j)
 * plus the exhaustive tile path sq_all_pairs (App. F.1, L733-738 Eq. 45).
 * What each step computes is fixed by SURVEY.md section 8(c) (spec C1-C3), restated in
 * DESIGN.md; the paper itself gives only the recurrence (Eq. 46) and the sketch sizes.
 *
 * Conventions
 *  - Unless a parameter says "host", every pointer is a DEVICE pointer owned by the caller
 *    (e.g. a torch tensor).  Inputs are borrowed and never modified.  The library never
 *    allocates or frees device memory: all scratch, and the packed copy of the sequences,
 *    live in the workspace the caller hands over with sq_set_workspace, which must outlive
 *    every later call on the context.
 *  - All work is enqueued on the CUDA stream given to sq_create.  Calls that return a count
 *    or an error detected on the device (sq_pack, sq_lsh_candidates, sq_all_pairs, and the
 *    *_host entry points) synchronise that stream before returning; sq_minhash and
 *    sq_edit_distance are asynchronous.
 *  - Pairs are (i, j), i < j, 0-based indices in input order, stored as uint32[n][2].
 *  - Return value: 0 = SQ_OK, negative = error (see below).  On SQ_ERR_CAPACITY the count
 *    returned through the host pointer is the REQUIRED count, so the caller can retry.
 */
#ifndef SUBQUAD_H_
#define SUBQUAD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SQ_OK                 0
#define SQ_ERR_INVALID_ARG   -1   /* null pointer, k<1, 5k>32, bands*rows>H, cap<1, ...      */
#define SQ_ERR_BAD_RESIDUE   -2   /* a residue code >= alphabet (detected by sq_pack)        */
#define SQ_ERR_NOT_PACKED    -3   /* an op that needs the packed sequences ran before sq_pack */
#define SQ_ERR_CAPACITY      -4   /* output did not fit; required count returned             */
#define SQ_ERR_WORKSPACE     -5   /* workspace missing or too small                          */
#define SQ_ERR_UNSUPPORTED   -6   /* sequence longer than max_len / SQ_MAX_LEN, H > SQ_MAX_H, ... */
#define SQ_ERR_CUDA          -7   /* a CUDA runtime call failed; see sq_last_cuda_error      */

#define SQ_MAX_LEN    240   /* longest sequence the packed layout and the DP kernels accept   */
#define SQ_MAX_H      256   /* largest signature length ({64,128,256})        */
#define SQ_MAX_BANDS   32

/* operations, for sq_workspace_bytes */
#define SQ_OP_PACK            0
#define SQ_OP_MINHASH         1
#define SQ_OP_LSH             2
#define SQ_OP_EDIT_DISTANCE   3
#define SQ_OP_ALL_PAIRS       4
#define SQ_OP_PIPELINE_HOST   5
#define SQ_OP_GRAPH           6   /* sizes->pair_capacity = number of pairs handed to the graph */
#define SQ_OP_JOIN            7   /* sizes->n = |A| (this context's set), sizes->n_other = |B|,
                                     sizes->pair_capacity = capacity (sq_join) or block_capacity
                                     (sq_join_host) */

/* flags of sq_lsh_candidates */
#define SQ_LSH_SORTED     0   /* pairs_out ascending by (i, j) (default)                      */
#define SQ_LSH_UNORDERED  1   /* caller does not need ascending j inside a row: pairs_out is
                                 ascending in i; row i's partners come grouped by the first
                                 band b in which the pair shares a bucket (b ascending), j
                                 ascending inside a group.  Deterministic; skips the row merge */

typedef struct sq_ctx sq_ctx;   /* opaque; owns only small host metadata + 2 pinned words */

/* Problem sizes for sq_workspace_bytes.  Fields an op does not use may be 0. */
typedef struct sq_sizes {
  int64_t n;             /* number of sequences                                              */
  int64_t total_len;     /* sum of lengths                                                   */
  int32_t max_len;       /* upper bound on the sequence length (<= SQ_MAX_LEN)               */
  int32_t H;             /* signature length                                                 */
  int32_t bands;         /* LSH bands                                                        */
  int32_t bucket_cap;    /* LSH bucket cap                                                   */
  int64_t pair_capacity; /* capacity of the pair output (LSH / all-pairs / pipeline)         */
  int64_t n_other;       /* SQ_OP_JOIN: number of sequences of the other set                 */
} sq_sizes;

/* Create / destroy a context bound to `device` and to `cuda_stream` (a cudaStream_t cast to
 * void*; NULL = the legacy default stream).  Fails with SQ_ERR_CUDA if there is no device. */
int  sq_create(sq_ctx** out, int device, void* cuda_stream);
void sq_destroy(sq_ctx* ctx);

/* Bytes of workspace needed so that `op` (and the packed copy made by sq_pack, which every
 * op needs) fits.  Pure host arithmetic.  Returns 0 for an unknown op. */
size_t sq_workspace_bytes(const sq_ctx* ctx, int op, const sq_sizes* sizes);

/* Hand over the workspace (device memory, 256-byte aligned).  Invalidates a previous pack. */
int  sq_set_workspace(sq_ctx* ctx, void* dev_ptr, size_t bytes);

/* a1  Pack (App. F.2 "contiguous memory blocks with proper alignment";
 * L157 "trim/pad").  seqs = uint8 residue codes, concatenated; offsets = int64[n+1], sequence
 * i is seqs[offsets[i]..offsets[i+1]); offsets[n] is the size of `seqs`.  Validates every code <
 * alphabet (<= 32, else SQ_ERR_BAD_RESIDUE), every length <= max_len (<= SQ_MAX_LEN, else
 * SQ_ERR_UNSUPPORTED) and the offsets themselves (offsets[0] >= 0, non-decreasing, none beyond
 * offsets[n]; else SQ_ERR_INVALID_ARG -- nothing outside [0, offsets[n]) is ever read); writes the internal layout into the workspace: one
 * fixed-stride slot per sequence, stride = round_up(max_len + 1, 16) bytes, residues at
 * [0, len), 0xFF padding, the length in the slot's last byte -- so a slot is read with
 * aligned 16-byte vector loads and a CDR3 (len <= 31) is exactly one 32-byte sector.
 * Also builds the length-sorted processing order used by sq_minhash.
 * n = 0 and empty sequences are legal.  Synchronises. */
int  sq_pack(sq_ctx* ctx, const uint8_t* seqs, const int64_t* offsets, int64_t n,
             int alphabet, int max_len);

/* a2  MinHash sketch (Alg. 1 step 1; sketch sizes L269; spec C2).
 * k-mer value x_p = sum_t code[p+t] * 32^(k-1-t) (needs 5k <= 32);
 * g(x): x^=x>>16; x*=0x6A09E667; x^=x>>15; x*=0xBB67AE85; x^=x>>16   (mod 2^32)
 * a_j = g(lo ^ g(2j+1)) | 1,  b_j = g(hi ^ g(2j+2))   (lo/hi = 32-bit halves of seed)
 * sig_out[i][j] = min_p ( a_j * g(x_p) + b_j mod 2^32 );  all 0xFFFFFFFF if len_i < k.
 * sig_out: uint32[n][H] row-major, 32-byte aligned (else SQ_ERR_INVALID_ARG), H a multiple of 32,
 * 32 <= H <= SQ_MAX_H.  Asynchronous. */
int  sq_minhash(sq_ctx* ctx, int k, int H, uint64_t seed, uint32_t* sig_out);

/* a3-a5  LSH banding -> capped buckets -> unique candidate pairs (Alg. 1
 * step 2, L273 "MinHash LSH index"; spec C3).  sig: uint32[n][H] (n = the packed n).
 * Band b is the tuple sig[i][b*rows .. b*rows+rows); its 64-bit key is
 *   acc = 0x6A09E667F3BCC908; for v in tuple: acc = (acc ^ v) * 0x9E3779B97F4A7C15;
 *   acc ^= acc >> 29;
 * a bucket is the set of sequences with equal (b, key); of each bucket the `bucket_cap`
 * smallest indices are kept; CAND = all i<j kept together in some bucket, as a set.
 * Sequences whose signature is all 0xFFFFFFFF take no part.  Needs bands*rows <= H,
 * 1 <= bands <= SQ_MAX_BANDS, bucket_cap >= 1.
 * pairs_out: uint32[capacity][2]; *n_pairs (host) = number of unique candidates.
 * flags: SQ_LSH_SORTED or SQ_LSH_UNORDERED.  Synchronises.  SQ_ERR_CAPACITY if
 * *n_pairs > capacity (pairs_out then holds nothing useful). */
int  sq_lsh_candidates(sq_ctx* ctx, const uint32_t* sig, int H, int bands, int rows,
                       int bucket_cap, int flags, uint32_t* pairs_out, int64_t capacity,
                       int64_t* n_pairs);

/* a3-a5 in two steps, for callers that emit the candidate list piecewise (the streamed entry point
 * below; one rank of a multi-GPU run).  sq_lsh_prepare runs band keys, bucket sort and bucket scan
 * once and keeps the sorted records, the bucket-id table and the work lists in the workspace scratch
 * (valid until the next call that resets the scratch: sq_pack, sq_lsh_prepare / sq_lsh_candidates,
 * sq_all_pairs, sq_join*, sq_affinity_graph without the schedule).  *n_raw (host, may be NULL) = pairs
 * before cross-band dedupe, over ALL rows.  sq_lsh_emit_range then writes the candidates (i, j) of
 * the rows row_lo <= i < row_hi -- the same pairs sq_lsh_candidates would list for those i, in the
 * same order -- into pairs_out; any number of calls, any ranges.  sq_lsh_candidates is
 * prepare + emit_range(0, n).  SQ_ERR_NOT_PACKED if the prepared state is gone; both synchronise;
 * SQ_ERR_CAPACITY as for sq_lsh_candidates (per call: fewer than 2^32 - 1 pairs per range). */
int  sq_lsh_prepare(sq_ctx* ctx, const uint32_t* sig, int H, int bands, int rows, int bucket_cap,
                    int64_t* n_raw);
int  sq_lsh_emit_range(sq_ctx* ctx, int64_t row_lo, int64_t row_hi, int flags, uint32_t* pairs_out,
                       int64_t capacity, int64_t* n_pairs);

/* next-3  Out-of-core and sharded candidates + distances (PAPER.md L139-143
 * Eq. 12 batch sizing, L334: 10^7 sequences at 186 GB).  The rows 0..n-1 are cut into batches of
 * `batch_rows` consecutive ids; batch b is handled by this call iff b % n_parts == part (one GPU:
 * part = 0, n_parts = 1; rank g of G: part = g, n_parts = G -- block-cyclic, because row i pairs only
 * with j > i and low ids carry more pairs).  Per batch: sq_lsh_emit_range into a device block of
 * `block_capacity` pairs, sq_edit_distance on it, both copied to the host buffers on the context's
 * second stream while the next batch is emitted.  A batch that overflows the block is halved and
 * redone, so only ONE block (twice, double-buffered) lives on the device: the list may exceed HBM and
 * 2^32 pairs (64-bit totals; each block < 2^32 - 1).  batch_rows <= 0: B of Eq. 12 with M_avail = 10 *
 * block_capacity bytes, c = 10 (bytes per candidate), l_max = 1.
 * pairs_host uint32[capacity][2], dist_host uint16[capacity] (pinned for full speed): the batches of
 * this part in ascending order, each ascending in (i, j) -- with n_parts = 1 exactly the output of
 * sq_lsh_candidates + sq_edit_distance.  *n_pairs (host) = pairs of this part; *n_raw (may be NULL) as
 * sq_lsh_prepare.  Workspace: SQ_OP_LSH with pair_capacity = block_capacity, plus 20 *
 * block_capacity + 1024 bytes.  SQ_ERR_CAPACITY (required count returned) if the part exceeds
 * `capacity`, or if one single row exceeds block_capacity.  Synchronises. */
int  sq_candidates_stream_host(sq_ctx* ctx, const uint32_t* sig, int H, int bands, int rows,
                               int bucket_cap, int max_d, int64_t batch_rows, int64_t block_capacity,
                               int part, int n_parts, uint32_t* pairs_host, uint16_t* dist_host,
                               int64_t capacity, int64_t* n_pairs, int64_t* n_raw);

/* a6  Batched exact Levenshtein distance (Eq. 46, unit costs, boundary
 * D[x][0]=x, D[0][y]=y; spec C1) by Myers/Hyyro bit-parallel DP.
 * pairs: uint32[n_pairs][2], any order, any i,j < n (i == j allowed, gives 0).
 * dist_out[p] = min(d, max_d + 1) for max_d >= 0, the exact distance for max_d < 0,
 * in input order.  Asynchronous. */
int  sq_edit_distance(sq_ctx* ctx, const uint32_t* pairs, int64_t n_pairs, int max_d,
                      uint16_t* dist_out);

/* a6 with compacted hits (north_star (d) "warp-ballot compaction of hits"; PAPER.md
 * L750-762 App. F.3): sq_edit_distance, then the pairs with d <= max_d (0 <= max_d <= 65534) are
 * compacted IN INPUT ORDER: hit_pairs_out uint32[capacity][2], hit_dist_out uint16[capacity] (hit k is
 * the k-th pair of `pairs` whose distance is within the threshold); dist_out uint16[n_pairs] as for
 * sq_edit_distance; *n_hits (host).  n_pairs < 2^32 - 1.  Scratch: one word per 2,048 pairs from the
 * free workspace (the schedule of sq_lsh_candidates survives).  Synchronises.  SQ_ERR_CAPACITY (with
 * the required *n_hits; the first `capacity` hits are written) if the hits do not fit. */
int  sq_edit_distance_hits(sq_ctx* ctx, const uint32_t* pairs, int64_t n_pairs, int max_d,
                           uint16_t* dist_out, uint32_t* hit_pairs_out, uint16_t* hit_dist_out,
                           int64_t capacity, int64_t* n_hits);

/* The same, for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): this entry point allocates NOTHING and takes no scratch from the
 * workspace -- its scratch is a file-scope __device__ array of 256 KB inside the library (every GPU
 * that loads libsubquad.so holds it until the process exits), which bounds the call to
 * n_pairs <= SQ_HITS_STATIC_MAX_PAIRS (SQ_ERR_UNSUPPORTED beyond).  Same outputs, same order, same
 * error codes as sq_edit_distance_hits.  All calls (all contexts of a device) share the array, and it
 * keeps the last call's contents: a call overwrites every word before it reads it, so consecutive
 * calls are independent, but two calls that OVERLAP on the GPU (different streams) race on it. */
#define SQ_HITS_STATIC_MAX_PAIRS (1ll << 27)
int  sq_edit_distance_hits_static(sq_ctx* ctx, const uint32_t* pairs, int64_t n_pairs, int max_d,
                                  uint16_t* dist_out, uint32_t* hit_pairs_out, uint16_t* hit_dist_out,
                                  int64_t capacity, int64_t* n_hits);

/* next-1  Weighted edit distance: Eq. 46 as printed, with
 * substitution_cost(a, b) from a table ("typically based on biochemical similarity", L760) and
 * one insertion/deletion cost; boundary D[x][0] = x*indel, D[0][y] = y*indel.
 * sub_cost: DEVICE uint8[alphabet][alphabet] row-major (alphabet = the one given to sq_pack),
 * entry [a][b] = cost of substituting residue a of sequence pairs[p][0] by residue b of sequence
 * pairs[p][1]; Eq. 46 multiplies the cost by the indicator I(a != b), so the table's diagonal is
 * never read: equal residues cost 0.  1 <= indel <= 255.
 * dist_out[p] = min(d, max_d + 1) for max_d >= 0, else min(d, 65535).  Asynchronous. */
int  sq_edit_distance_weighted(sq_ctx* ctx, const uint32_t* pairs, int64_t n_pairs,
                               const uint8_t* sub_cost, int indel, int max_d, uint16_t* dist_out);

/* next-2  Verified candidates -> sparse similarity graph G = (V, E, W) (
 * PAPER.md L71-73 Eq. 1, L185 Alg. 1 step 12; Jaccard estimate from the sketches L495-497 Eq. 30,
 * thresholded at tau = 0.7 in L269 / L638).  Edge (i, j), i < j, is kept iff dist[p] <= max_d AND
 * the signatures of i and j agree in at least `min_matches` of the H columns (the caller passes
 * min_matches = ceil(tau * H); 0 = no sketch filter, sig may then be NULL; else sig = uint32[n][H],
 * H a multiple of 32, 16-byte aligned: SQ_ERR_INVALID_ARG otherwise).
 * weight = 1 - d / max(len_i, len_j) in fp32 (1 for two empty sequences).
 * pairs/dist: as produced by sq_lsh_candidates + sq_edit_distance (first index non-decreasing).
 * Output, device: row_ptr int64[n+1], col uint32[capacity] (ascending inside a row when the pairs
 * are SQ_LSH_SORTED), weight float[capacity]: the upper-triangular CSR.  *n_edges (host).
 * Uses the workspace scratch (4 bytes per pair + 4 per sequence).  Synchronises.
 * SQ_ERR_CAPACITY if *n_edges > capacity (row_ptr is still complete). */
int  sq_affinity_graph(sq_ctx* ctx, const uint32_t* pairs, const uint16_t* dist, int64_t n_pairs,
                       int max_d, const uint32_t* sig, int H, int min_matches, int64_t* row_ptr,
                       uint32_t* col, float* weight, int64_t capacity, int64_t* n_edges);

/* a7  Exhaustive tile path over all i<j (Eq. 45, read as a self-join).
 * max_d < 0 : dist_out = uint16[n(n-1)/2], condensed row-major (0,1),(0,2)..(n-2,n-1);
 *             pairs_out ignored (may be NULL); capacity must be >= n(n-1)/2.
 * max_d >= 0: hits with d <= max_d, ascending by (i,j): pairs_out uint32[capacity][2],
 *             dist_out uint16[capacity]; *n_out (host) = number of hits.
 * Synchronises. */
int  sq_all_pairs(sq_ctx* ctx, int max_d, uint32_t* pairs_out, uint16_t* dist_out,
                  int64_t capacity, int64_t* n_out);

/* next-4  Cross-repertoire join (Eq. 45: "N and M
 * represent the sizes of the two sequence batches being compared").  A = the set packed in `a`,
 * B = the set packed in `b` (same device, and packed with the same alphabet and the same max_len
 * class so that both have one slot stride; `b` may be `a` itself).  Result: every (i, j) with
 * a_begin <= i < a_end, 0 <= j < n_b and Levenshtein d(A_i, B_j) <= max_d (max_d >= 0), ascending
 * by (i, j); with SQ_JOIN_UPPER only j > i (the self-join's upper triangle when b == a).
 * pairs_out: DEVICE uint32[capacity][2] (i indexes A, j indexes B), dist_out: DEVICE
 * uint16[capacity]; *n_out (host) = number of hits.  Runs on a's stream and scratch (size it with
 * SQ_OP_JOIN); b's pack must be complete (sq_pack synchronises).  Synchronises.
 * SQ_ERR_CAPACITY if *n_out > capacity; SQ_ERR_WORKSPACE if even one row of A against B leaves
 * more bag-filter survivors than the scratch holds (4 * capacity + 65536). */
#define SQ_JOIN_UPPER 1
int  sq_join(sq_ctx* a, const sq_ctx* b, int64_t a_begin, int64_t a_end, int max_d, int flags,
             uint32_t* pairs_out, uint16_t* dist_out, int64_t capacity, int64_t* n_out);

/* next-3  Batch size of PAPER.md L139-143 Eq. (12):
 *   B = min(n_seqs, max(32, floor(sqrt(avail_bytes / (c * l_max))))),
 * c = "per-sequence memory overhead constant" (the paper gives no value).  Integer arithmetic
 * (floor of the integer quotient, then the integer square root).  Host only; -1 on c == 0,
 * l_max == 0 or n_seqs < 0. */
int64_t sq_batch_size(int64_t n_seqs, uint64_t avail_bytes, uint32_t c, uint32_t l_max);

/* next-3  Out-of-core join: sq_join over all of A in blocks of `batch_rows` rows, every block's
 * hits copied to HOST buffers (pinned for full speed) on a second stream while the next block is
 * computed -- the device holds one block's hits (block_capacity >= 1) and survivors only, so the
 * hit list may exceed HBM.  batch_rows <= 0: B from Eq. (12) with c = 1 and avail_bytes = the
 * free scratch, rows per block = B*B / n_b (a block of rows x n_b holds the cells of Eq. 12's
 * B x B tile).  A block that overflows block_capacity or the survivor scratch is halved and
 * redone; SQ_ERR_CAPACITY / SQ_ERR_WORKSPACE only if a single row does not fit.
 * pairs_host: uint32[capacity][2], dist_host: uint16[capacity], ascending by (i, j) overall.
 * SQ_ERR_CAPACITY (with the required *n_out) if the total exceeds `capacity`.  Synchronises. */
int  sq_join_host(sq_ctx* a, const sq_ctx* b, int max_d, int flags, int64_t batch_rows,
                  int64_t block_capacity, uint32_t* pairs_host, uint16_t* dist_host,
                  int64_t capacity, int64_t* n_out);

/* The whole path from HOST buffers (the end-to-end entry point bench.py times as `e2e`):
 * copies seqs/offsets host->device, runs pack, minhash, lsh (sorted), edit distance, and
 * copies pairs + distances device->host.  All device buffers come from the workspace
 * (size it with SQ_OP_PIPELINE_HOST).  Host buffers should be pinned for full copy speed.
 * pairs_out_host: uint32[capacity][2], dist_out_host: uint16[capacity].  Synchronises. */
int  sq_pipeline_host(sq_ctx* ctx, const uint8_t* seqs_host, const int64_t* offsets_host,
                      int64_t n, int alphabet, int max_len, int k, int H, uint64_t seed,
                      int bands, int rows, int bucket_cap, int max_d,
                      uint32_t* pairs_out_host, uint16_t* dist_out_host, int64_t capacity,
                      int64_t* n_pairs);

/* The same path, results as a compressed sparse row structure: the pair list is ascending in
 * (i, j), so i is carried by row offsets and a thresholded distance fits a byte -- 5 bytes per
 * candidate cross PCIe instead of 10.  Row i's partners j > i are
 * col_host[row_ptr_host[i] .. row_ptr_host[i+1]) (ascending), dist_host[...] = min(d, max_d + 1).
 * row_ptr_host: int64[n+1], col_host: uint32[capacity], dist_host: uint8[capacity].
 * 0 <= max_d <= 254 (else SQ_ERR_UNSUPPORTED).  Workspace: SQ_OP_PIPELINE_HOST.  Synchronises. */
int  sq_pipeline_host_csr(sq_ctx* ctx, const uint8_t* seqs_host, const int64_t* offsets_host,
                          int64_t n, int alphabet, int max_len, int k, int H, uint64_t seed,
                          int bands, int rows, int bucket_cap, int max_d,
                          int64_t* row_ptr_host, uint32_t* col_host, uint8_t* dist_host,
                          int64_t capacity, int64_t* n_pairs);

/* Tuning knobs; none changes any result.
 * SQ_OPT_SORT_KEY_BYTES (1..8, default 4): the bucket sort of sq_lsh_candidates orders each band by
 * the top `value` bytes of the 64-bit band key (that many radix passes) and then puts the few
 * prefix runs that hold several full keys in order, so buckets are always the sets of equal
 * 64-bit keys the spec defines; 8 = a plain sort on the whole key.  SQ_ERR_INVALID_ARG otherwise. */
#define SQ_OPT_SORT_KEY_BYTES 1
/* SQ_OPT_SCHED_MIN_BYTES (>= 0, default 96 MiB): sq_edit_distance (and the weighted / graph steps)
 * visits the pairs sq_lsh_candidates just wrote in the family order of its internal schedule when the
 * packed sequences exceed this many bytes (they then do not fit the L2); 0 = always, so tests can
 * force that path on small inputs.  The schedule only permutes the order of the work. */
#define SQ_OPT_SCHED_MIN_BYTES 2
/* SQ_OPT_SCHED_BY_LABEL (0 / 1, default 1): order of the rows in that schedule.  1: by a family label
 * (the smallest sequence index among the row and the heads of all buckets it shares), so that the rows
 * of one clonal family are neighbours and their partners' texts stay in L2; 0: band 0's bucket order.
 * A performance hint like the schedule itself: outputs do not depend on it. */
#define SQ_OPT_SCHED_BY_LABEL 3
int  sq_set_option(sq_ctx* ctx, int option, int64_t value);

/* Introspection (host values, valid after the call they describe). */
int64_t sq_packed_n(const sq_ctx* ctx);          /* n of the current pack, -1 if none        */
int     sq_packed_stride(const sq_ctx* ctx);     /* slot stride in bytes                     */
int64_t sq_last_raw_pairs(const sq_ctx* ctx);    /* pairs before cross-band dedupe (last LSH); after a
                                                    thresholded sq_all_pairs: survivors of its bag filter */
int64_t sq_kernel_launches(const sq_ctx* ctx);   /* kernels launched by this context so far  */
const char* sq_last_cuda_error(const sq_ctx* ctx);
const char* sq_strerror(int code);

/* Built-in per-kernel timer: when enabled, every kernel launch of the context is bracketed by
 * CUDA events on the context's stream and its duration is accumulated per kernel class
 * (0 pack, 1 minhash, 2 band_key, 3 sort_hist, 4 scan, 5 sort_scatter, 6 bucket_scan, 7 emit,
 * 8 edit_distance, 9 all_pairs, 10 misc, 11 row_sort).  sq_profile_read synchronises the pending events and
 * returns the accumulated milliseconds and launch count of one class (host values). */
int  sq_profile_enable(sq_ctx* ctx, int on);
int  sq_profile_reset(sq_ctx* ctx);
int  sq_profile_read(sq_ctx* ctx, int kernel_class, double* ms, int64_t* launches);
const char* sq_profile_name(int kernel_class);   /* NULL past the last class */

/* Integer-pipe micro-benchmark (roofline denominator for the DP stage):
 * runs `iters` dependent-free instructions of `kind` per thread on a full grid and returns
 * achieved lane-operations per second in *ops_per_s (host).
 * kind: 0 LOP3, 1 IADD3, 2 SHF, 3 IMAD, 4 min.u32, 5 LOP3+IMAD mix, 6 POPC, 7 byte-wise sum of
 * absolute differences (vabsdiff4 ... add; the instruction of the bag-distance filter); 8 LOP3 / IMAD
 * alternating with three FRESH register operands each and 9 the DP column's mix (7 LOP3 : 4 IMAD, fresh
 * operands): what the register file feeds two pipes at once (kinds 0-7 reuse two loop-invariant operands).
 * Kinds 5, 8 and 9 count the instructions of both pipes. */
int  sq_int_peak(sq_ctx* ctx, int kind, int iters, double* ops_per_s);

/* The column chain of the single-word DP kernel ALONE (App. F.3, Eq. 46 as the
 * Myers/Hyyro column step): tables and texts resident in shared memory with synthetic contents, no
 * global memory, every warp slot of the device filled; `iters` chains of `text_len` (1..31) columns
 * per lane.  *lane_columns_per_s (host) = achieved (lane, text column) steps per second; times 7 it is
 * the LOP3 rate this formulation of the column reaches at best -- the ceiling bench.py quotes beside
 * the plain LOP3 peak.  Needs a workspace (one 1 KB sink).  SQ_ERR_INVALID_ARG on bad arguments. */
int  sq_dp_chain_peak(sq_ctx* ctx, int text_len, int iters, double* lane_columns_per_s);

#ifdef __cplusplus
}
#endif
#endif  /* SUBQUAD_H_ */
