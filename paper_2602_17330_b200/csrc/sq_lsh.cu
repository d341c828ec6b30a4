// sq_lsh.cu -- steps a3-a5: LSH banding of MinHash signatures into capped buckets that emit
// de-duplicated candidate pairs (Alg. 1 step 2 "build MinHash index; generate
// candidate list CAND"; L273 "MinHash LSH index with block-aligned storage"; spec C3).
//
//   a3 band_key_kernel   one thread per sequence: B 64-bit band keys + the "empty signature"
//                        test; records (key, id) are written band-major.
//   a4 sq_radix_sort     stable LSD radix sort of every band's records by key (ids ascend
//                        inside a bucket because the sort is stable and ids start ascending).
//   a5 head_flag / segment kernels: bucket boundaries of the sorted records;
//      range_kernel      for every (sequence, band): the slice of the sorted id array holding
//                        the kept members AFTER it in its bucket (the `cap` smallest ids of a
//                        bucket are kept) -- an ascending run of partner ids;
//      merge_rows_kernel one warp per sequence i, lane b = band b: warp-wide B-way merge of the
//                        <= 32 ascending runs.  Equal heads advance together, so a pair found in
//                        several bands is emitted once, and row i comes out ascending in j.
//                        Pass 1 counts, a scan gives row offsets (and the total, so a too-small
//                        output is reported before anything is written), pass 2 writes (i, j).
//   The output is ascending in (i, j) by construction: no pair sort, no raw-pair buffer.
#include "sq_common.cuh"

namespace {

constexpr uint64_t kKeyInit = 0x6A09E667F3BCC908ull;
constexpr uint64_t kKeyMult = 0x9E3779B97F4A7C15ull;

__global__ void __launch_bounds__(256)
band_key_kernel(const uint32_t* __restrict__ sig, int64_t n, int H, int bands, int rows,
                uint64_t* __restrict__ keys, uint32_t* __restrict__ ids,
                uint32_t* __restrict__ nonempty) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t* row = sig + i * H;
  uint32_t all = 0xFFFFFFFFu;
  for (int j = bands * rows; j < H; ++j) all &= row[j];     // columns outside the bands
  for (int b = 0; b < bands; ++b) {
    uint64_t acc = kKeyInit;
    for (int r = 0; r < rows; ++r) {
      const uint32_t v = row[b * rows + r];
      all &= v;
      acc = (acc ^ (uint64_t)v) * kKeyMult;
      acc ^= acc >> 29;
    }
    keys[(int64_t)b * n + i] = acc;
    ids[(int64_t)b * n + i] = (uint32_t)i;
  }
  nonempty[i] = (all != SQ_EMPTY_SIG) ? 1u : 0u;
}

// drop the records of empty signatures: record of sequence i moves to slot rank[i]
__global__ void __launch_bounds__(256)
compact_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ rank,
               const uint32_t* __restrict__ sig, int H, int64_t n, int64_t n2, int bands,
               uint64_t* __restrict__ keys_out, uint32_t* __restrict__ ids_out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const bool keep = (i + 1 < n) ? (rank[i + 1] != rank[i]) : (rank[i] < (uint32_t)n2);
  if (!keep) return;
  const uint32_t r = rank[i];
  for (int b = 0; b < bands; ++b) {
    keys_out[(int64_t)b * n2 + r] = keys_in[(int64_t)b * n + i];
    ids_out[(int64_t)b * n2 + r] = (uint32_t)i;
  }
}

__global__ void __launch_bounds__(256)
head_flag_kernel(const uint64_t* __restrict__ keys, int64_t n2, int64_t total,
                 uint32_t* __restrict__ head) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= total) return;
  const bool h = (p % n2 == 0) || (keys[p] != keys[p - 1]);
  head[p] = h ? 1u : 0u;
}

// in: excl = exclusive scan of the head flags (segment id of p = excl[p] + head - 1, and a
// record is a head iff excl[p+1] != excl[p]).  Writes seg id in place and the head positions.
__global__ void __launch_bounds__(256)
segment_kernel(const uint32_t* __restrict__ excl_to_seg, int64_t total, uint32_t nseg,
               uint32_t* __restrict__ heads_pos) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p > total) return;
  if (p == total) { heads_pos[nseg] = (uint32_t)total; return; }
  const uint32_t ex = excl_to_seg[p];
  const uint32_t nx = (p + 1 < total) ? excl_to_seg[p + 1] : nseg;
  const bool is_head = nx != ex;
  if (is_head) heads_pos[ex] = (uint32_t)p;
}

__global__ void __launch_bounds__(256)
seg_fix_kernel(const uint32_t* excl, const uint32_t* __restrict__ head, int64_t total,
               uint32_t* seg) {   // in place: excl == seg
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= total) return;
  seg[p] = excl[p] + head[p] - 1u;
}

// For every sorted record p (band b, sequence id): the slice of the sorted id array holding the
// partners id can be paired with in this band -- the kept members AFTER p in p's bucket:
// range[id][b] = (p+1, min(bucket end, bucket start + cap)) if p itself is kept, else (0,0).
// Also accumulates the number of raw (pre-dedupe) pairs.
__global__ void __launch_bounds__(256)
range_kernel(const uint32_t* __restrict__ ids, const uint32_t* __restrict__ seg,
             const uint32_t* __restrict__ heads_pos, int64_t n2, int64_t total, int bands, int cap,
             uint2* __restrict__ range, unsigned long long* __restrict__ raw_counter) {
  __shared__ unsigned long long raw_block;
  if (threadIdx.x == 0) raw_block = 0ull;
  __syncthreads();
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  uint32_t cnt = 0;
  if (p < total) {
    const int b = (int)(p / n2);
    const uint32_t sg = seg[p];
    const uint32_t s = heads_pos[sg], e = heads_pos[sg + 1];
    const uint32_t ek = min(e, s + (uint32_t)cap);
    uint2 r = make_uint2(0u, 0u);
    if ((uint32_t)p + 1u < ek) { r = make_uint2((uint32_t)p + 1u, ek); cnt = ek - (uint32_t)p - 1u; }
    range[(int64_t)ids[p] * bands + b] = r;
  }
  const uint32_t wsum = __reduce_add_sync(0xFFFFFFFFu, cnt);
  if ((threadIdx.x & 31) == 0 && wsum) atomicAdd(&raw_block, (unsigned long long)wsum);
  __syncthreads();
  if (threadIdx.x == 0 && raw_block) atomicAdd(raw_counter, raw_block);
}

// Row-centric emission.  A group of G lanes (G = 16 for <= 16 bands, else 32) owns sequence i;
// lane l of the group owns band l's partner slice (an ascending run of ids, all > i).  The union
// of the runs is produced by a group-wide B-way merge: every step takes the minimum head (REDUX),
// emits it once, and advances EVERY lane whose head equals it -- duplicates across bands vanish
// and the row comes out ascending.  Each lane keeps its head plus kLook look-ahead ids in
// registers; the load issued at an advance is consumed kLook advances later, so the serial merge
// chain does not wait on global memory.
// FILL = false: count the row's unique partners.  FILL = true: write (i, j) pairs at the row's
// offset, G at a time.
constexpr int kMergeWarps = 8;
constexpr int kLook = 6;

template <int G, bool FILL>
__global__ void __launch_bounds__(kMergeWarps * 32)
merge_rows_kernel(const uint32_t* __restrict__ ids, const uint2* __restrict__ range, int64_t n,
                  int bands, uint32_t* __restrict__ row_cnt, const uint32_t* __restrict__ row_off,
                  uint2* __restrict__ pairs_out) {
  constexpr int RPW = 32 / G;                        // rows per warp
  constexpr uint32_t INF = 0xFFFFFFFFu;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int sub = lane / G, l = lane % G;
  const int64_t row = ((int64_t)blockIdx.x * kMergeWarps + w) * RPW + sub;
  const bool valid = row < n;
  uint32_t cur = 0, end = 0;                         // next id to LOAD of this lane's run
  if (valid && l < bands) {
    const uint2 r = range[row * bands + l];
    cur = r.x; end = r.y;
  }
  if (FILL && valid && row_cnt[row] == 0) end = cur;
  if (__ballot_sync(0xFFFFFFFFu, cur < end) == 0) {
    if (!FILL && valid && l == 0) row_cnt[row] = 0;
    return;
  }
  uint32_t q[kLook + 1];                             // q[0] = head, q[1..] = look-ahead
#pragma unroll
  for (int t = 0; t <= kLook; ++t) { q[t] = cur < end ? ids[cur] : INF; ++cur; }
  uint32_t c = 0, out = 0;
  const uint32_t base = (FILL && valid) ? row_off[row] : 0u;
  for (;;) {
    uint32_t m;
    if (RPW == 1) {
      m = __reduce_min_sync(0xFFFFFFFFu, q[0]);
      if (m == INF) break;
    } else {
      const uint32_t m0 = __reduce_min_sync(0xFFFFFFFFu, sub == 0 ? q[0] : INF);
      const uint32_t m1 = __reduce_min_sync(0xFFFFFFFFu, sub == 1 ? q[0] : INF);
      if ((m0 & m1) == INF) break;
      m = sub == 0 ? m0 : m1;
    }
    const bool live = m != INF;
    if (FILL && live) {
      if (l == (int)(c & (G - 1))) out = m;
      if ((c & (G - 1)) == G - 1)
        pairs_out[base + (c & ~(uint32_t)(G - 1)) + l] = make_uint2((uint32_t)row, out);
    }
    c += live ? 1u : 0u;
    if (live && q[0] == m) {
#pragma unroll
      for (int t = 0; t < kLook; ++t) q[t] = q[t + 1];
      q[kLook] = cur < end ? ids[cur] : INF;
      ++cur;
    }
  }
  if (FILL) {
    if (valid && l < (int)(c & (G - 1)))
      pairs_out[base + (c & ~(uint32_t)(G - 1)) + l] = make_uint2((uint32_t)row, out);
  } else {
    if (valid && l == 0) row_cnt[row] = c;
  }
}

template <bool FILL>
int launch_merge(sq_ctx* c, const uint32_t* ids, const uint2* range, int64_t n, int bands,
                 uint32_t* row_cnt, const uint32_t* row_off, uint2* pairs_out) {
  if (bands <= 16) {
    const int64_t rows_per_block = kMergeWarps * 2;
    const unsigned g = (unsigned)((n + rows_per_block - 1) / rows_per_block);
    SQ_TIMED(c, SQ_K_EMIT, merge_rows_kernel<16, FILL><<<g, kMergeWarps * 32, 0, c->stream>>>(
        ids, range, n, bands, row_cnt, row_off, pairs_out));
  } else {
    const unsigned g = (unsigned)((n + kMergeWarps - 1) / kMergeWarps);
    SQ_TIMED(c, SQ_K_EMIT, merge_rows_kernel<32, FILL><<<g, kMergeWarps * 32, 0, c->stream>>>(
        ids, range, n, bands, row_cnt, row_off, pairs_out));
  }
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

}  // namespace

size_t sq_lsh_scratch_bytes(int64_t n, int bands, int64_t /*pair_capacity*/) {
  size_t nn = (size_t)(n > 0 ? n : 1), B = (size_t)(bands > 0 ? bands : 1);
  size_t rec = nn * B;
  size_t s = 0;
  s += 2 * sq_align_up(rec * 8 + 16);          // keys ping-pong (the range table reuses one)
  s += 2 * sq_align_up(rec * 4 + 16);          // ids ping-pong
  s += 3 * sq_align_up((rec + 2) * 4 + 16);    // head flags, scan / seg ids, head positions
  s += 2 * sq_align_up((nn + 2) * 4 + 16);     // non-empty flags / ranks; row counts / offsets
  s += sq_sort_scratch_bytes(n, bands);
  return s + 4096;
}

extern "C" int sq_lsh_candidates(sq_ctx* c, const uint32_t* sig, int H, int bands, int rows,
                                 int bucket_cap, int flags, uint32_t* pairs_out, int64_t capacity,
                                 int64_t* n_pairs) {
  (void)flags;   // the row-centric merge always produces ascending (i, j)
  if (!c || !n_pairs) return SQ_ERR_INVALID_ARG;
  *n_pairs = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (H < 1 || bands < 1 || rows < 1 || bucket_cap < 1 || capacity < 0 ||
      (int64_t)bands * rows > H)
    return SQ_ERR_INVALID_ARG;
  if (bands > SQ_MAX_BANDS || H > SQ_MAX_H) return SQ_ERR_UNSUPPORTED;
  const int64_t n = c->n;
  c->last_raw_pairs = 0;
  if (n == 0) return SQ_OK;
  if (!sig || (capacity > 0 && !pairs_out)) return SQ_ERR_INVALID_ARG;
  if (n * bands >= (1ll << 31)) return SQ_ERR_UNSUPPORTED;

  sq_scratch_reset(c);
  const size_t rec = (size_t)n * bands;
  uint64_t* k0 = sq_scratch<uint64_t>(c, rec);
  uint64_t* k1 = sq_scratch<uint64_t>(c, rec);
  uint32_t* v0 = sq_scratch<uint32_t>(c, rec);
  uint32_t* v1 = sq_scratch<uint32_t>(c, rec);
  uint32_t* head = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* seg = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* heads_pos = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* nonempty = sq_scratch<uint32_t>(c, (size_t)n + 2);
  uint32_t* row_cnt = sq_scratch<uint32_t>(c, (size_t)n + 2);
  uint8_t* tmp = sq_scratch<uint8_t>(c, sq_sort_scratch_bytes(n, bands));
  if (!k0 || !k1 || !v0 || !v1 || !head || !seg || !heads_pos || !nonempty || !row_cnt || !tmp)
    return SQ_ERR_WORKSPACE;
  cudaStream_t st = c->stream;
  unsigned long long* counters = c->dflags;      // [0] unique, [1] raw, [2] n2, [3] nseg
  SQ_CUDA(c, cudaMemsetAsync(counters, 0, 64, st));

  // a3: band keys + non-empty flags
  const unsigned gb = (unsigned)((n + 255) / 256);
  SQ_TIMED(c, SQ_K_BANDKEY, band_key_kernel<<<gb, 256, 0, st>>>(sig, n, H, bands, rows, k0, v0, nonempty));
  SQ_LAUNCH_CHECK(c);
  int rc = sq_exclusive_scan_u32(c, nonempty, nonempty, n, reinterpret_cast<uint32_t*>(tmp),
                                 counters + 2);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters + 2, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t n2 = (int64_t)c->pinned[0];
  if (n2 < 2) return SQ_OK;                       // fewer than two usable signatures: no pairs
  uint64_t* kin = k0; uint64_t* kalt = k1; uint32_t* vin = v0; uint32_t* valt = v1;
  if (n2 != n) {
    SQ_TIMED(c, SQ_K_BANDKEY, compact_kernel<<<gb, 256, 0, st>>>(k0, nonempty, sig, H, n, n2, bands, k1, v1));
    SQ_LAUNCH_CHECK(c);
    kin = k1; kalt = k0; vin = v1; valt = v0;
  }
  // a4: stable radix sort of every band's records by the 64-bit key
  {
    int shifts[8], widths[8];
    for (int p = 0; p < 8; ++p) { shifts[p] = 8 * p; widths[p] = 8; }
    int in_alt = 0;
    rc = sq_radix_sort(c, kin, kalt, vin, valt, n2, bands, shifts, widths, 8, tmp, &in_alt);
    if (rc != SQ_OK) return rc;
    if (in_alt) { uint64_t* t = kin; kin = kalt; kalt = t; uint32_t* tv = vin; vin = valt; valt = tv; }
  }
  // a5: buckets -> per (sequence, band) partner slices
  const int64_t total = n2 * bands;
  const unsigned gt = (unsigned)((total + 255) / 256);
  SQ_TIMED(c, SQ_K_SEGMENT, head_flag_kernel<<<gt, 256, 0, st>>>(kin, n2, total, head));
  SQ_LAUNCH_CHECK(c);
  rc = sq_exclusive_scan_u32(c, head, seg, total, reinterpret_cast<uint32_t*>(tmp), counters + 3);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters + 3, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const uint32_t nseg = (uint32_t)c->pinned[0];
  SQ_TIMED(c, SQ_K_SEGMENT, segment_kernel<<<(unsigned)((total + 256) / 256), 256, 0, st>>>(seg, total, nseg, heads_pos));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SEGMENT, seg_fix_kernel<<<gt, 256, 0, st>>>(seg, head, total, seg));
  SQ_LAUNCH_CHECK(c);
  // the sorted keys are dead now: their buffer becomes the [n][bands] range table (8 B / entry)
  uint2* range = reinterpret_cast<uint2*>(kalt);
  SQ_CUDA(c, cudaMemsetAsync(range, 0, rec * 8, st));
  SQ_TIMED(c, SQ_K_SEGMENT, range_kernel<<<gt, 256, 0, st>>>(vin, seg, heads_pos, n2, total, bands,
                                                             bucket_cap, range, counters + 1));
  SQ_LAUNCH_CHECK(c);
  // a5: row-centric merge, pass 1 = count, scan, pass 2 = fill
  rc = launch_merge<false>(c, vin, range, n, bands, row_cnt, nullptr, nullptr);
  if (rc != SQ_OK) return rc;
  uint32_t* row_off = nonempty;                  // ranks are dead: reuse for the row offsets
  rc = sq_exclusive_scan_u32(c, row_cnt, row_off, n, reinterpret_cast<uint32_t*>(tmp), counters);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters, 16, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t uniq = (int64_t)c->pinned[0];
  c->last_raw_pairs = (int64_t)c->pinned[1];
  *n_pairs = uniq;
  if (uniq > capacity) return SQ_ERR_CAPACITY;
  if (uniq >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;   // 32-bit row offsets
  if (uniq > 0) {
    rc = launch_merge<true>(c, vin, range, n, bands, row_cnt, row_off,
                            reinterpret_cast<uint2*>(pairs_out));
    if (rc != SQ_OK) return rc;
    SQ_CUDA(c, cudaStreamSynchronize(st));
  }
  return SQ_OK;
}
