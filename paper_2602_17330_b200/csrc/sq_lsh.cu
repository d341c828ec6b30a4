// sq_lsh.cu -- steps a3-a5: LSH banding of MinHash signatures into capped buckets that emit
// de-duplicated candidate pairs (Alg. 1 step 2 "build MinHash index; generate
// candidate list CAND"; L273 "MinHash LSH index with block-aligned storage"; spec C3).
//
//   a3 band_key_kernel   one thread per sequence: B 64-bit band keys + the "empty signature"
//                        test; records (key, id) are written band-major.
//   a4 sq_radix_sort     stable LSD radix sort of every band's records by key (ids ascend
//                        inside a bucket because the sort is stable and ids start ascending).
//   a5 segment_kernel    bucket boundaries -> bucket id of every sorted record;
//      bucket_id_kernel  bid[id][b] = bucket id if the record is among the `cap` smallest ids
//                        of its bucket, else a unique "not kept" value;
//      emit_kernel       one thread per sorted record p: pairs (id[p], id[q]) for the kept q > p
//                        of the same bucket.  A pair is emitted only from the FIRST band in which
//                        both ends are kept in the same bucket (checked against bid[][0..b)), so
//                        the output is duplicate free without ever materialising the raw pairs.
//      final radix sort  of the unique pairs by (i, j)   (skipped with SQ_LSH_UNORDERED).
#include "sq_common.cuh"

namespace {

constexpr uint64_t kKeyInit = 0x6A09E667F3BCC908ull;
constexpr uint64_t kKeyMult = 0x9E3779B97F4A7C15ull;
constexpr uint32_t kNotKept = 0x80000000u;

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

__global__ void __launch_bounds__(256)
bucket_id_kernel(const uint32_t* __restrict__ ids, const uint32_t* __restrict__ seg,
                 const uint32_t* __restrict__ heads_pos, int64_t n2, int64_t total, int bands,
                 int cap, uint32_t* __restrict__ bid) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= total) return;
  const int b = (int)(p / n2);
  const uint32_t sg = seg[p];
  const uint32_t s = heads_pos[sg];
  const bool kept = (uint32_t)p - s < (uint32_t)cap;
  bid[(int64_t)ids[p] * bands + b] = kept ? sg : (kNotKept | (uint32_t)p);
}

constexpr int kEmitThreads = 256;
constexpr int kEmitStage = 256;   // pairs staged per warp before one global reservation

__global__ void __launch_bounds__(kEmitThreads)
emit_kernel(const uint32_t* __restrict__ ids, const uint32_t* __restrict__ seg,
            const uint32_t* __restrict__ heads_pos, const uint32_t* __restrict__ bid, int64_t n2,
            int64_t total, int bands, int cap, uint64_t* __restrict__ out,
            unsigned long long capacity, unsigned long long* __restrict__ counters) {
  __shared__ uint64_t stage[kEmitThreads / 32][kEmitStage];
  __shared__ unsigned long long raw_block;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  if (threadIdx.x == 0) raw_block = 0ull;
  __syncthreads();
  const int64_t p = (int64_t)blockIdx.x * kEmitThreads + threadIdx.x;
  uint32_t cnt = 0, u = 0;
  int b = 0;
  if (p < total) {
    b = (int)(p / n2);
    const uint32_t sg = seg[p];
    const uint32_t s = heads_pos[sg], e = heads_pos[sg + 1];
    const uint32_t ek = min(e, s + (uint32_t)cap);
    if ((uint32_t)p < ek) cnt = ek - (uint32_t)p - 1u;
    u = ids[p];
  }
  const uint32_t maxcnt = __reduce_max_sync(0xFFFFFFFFu, cnt);
  const uint32_t* urow = bid + (int64_t)u * bands;
  uint32_t wcount = 0;   // warp-uniform fill of stage[w]
  for (uint32_t off = 1; off <= maxcnt; ++off) {
    bool ok = false;
    uint32_t v = 0;
    if (off <= cnt) {
      v = ids[p + off];
      ok = true;
      const uint32_t* vrow = bid + (int64_t)v * bands;
      for (int bb = 0; bb < b; ++bb)
        if (urow[bb] == vrow[bb]) { ok = false; break; }
    }
    const uint32_t mask = __ballot_sync(0xFFFFFFFFu, ok);
    const uint32_t add = __popc(mask);
    if (wcount + add > kEmitStage) {         // flush the warp's stage
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(&counters[0], (unsigned long long)wcount);
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      for (uint32_t t = lane; t < wcount; t += 32)
        if (base + t < capacity) out[base + t] = stage[w][t];
      __syncwarp();
      wcount = 0;
    }
    if (ok) stage[w][wcount + __popc(mask & lt)] = (uint64_t)u | ((uint64_t)v << 32);
    wcount += add;
    __syncwarp();
  }
  if (wcount) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(&counters[0], (unsigned long long)wcount);
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    for (uint32_t t = lane; t < wcount; t += 32)
      if (base + t < capacity) out[base + t] = stage[w][t];
  }
  // raw (pre-dedupe) pair count, for reporting
  uint32_t wsum = __reduce_add_sync(0xFFFFFFFFu, cnt);
  if (lane == 0 && wsum) atomicAdd(&raw_block, (unsigned long long)wsum);
  __syncthreads();
  if (threadIdx.x == 0 && raw_block) atomicAdd(&counters[1], raw_block);
}

inline int bits_for(int64_t n) {   // bits needed to represent values in [0, n)
  int b = 1;
  while (b < 32 && (1ll << b) < n) ++b;
  return b;
}

}  // namespace

size_t sq_lsh_scratch_bytes(int64_t n, int bands, int64_t pair_capacity) {
  size_t nn = (size_t)(n > 0 ? n : 1), B = (size_t)(bands > 0 ? bands : 1);
  size_t cap = (size_t)(pair_capacity > 0 ? pair_capacity : 1);
  size_t rec = nn * B;
  size_t s = 0;
  s += 2 * sq_align_up(rec * 8 + 16);          // keys ping-pong
  s += 2 * sq_align_up(rec * 4 + 16);          // ids ping-pong
  s += 3 * sq_align_up((rec + 2) * 4 + 16);    // head flags, scan / seg ids, head positions
  s += sq_align_up(rec * 4 + 16);              // bid table
  s += sq_align_up((nn + 2) * 4 + 16);         // non-empty flags / ranks
  size_t sort_recs = sq_sort_scratch_bytes(n, bands);
  size_t sort_pairs = sq_sort_scratch_bytes(pair_capacity, 1);
  s += sort_recs > sort_pairs ? sort_recs : sort_pairs;
  s += sq_align_up(cap * 8 + 16);              // alternate pair buffer for the final sort
  return s + 4096;
}

extern "C" int sq_lsh_candidates(sq_ctx* c, const uint32_t* sig, int H, int bands, int rows,
                                 int bucket_cap, int flags, uint32_t* pairs_out, int64_t capacity,
                                 int64_t* n_pairs) {
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
  if (n * bands >= (1ll << 31) || capacity >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;

  sq_scratch_reset(c);
  const size_t rec = (size_t)n * bands;
  uint64_t* k0 = sq_scratch<uint64_t>(c, rec);
  uint64_t* k1 = sq_scratch<uint64_t>(c, rec);
  uint32_t* v0 = sq_scratch<uint32_t>(c, rec);
  uint32_t* v1 = sq_scratch<uint32_t>(c, rec);
  uint32_t* head = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* seg = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* heads_pos = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* bid = sq_scratch<uint32_t>(c, rec);
  uint32_t* nonempty = sq_scratch<uint32_t>(c, (size_t)n + 2);
  size_t sort_recs = sq_sort_scratch_bytes(n, bands), sort_pairs = sq_sort_scratch_bytes(capacity, 1);
  uint8_t* tmp = sq_scratch<uint8_t>(c, sort_recs > sort_pairs ? sort_recs : sort_pairs);
  uint64_t* pairs_alt = sq_scratch<uint64_t>(c, (size_t)(capacity > 0 ? capacity : 1));
  if (!k0 || !k1 || !v0 || !v1 || !head || !seg || !heads_pos || !bid || !nonempty || !tmp ||
      !pairs_alt)
    return SQ_ERR_WORKSPACE;
  cudaStream_t st = c->stream;
  unsigned long long* counters = c->dflags;      // [0] unique, [1] raw, [2] n2, [3] nseg
  SQ_CUDA(c, cudaMemsetAsync(counters, 0, 64, st));

  // a3: band keys + non-empty flags
  const unsigned gb = (unsigned)((n + 255) / 256);
  SQ_TIMED(c, SQ_K_BANDKEY, band_key_kernel<<<gb, 256, 0, st>>>(sig, n, H, bands, rows, k0, v0, nonempty));
  SQ_LAUNCH_CHECK(c);
  uint32_t* d_n2 = reinterpret_cast<uint32_t*>(counters + 2);
  uint32_t* d_nseg = reinterpret_cast<uint32_t*>(counters + 3);
  int rc = sq_exclusive_scan_u32(c, nonempty, nonempty, n, reinterpret_cast<uint32_t*>(tmp), d_n2);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters + 2, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t n2 = (int64_t)(uint32_t)c->pinned[0];
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
  // a5: buckets
  const int64_t total = n2 * bands;
  const unsigned gt = (unsigned)((total + 255) / 256);
  SQ_TIMED(c, SQ_K_SEGMENT, head_flag_kernel<<<gt, 256, 0, st>>>(kin, n2, total, head));
  SQ_LAUNCH_CHECK(c);
  rc = sq_exclusive_scan_u32(c, head, seg, total, reinterpret_cast<uint32_t*>(tmp), d_nseg);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters + 3, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const uint32_t nseg = (uint32_t)c->pinned[0];
  SQ_TIMED(c, SQ_K_SEGMENT, segment_kernel<<<(unsigned)((total + 256) / 256), 256, 0, st>>>(seg, total, nseg, heads_pos));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SEGMENT, seg_fix_kernel<<<gt, 256, 0, st>>>(seg, head, total, seg));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SEGMENT, bucket_id_kernel<<<gt, 256, 0, st>>>(vin, seg, heads_pos, n2, total, bands, bucket_cap, bid));
  SQ_LAUNCH_CHECK(c);
  // unique pairs, unordered; land them so that the final sort ends in pairs_out
  const int nb = bits_for(n);
  const int per_field = (nb + 7) / 8;
  const int npasses = (flags & SQ_LSH_UNORDERED) ? 0 : 2 * per_field;
  uint64_t* pout = reinterpret_cast<uint64_t*>(pairs_out);
  uint64_t* emit_to = (npasses & 1) ? pairs_alt : pout;
  SQ_TIMED(c, SQ_K_EMIT, emit_kernel<<<gt, kEmitThreads, 0, st>>>(
      vin, seg, heads_pos, bid, n2, total, bands, bucket_cap, emit_to,
      (unsigned long long)capacity, counters));
  SQ_LAUNCH_CHECK(c);
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters, 16, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t uniq = (int64_t)c->pinned[0];
  c->last_raw_pairs = (int64_t)c->pinned[1];
  *n_pairs = uniq;
  if (uniq > capacity) return SQ_ERR_CAPACITY;
  if (npasses > 0 && uniq > 0) {
    int shifts[8], widths[8];
    int q = 0;
    for (int f = 0; f < 2; ++f) {                 // minor field j (high word) first, then i
      const int base = f == 0 ? 32 : 0;
      for (int p = 0; p < per_field; ++p) {
        shifts[q] = base + 8 * p;
        widths[q] = (nb - 8 * p) >= 8 ? 8 : (nb - 8 * p);
        ++q;
      }
    }
    int in_alt = 0;
    uint64_t* other = (emit_to == pout) ? pairs_alt : pout;
    rc = sq_radix_sort(c, emit_to, other, nullptr, nullptr, uniq, 1, shifts, widths, npasses, tmp,
                       &in_alt);
    if (rc != SQ_OK) return rc;
    SQ_CUDA(c, cudaStreamSynchronize(st));
  }
  return SQ_OK;
}
