// sq_lsh.cu -- steps a3-a5: LSH banding of MinHash signatures into capped buckets that emit
// de-duplicated candidate pairs (Alg. 1 step 2 "build MinHash index; generate
// candidate list CAND"; L273 "MinHash LSH index with block-aligned storage"; spec C3).
//
//   a3 band_key_kernel     one thread per sequence: B 64-bit band keys + the "empty signature"
//                          test; records (key, id) are written band-major.
//   a4 sq_radix_sort       stable LSD radix sort of every band's records by key (ids ascend
//                          inside a bucket because the sort is stable and ids start ascending).
//   a5 bucket_scan_kernel  one pass over the sorted keys: every record learns its bucket
//                          [head, end) (block max-/min-scans, galloping search across tile
//                          borders), hence its rank r and whether it is KEPT (r < cap).  Writes
//                          the bucket-id table S[id][b] (= head position if kept, else a value
//                          unique to the sequence) and the work list: one UNIT per 32 kept rows
//                          of a bucket that still have partners after them.
//      emit_kernel         one warp per unit, lane = row (a kept member), sweeping the later kept
//                          members of the bucket (columns) 32 at a time through shared memory.
//                          Pair (row, column) of band b is NEW iff no earlier band b' < b has
//                          S[row][b'] == S[col][b'] -- i.e. b is the first band in which both
//                          are kept in the same bucket -- so every candidate is produced exactly
//                          once, by one compare per earlier band (broadcast LDS.128 + 4 ISETP).
//                          Pass 1 counts per (sequence, band); an exclusive scan turns the
//                          counts into output offsets (and the total, so a too-small output is
//                          reported before anything is written); pass 2 writes.
//      row_sort_kernel     SQ_LSH_SORTED only: row i's partners arrive as <= B ascending
//                          groups (one per band); one warp per row orders them with a single
//                          most-significant-digit pass over 1,024 value bins (shared-memory
//                          counters) plus a rank inside the bin.
//   No raw-pair buffer and no atomics on the data path: results are deterministic.
#include "sq_common.cuh"

namespace {

constexpr uint64_t kKeyInit = 0x6A09E667F3BCC908ull;
constexpr uint64_t kKeyMult = 0x9E3779B97F4A7C15ull;
constexpr uint32_t kFull = 0xFFFFFFFFu;

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

// rows == 4 (every BASELINE config): a band is one aligned 16-byte chunk of the signature row.
// Four bands (four independent 16-byte loads) are in flight per step.
__global__ void __launch_bounds__(256)
band_key4_kernel(const uint32_t* __restrict__ sig, int64_t n, int H, int bands,
                 uint64_t* __restrict__ keys, uint32_t* __restrict__ ids,
                 uint32_t* __restrict__ nonempty) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4* __restrict__ row = reinterpret_cast<const uint4*>(sig + i * H);
  uint32_t all = 0xFFFFFFFFu;
  for (int j = bands; j < H / 4; ++j) { const uint4 v = row[j]; all &= v.x & v.y & v.z & v.w; }
  for (int b0 = 0; b0 < bands; b0 += 4) {
    uint4 v[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) v[q] = b0 + q < bands ? row[b0 + q] : make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (b0 + q < bands) {
        all &= v[q].x & v[q].y & v[q].z & v[q].w;
        uint64_t acc = kKeyInit;
        acc = (acc ^ (uint64_t)v[q].x) * kKeyMult; acc ^= acc >> 29;
        acc = (acc ^ (uint64_t)v[q].y) * kKeyMult; acc ^= acc >> 29;
        acc = (acc ^ (uint64_t)v[q].z) * kKeyMult; acc ^= acc >> 29;
        acc = (acc ^ (uint64_t)v[q].w) * kKeyMult; acc ^= acc >> 29;
        keys[(int64_t)(b0 + q) * n + i] = acc;
        ids[(int64_t)(b0 + q) * n + i] = (uint32_t)i;
      }
    }
  }
  nonempty[i] = (all != SQ_EMPTY_SIG) ? 1u : 0u;
}

// drop the records of empty signatures: record of sequence i moves to slot rank[i]
__global__ void __launch_bounds__(256)
compact_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ rank,
               int64_t n, int64_t n2, int bands,
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

// internal row of a sequence = its position in band 0's sorted order (families end up adjacent)
__global__ void __launch_bounds__(256)
rowidx_kernel(const uint32_t* __restrict__ ids0, int64_t n2, uint32_t* __restrict__ rowidx) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n2) rowidx[ids0[p]] = (uint32_t)p;
}

__global__ void __launch_bounds__(256)
translate_kernel(const uint32_t* __restrict__ ids, int64_t total, const uint32_t* __restrict__ rowidx,
                 uint32_t* __restrict__ ids_int) {
  const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g < total) ids_int[g] = rowidx[ids[g]];
}

// partners of internal row r over all bands (offsets are band-major: off[b*n2 + r])
__global__ void __launch_bounds__(256)
row_total_kernel(const uint32_t* __restrict__ off, const uint2* __restrict__ loc, int64_t n2, int bands,
                 uint32_t* __restrict__ row_tot) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r > n2) return;
  uint32_t t = 0;
  if (r < n2) {
    t = off[r + 1] - off[r];                       // band 0: the record of row r is record r
    for (int b = 1; b < bands; ++b) t += loc[(int64_t)b * n2 + r].y;
  }
  row_tot[r] = t;                              // row_tot[n2] = 0: the scan leaves the total there
}

// partners of every EXTERNAL id (0 for sequences without a signature), to be scanned into ext_off
__global__ void __launch_bounds__(256)
ext_count_kernel(const uint32_t* __restrict__ rowidx, const uint32_t* __restrict__ row_tot, int64_t n,
                 uint32_t* __restrict__ ext_cnt) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t r = rowidx[i];
  ext_cnt[i] = r == 0xFFFFFFFFu ? 0u : row_tot[r];
}

// ---------------------------------------------------------------------------------------------
// a5.1  bucket scan
// ---- a4 fix-up: the sort orders every band by only the top `kb` bytes of the 64-bit key --------
// (half the radix passes for kb = 4).  A bucket is a run of equal FULL keys, so a run of equal
// prefixes that holds more than one full key ("mixed": ~n^2 / 2^(8 kb + 1) per band) is put in order
// afterwards: detect_mixed lists the start of every mixed prefix run (the first full-key change
// inside the run registers it), fix_mixed gives each listed run to a warp, which copies the
// records key by key -- smallest remaining full key first, records of one key in their current,
// id-ascending order (ballot compaction) -- into the dead ping-pong buffers and back.  The result
// is exactly the order of a sort on (prefix, full key), so every bucket is contiguous again.
__device__ __forceinline__ uint64_t key_prefix(uint64_t k, int pshift) { return k >> pshift; }

__global__ void __launch_bounds__(256)
detect_mixed_kernel(const uint64_t* __restrict__ keys, int64_t n2, int pshift,
                    uint32_t* __restrict__ list, unsigned long long* __restrict__ nlist) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;     // position inside the band
  if (q == 0 || q >= n2) return;
  const int64_t g = (int64_t)blockIdx.y * n2 + q;
  const uint64_t k = keys[g], kp = keys[g - 1];
  if (k == kp || key_prefix(k, pshift) != key_prefix(kp, pshift)) return;
  // a full-key change inside a prefix run: walk back to the run's start; an earlier change in the
  // same run means this one is not the first
  int64_t t = g - 1;
  const int64_t band_lo = g - q;
  while (t > band_lo) {
    const uint64_t a = keys[t - 1];
    if (key_prefix(a, pshift) != key_prefix(kp, pshift)) break;
    if (a != kp) return;
    --t;
  }
  list[atomicAdd(nlist, 1ull)] = (uint32_t)t;
}

__global__ void __launch_bounds__(256)
fix_mixed_kernel(uint64_t* __restrict__ keys, uint32_t* __restrict__ vals, uint64_t* __restrict__ kalt,
                 uint32_t* __restrict__ valt, int64_t n2, int pshift, const uint32_t* __restrict__ list,
                 const unsigned long long* __restrict__ nlist) {
  const int lane = threadIdx.x & 31;
  const int64_t nw = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int64_t nl = (int64_t)*nlist;
  for (int64_t e = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; e < nl; e += nw) {
    const int64_t s = list[e];
    const int64_t band_hi = (s / n2 + 1) * n2;
    const uint64_t pre = key_prefix(keys[s], pshift);
    // end of the prefix run
    int64_t end = s + 1;
    for (;;) {
      const int64_t t = end + lane;
      const bool same = t < band_hi && key_prefix(keys[t], pshift) == pre;
      const uint32_t m = __ballot_sync(0xFFFFFFFFu, same);
      if (m == 0xFFFFFFFFu) { end += 32; continue; }
      end += __ffs(~m) - 1;
      break;
    }
    // smallest remaining full key first
    int64_t out = s;
    bool first = true;
    uint64_t prev = 0;
    for (;;) {
      uint64_t best = ~0ull;
      bool any = false;
      for (int64_t t = s + lane; t < end; t += 32) {
        const uint64_t k = keys[t];
        if ((first || k > prev) && (!any || k < best)) { best = k; any = true; }
      }
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        const uint64_t ob = __shfl_xor_sync(0xFFFFFFFFu, best, d);
        const bool oa = __shfl_xor_sync(0xFFFFFFFFu, (int)any, d) != 0;
        if (oa && (!any || ob < best)) { best = ob; any = true; }
      }
      if (!any) break;
      for (int64_t t0 = s; t0 < end; t0 += 32) {
        const int64_t t = t0 + lane;
        const bool hit = t < end && keys[t] == best;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, hit);
        if (hit) {
          const int64_t o = out + __popc(m & ((1u << lane) - 1u));
          kalt[o] = best;
          valt[o] = vals[t];
        }
        out += __popc(m);
      }
      prev = best;
      first = false;
    }
    __syncwarp();
    for (int64_t t = s + lane; t < end; t += 32) { keys[t] = kalt[t]; vals[t] = valt[t]; }
    __syncwarp();
  }
}

// ---------------------------------------------------------------------------------------------
constexpr int kBsThreads = 256;
constexpr int kBsItems = 4;
constexpr int kBsTile = kBsThreads * kBsItems;

// first position of the run of `key` that contains position `at` (keys sorted, k[at] == key)
__device__ int64_t run_begin(const uint64_t* __restrict__ k, int64_t at, uint64_t key) {
  int64_t hi = at, lo = -1, step = 1;
  for (;;) {
    const int64_t p = hi - step;
    if (p < 0) break;
    if (k[p] == key) { hi = p; step <<= 1; } else { lo = p; break; }
  }
  while (hi - lo > 1) {
    const int64_t mid = lo + (hi - lo) / 2;
    if (k[mid] == key) hi = mid; else lo = mid;
  }
  return hi;
}

// one past the last position of the run of `key` that contains position `at`
__device__ int64_t run_end(const uint64_t* __restrict__ k, int64_t at, uint64_t key, int64_t n) {
  int64_t lo = at, hi = n, step = 1;
  for (;;) {
    const int64_t p = lo + step;
    if (p >= n) break;
    if (k[p] == key) { lo = p; step <<= 1; } else { hi = p; break; }
  }
  while (hi - lo > 1) {
    const int64_t mid = lo + (hi - lo) / 2;
    if (k[mid] == key) lo = mid; else hi = mid;
  }
  return hi;
}

// every S entry starts as the row's own sentinel (coalesced); bucket_scan_kernel then scatters bucket
// ids only into the entries of rows that share a bucket with someone
__global__ void __launch_bounds__(256)
s_prefill_kernel(uint32_t* __restrict__ S, int64_t n2, int SW) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;     // one uint4 of S
  const int per_row = SW >> 2;
  if (t >= n2 * per_row) return;
  const uint32_t v = 0x80000000u | (uint32_t)(t / per_row);
  reinterpret_cast<uint4*>(S)[t] = make_uint4(v, v, v, v);
}

// S layout: [n][SW] uint32, SW = 4 * BW (rows are 16-byte aligned for vector loads).
// units: (global sorted position of the unit's first row, kept members from there to the end
// of the bucket); band 0's units go to their own list units0 (they need no compares).
// ubase[u] = index of unit u's first 32-word tile in the mask cache (bands >= 1).
// counters: [1] raw pairs, [4] units of bands >= 1, [5] units of band 0, [7] mask tiles, [8] small units.
// A bucket of bands >= 1 with at most kSmallMax kept members is ONE small unit (list units_s): it is
// handled by a single thread (small_units_kernel), not by a warp, and has no mask tiles -- three
// quarters of all units are of this kind and hold under 1 % of the pairs.
constexpr int kSmallMax = 8;

__global__ void __launch_bounds__(kBsThreads)
bucket_scan_kernel(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ ids, int64_t n2,
                   int cap, int SW, uint32_t* __restrict__ S, uint2* __restrict__ units,
                   uint2* __restrict__ units0, uint2* __restrict__ units_s, uint32_t* __restrict__ ubase,
                   unsigned long long* __restrict__ counters) {
  __shared__ int sh_w[kBsThreads / 32];
  __shared__ int sh_carry_head, sh_carry_end;
  __shared__ unsigned long long sh_raw;
  __shared__ uint32_t sh_unit_base, sh_unit_cnt, sh_tile_cnt, sh_small_base, sh_small_cnt;
  __shared__ unsigned long long sh_tile_base;
  const int band = blockIdx.y;
  const uint64_t* __restrict__ k = keys + (int64_t)band * n2;
  const uint32_t* __restrict__ idb = ids + (int64_t)band * n2;
  const int64_t tile0 = (int64_t)blockIdx.x * kBsTile;
  const int64_t tile_end = min(n2, tile0 + kBsTile);             // exclusive
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t p0 = tile0 + (int64_t)threadIdx.x * kBsItems;
  if (threadIdx.x == 0) { sh_raw = 0ull; sh_unit_cnt = 0u; sh_tile_cnt = 0u; sh_small_cnt = 0u; }

  uint64_t kk[kBsItems];
  bool valid[kBsItems], head[kBsItems], tail[kBsItems];
  uint64_t prev = 0, next = 0;
  bool has_prev = p0 > 0 && p0 < n2, has_next = false;
  if (has_prev) prev = k[p0 - 1];
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) {
    valid[t] = p0 + t < n2;
    kk[t] = valid[t] ? k[p0 + t] : 0ull;
  }
  if (p0 + kBsItems < n2) { has_next = true; next = k[p0 + kBsItems]; }
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) {
    const bool hp = t == 0 ? (!has_prev || kk[0] != prev) : (kk[t] != kk[t - 1]);
    bool tl;
    if (t == kBsItems - 1) tl = !has_next || kk[t] != next;
    else tl = !valid[t + 1] || kk[t] != kk[t + 1];
    head[t] = valid[t] && hp;
    tail[t] = valid[t] && tl;
  }
  // the two tile-border searches (done by one thread each, overlapped with the scans below)
  if (threadIdx.x == 0)
    sh_carry_head = head[0] ? (int)tile0 : (int)run_begin(k, tile0, kk[0]);
#pragma unroll
  for (int t = 0; t < kBsItems; ++t)
    if (p0 + t == tile_end - 1)                                  // thread owning the last record
      sh_carry_end = tail[t] ? (int)tile_end : (int)run_end(k, tile_end - 1, kk[t], n2);
  // forward max-scan of head positions
  int hpos[kBsItems];
  int run = -1;
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) { if (head[t]) run = (int)(p0 + t); hpos[t] = run; }
  int inc = run;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int o = __shfl_up_sync(kFull, inc, d);
    if (lane >= d) inc = max(inc, o);
  }
  if (lane == 31) sh_w[w] = inc;
  __syncthreads();
  int ex = __shfl_up_sync(kFull, inc, 1);
  if (lane == 0) ex = -1;
  for (int q = 0; q < w; ++q) ex = max(ex, sh_w[q]);
  if (ex < 0) ex = sh_carry_head;
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) if (hpos[t] < 0) hpos[t] = ex;
  __syncthreads();
  // backward min-scan of end positions
  int epos[kBsItems];
  constexpr int kInf = 0x7FFFFFFF;
  run = kInf;
#pragma unroll
  for (int t = kBsItems - 1; t >= 0; --t) { if (tail[t]) run = (int)(p0 + t + 1); epos[t] = run; }
  inc = run;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int o = __shfl_down_sync(kFull, inc, d);
    if (lane + d < 32) inc = min(inc, o);
  }
  if (lane == 0) sh_w[w] = inc;
  __syncthreads();
  int ee = __shfl_down_sync(kFull, inc, 1);
  if (lane == 31) ee = kInf;
  for (int q = w + 1; q < kBsThreads / 32; ++q) ee = min(ee, sh_w[q]);
  if (ee == kInf) ee = sh_carry_end;
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) if (epos[t] == kInf) epos[t] = ee;

  // per record: rank, kept, S entry, unit, raw pairs
  unsigned long long raw = 0;
  uint32_t nunit = 0;
  uint2 unit[kBsItems];
  bool has_unit[kBsItems], is_small[kBsItems];
  uint32_t nsmall = 0;
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) {
    has_unit[t] = false; is_small[t] = false;
    if (!valid[t]) continue;
    const uint32_t id = idb[p0 + t];
    const int r = (int)(p0 + t) - hpos[t];
    const int size = epos[t] - hpos[t];
    const int m = min(size, cap);
    const bool kept = r < m;
    // (rows outside any shared bucket keep the sentinel 0x80000000 | row written by s_prefill_kernel:
    // it equals no bucket id and no other row's sentinel)
    if (kept && m >= 2) S[(int64_t)id * SW + band] = (uint32_t)hpos[t];
    if (kept) {
      raw += (unsigned long long)(m - 1 - r);
      if ((r & 31) == 0 && r + 1 < m) {
        unit[t] = make_uint2((uint32_t)((int64_t)band * n2 + p0 + t), (uint32_t)(m - r));
        if (band != 0 && m <= kSmallMax) { is_small[t] = true; ++nsmall; }      // (then r == 0)
        else { has_unit[t] = true; ++nunit; }
      }
    }
  }
  // append the units (order across blocks is irrelevant: output positions never depend on it)
  uint32_t my = 0, my_tiles = 0, ntiles = 0;
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) if (has_unit[t]) ntiles += (unit[t].y + 31u) >> 5;
  if (nunit) { my = atomicAdd(&sh_unit_cnt, nunit); my_tiles = atomicAdd(&sh_tile_cnt, ntiles); }
  uint32_t my_small = 0;
  if (nsmall) my_small = atomicAdd(&sh_small_cnt, nsmall);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) raw += __shfl_xor_sync(kFull, raw, d);
  if (lane == 0 && raw) atomicAdd(&sh_raw, raw);
  __syncthreads();
  if (threadIdx.x == 0) {
    if (sh_unit_cnt)
      sh_unit_base = (uint32_t)atomicAdd(counters + (band == 0 ? 5 : 4), (unsigned long long)sh_unit_cnt);
    if (sh_raw) atomicAdd(counters + 1, sh_raw);
    if (band != 0 && sh_tile_cnt) sh_tile_base = atomicAdd(counters + 7, (unsigned long long)sh_tile_cnt);
    if (sh_small_cnt) sh_small_base = (uint32_t)atomicAdd(counters + 8, (unsigned long long)sh_small_cnt);
  }
  __syncthreads();
  uint2* __restrict__ ulist = band == 0 ? units0 : units;
  uint32_t q = sh_unit_base + my;
  unsigned long long tb = sh_tile_base + my_tiles;   // (band >= 1) first tile of the unit's masks
#pragma unroll
  for (int t = 0; t < kBsItems; ++t) {
    if (has_unit[t]) {
      if (band != 0) { ubase[q] = (uint32_t)tb; tb += (unit[t].y + 31u) >> 5; }
      ulist[q++] = unit[t];
    }
  }
  uint32_t qs = sh_small_base + my_small;
#pragma unroll
  for (int t = 0; t < kBsItems; ++t)
    if (is_small[t]) units_s[qs++] = unit[t];
}

// ---------------------------------------------------------------------------------------------
// a5.2  emission: lane = row, columns swept through shared memory
// ---------------------------------------------------------------------------------------------
constexpr int kEmWarps = 4;
enum { EM_COUNT = 0, EM_FILL_J = 1 };

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// Band 0: every pair of kept members is new.  One warp per unit.
// `active` (may be nullptr = all): the units that hold a row of the id range [row_lo, row_hi) the
// call emits (sq_lsh_emit_range); rows outside the range emit nothing.
template <int MODE>
__global__ void __launch_bounds__(kEmWarps * 32)
emit_band0_kernel(const uint2* __restrict__ units, const uint32_t* __restrict__ active, uint32_t nunits,
                  const uint32_t* __restrict__ ids, int bands, uint32_t* __restrict__ cnt_off,
                  uint32_t* __restrict__ outJ, uint32_t row_lo, uint32_t row_hi) {
  const int lane = threadIdx.x & 31;
  const uint32_t ua = blockIdx.x * kEmWarps + (threadIdx.x >> 5);
  if (ua >= nunits) return;
  const uint2 unit = units[active ? active[ua] : ua];
  const uint32_t mrem = unit.y;
  const uint32_t* __restrict__ idp = ids + unit.x;
  const uint32_t nrows = min(32u, mrem - 1u);
  bool rowok = (uint32_t)lane < nrows;
  if (rowok) { const uint32_t me = idp[lane]; rowok = me >= row_lo && me < row_hi; }
  const uint32_t okm = __ballot_sync(kFull, rowok);
  // internal row of a band-0 record = its sorted position: the rows of a unit are consecutive
  const int64_t myrow = (int64_t)unit.x + lane;
  if (MODE == EM_COUNT) {
    if (rowok) cnt_off[myrow] = mrem - 1u - (uint32_t)lane;       // band 0: index 0*n2 + row
    return;
  }
  const uint32_t off = rowok ? cnt_off[myrow] : 0u;
  for (uint32_t l = 0; l < nrows; ++l) {     // coalesced: the warp writes row l's partners
    if (!((okm >> l) & 1u)) continue;
    const uint32_t o = __shfl_sync(kFull, off, l);
    for (uint32_t cc = l + 1 + lane; cc < mrem; cc += 32) outJ[o + cc - l - 1] = idp[cc];
  }
}

// One column tile against the warp's 32 rows: NCH chunks of 4 earlier bands are compared.
template <int BW, int NCH, int MODE>
__device__ __forceinline__ void sweep_tile(const uint32_t* __restrict__ sm,
                                           const uint32_t* __restrict__ idt, const uint4 (&R)[BW],
                                           uint32_t cbeg, uint32_t ncol, uint32_t c0, uint32_t lane,
                                           bool rowok, uint32_t myid, uint32_t& acc,
                                           uint32_t& tmask, uint32_t* __restrict__ outJ) {
  constexpr int RS = 4 * BW + 4;
  if constexpr (NCH <= BW && MODE == EM_COUNT) {
    // Count pass.  Per column and chunk of four earlier bands: one broadcast LDS.128, four chained
    // ISETP.NE.AND and one SEL that keeps the column's bit while every band differs -- written as PTX
    // so that the predicate chain survives the compiler.  The row's validity and the triangle of the
    // unit's first tile (row l pairs with columns > l only) are applied ONCE per tile.
    auto keep = [&](uint32_t c, uint32_t bit) -> uint32_t {       // bit if (row, column c) is new, else 0
#pragma unroll
      for (int ch = 0; ch < NCH; ++ch) {
        const uint4 v = *reinterpret_cast<const uint4*>(sm + c * RS + 4 * ch);   // broadcast
        asm("{\n\t.reg .pred p;\n\t"
            "setp.ne.u32 p, %1, %5;\n\t"
            "setp.ne.and.u32 p, %2, %6, p;\n\t"
            "setp.ne.and.u32 p, %3, %7, p;\n\t"
            "setp.ne.and.u32 p, %4, %8, p;\n\t"
            "selp.u32 %0, %0, 0, p;\n\t}"
            : "+r"(bit)
            : "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "r"(R[ch].x), "r"(R[ch].y), "r"(R[ch].z), "r"(R[ch].w));
      }
      return bit;
    };
    uint32_t tm = 0u, c = 0u;
#pragma unroll 1
    for (; c + 4 <= ncol; c += 4) {
      const uint32_t m4 = keep(c, 1u) | keep(c + 1, 2u) | keep(c + 2, 4u) | keep(c + 3, 8u);
      tm |= m4 << c;
    }
    for (; c < ncol; ++c) tm |= keep(c, 1u) << c;
    if (c0 == 0) tm &= lane < 31u ? (0xFFFFFFFEu << lane) : 0u;      // columns c > lane
    tmask = rowok ? tm : 0u;
    (void)cbeg;
  } else if constexpr (NCH <= BW) {
#pragma unroll 4
    for (uint32_t c = cbeg; c < ncol; ++c) {
      bool dup = false;
#pragma unroll
      for (int ch = 0; ch < NCH; ++ch) {
        const uint4 v = *reinterpret_cast<const uint4*>(sm + c * RS + 4 * ch);   // broadcast
        dup |= (v.x == R[ch].x) | (v.y == R[ch].y) | (v.z == R[ch].z) | (v.w == R[ch].w);
      }
      const bool isnew = !dup && rowok && (c0 + c > lane);
      if (MODE == EM_COUNT) {
        tmask |= isnew ? (1u << c) : 0u;
      } else if (isnew) {
        outJ[acc] = idt[c];
        ++acc;
      }
    }
  }
}

struct EmDesc { uint32_t u, uid, g0, mrem, c0; int b; bool ok; };   // u = place in the (active) list, uid = unit

// Bands >= 1.  Persistent warps stride over the unit list; the stream of (unit, column tile)
// items is software-pipelined: ids two tiles ahead (registers), S rows one tile ahead
// (cp.async into the other shared-memory buffer), compares on the current tile.
// BW = 16-byte chunks per S row (S row width SW = 4*BW >= bands).
// ids = external sequence ids of the sorted records (the values that are emitted); ids_int =
// their internal rows (position in band 0's sorted order), which index S and the counts.
// Counts / offsets are indexed by SORTED RECORD g (band-major, bucket order): the 32 rows of a
// unit are 32 consecutive records, so a warp's counts are one coalesced store and its groups in
// the partner scratch are adjacent -- the appends of a unit land in one contiguous piece.  The
// fill pass leaves, for every non-empty group, loc[band][row] = (start, length) for the row kernel.
// MODE EM_COUNT:  cnt[g] = number of NEW partners of the row at sorted record g.
// MODE EM_FILL_J: outJ[off[g] + t] = external id of its t-th new partner.
template <int BW, int MODE>
__global__ void __launch_bounds__(kEmWarps * 32)
emit_kernel(const uint2* __restrict__ units, const uint32_t* __restrict__ active, uint32_t nunits,
            const uint32_t* __restrict__ ids, const uint32_t* __restrict__ ids_int, uint32_t n2, int bands,
            const uint32_t* __restrict__ S, uint32_t* __restrict__ cnt_off,
            uint32_t* __restrict__ outJ, const uint32_t* __restrict__ ubase,
            uint32_t* __restrict__ masks, uint2* __restrict__ loc, uint32_t row_lo, uint32_t row_hi) {
  constexpr int SW = 4 * BW;
  constexpr int RS = SW + 4;                 // shared row stride in words (16-byte aligned)
  constexpr int RPR = 32 / BW;               // S rows fetched per load round
  __shared__ __align__(16) uint32_t Sm[kEmWarps][2][32 * RS];
  __shared__ uint32_t idsm[kEmWarps][2][32];
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t nw = gridDim.x * kEmWarps;
  const uint32_t wg = blockIdx.x * kEmWarps + w;
  if (wg >= nunits) return;
  auto uidx = [&](uint32_t k) -> uint32_t { return active ? active[k] : k; };
  uint32_t uid_pref = uidx(wg);              // always the next unit this warp will open
  uint2 unit_pref = units[uid_pref];

  auto next_desc = [&](EmDesc d) -> EmDesc {
    if (d.ok && d.c0 + 32 < d.mrem) { d.c0 += 32; return d; }
    EmDesc r;
    r.u = d.u + nw;
    r.ok = d.ok && r.u < nunits;
    r.g0 = unit_pref.x; r.mrem = unit_pref.y; r.c0 = 0; r.uid = uid_pref;
    r.b = (int)(r.g0 / n2);
    if (r.ok && r.u + nw < nunits) { uid_pref = uidx(r.u + nw); unit_pref = units[uid_pref]; }
    return r;
  };
  auto load_ids = [&](const EmDesc& d) -> uint32_t {          // internal rows of a column tile
    return (d.ok && d.c0 + lane < d.mrem) ? ids_int[(int64_t)d.g0 + d.c0 + lane] : 0u;
  };
  auto load_ext = [&](const EmDesc& d) -> uint32_t {          // external ids (fill mode only)
    return (MODE != EM_COUNT && d.ok && d.c0 + lane < d.mrem) ? ids[(int64_t)d.g0 + d.c0 + lane] : 0u;
  };
  auto issue_rows = [&](const EmDesc& d, uint32_t idc, uint32_t* sm) {
    const uint32_t ncol = min(32u, d.mrem - d.c0);
    const int nch = (d.b + 3) >> 2;
#pragma unroll
    for (int it = 0; it < BW; ++it) {
      const uint32_t rr = it * RPR + lane / BW;
      const int ch = lane % BW;
      const uint32_t rid = __shfl_sync(kFull, idc, rr);
      if (ch < nch && rr < ncol) cp_async16(sm + rr * RS + 4 * ch, S + (int64_t)rid * SW + 4 * ch);
    }
  };

  EmDesc dc;                                  // current tile
  dc.u = wg - nw; dc.uid = 0; dc.ok = true; dc.mrem = 0; dc.c0 = 0; dc.g0 = 0; dc.b = 0;
  dc = next_desc(dc);
  uint32_t idc_c = load_ids(dc), idx_c = load_ext(dc);
  EmDesc dn = next_desc(dc);                  // next tile
  uint32_t idc_n = load_ids(dn), idx_n = load_ext(dn);
  issue_rows(dc, idc_c, Sm[w][0]);
  cp_async_commit();

  uint4 R[BW];
  uint32_t acc = 0, myid = 0, ub = 0;
  bool rowok = false;
  int k = 0;
  while (dc.ok) {
    if (dn.ok) issue_rows(dn, idc_n, Sm[w][(k + 1) & 1]);
    cp_async_commit();
    const EmDesc d2 = next_desc(dn);
    const uint32_t id2 = load_ids(d2), ix2 = load_ext(d2);
    cp_async_wait<1>();
    __syncwarp();
    const uint32_t* sm = Sm[w][k & 1];
    const int b = dc.b;
    if (dc.c0 == 0) {                         // a unit starts: its rows are the first 32 columns
      myid = idc_c;
      rowok = lane < min(32u, dc.mrem - 1u);
      if (rowok) { const uint32_t me = ids[(int64_t)dc.g0 + lane]; rowok = me >= row_lo && me < row_hi; }
      acc = 0;
      if (MODE != EM_COUNT && rowok) {
        acc = cnt_off[(int64_t)dc.g0 + lane];
        const uint32_t nxt = cnt_off[(int64_t)dc.g0 + lane + 1];
        if (nxt > acc) loc[(int64_t)b * n2 + myid] = make_uint2(acc, nxt - acc);
      }
      if (MODE == EM_COUNT && masks) ub = ubase[dc.uid];
#pragma unroll
      for (int ch = 0; ch < BW; ++ch) {
        if (4 * ch < b) {
          uint4 v = *reinterpret_cast<const uint4*>(sm + lane * RS + 4 * ch);
          if (4 * ch + 1 >= b) v.y = kFull;   // bands >= b never match (no S value is 0xFFFFFFFF)
          if (4 * ch + 2 >= b) v.z = kFull;
          if (4 * ch + 3 >= b) v.w = kFull;
          R[ch] = v;
        }
      }
    }
    if (MODE != EM_COUNT) { idsm[w][k & 1][lane] = idx_c; __syncwarp(); }
    const uint32_t ncol = min(32u, dc.mrem - dc.c0);
    const uint32_t cbeg = dc.c0 == 0 ? 1u : 0u;
    const uint32_t* idt = idsm[w][k & 1];
    uint32_t tmask = 0;                       // EM_COUNT: bit c = pair (my row, column c) is new
    switch ((b + 3) >> 2) {
      case 1: sweep_tile<BW, 1, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      case 2: sweep_tile<BW, 2, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      case 3: sweep_tile<BW, 3, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      case 4: sweep_tile<BW, 4, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      case 5: sweep_tile<BW, 5, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      case 6: sweep_tile<BW, 6, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      case 7: sweep_tile<BW, 7, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
      default: sweep_tile<BW, 8, MODE>(sm, idt, R, cbeg, ncol, dc.c0, lane, rowok, myid, acc, tmask, outJ); break;
    }
    if (MODE == EM_COUNT) {
      acc += __popc(tmask);
      if (masks) masks[((size_t)ub + (dc.c0 >> 5)) * 32 + lane] = tmask;   // kept for the fill pass
      if (rowok && dc.c0 + 32 >= dc.mrem) cnt_off[(int64_t)dc.g0 + lane] = acc;
    }
    __syncwarp();
    dc = dn; idc_c = idc_n; idx_c = idx_n; dn = d2; idc_n = id2; idx_n = ix2; ++k;
  }
  cp_async_wait<0>();
}

// Pass 2 when the count pass could keep its per-tile masks: no S rows, no compares.  One
// (persistent) warp per unit walks the unit's tiles; lane = row holds the mask of its new columns
// of the tile and the id of column `lane`; every round each lane with a bit left takes its next
// column's id from the owning lane (SHFL) and appends it to its row's group.  A unit is a chain
// of three dependent loads (descriptor -> ids + first mask -> output offset); the warp keeps the
// chains of its next kFillDepth units in flight while it works on the current one.
constexpr int kFillDepth = 12;

__global__ void __launch_bounds__(kEmWarps * 32)
emit_fill_masks_kernel(const uint2* __restrict__ units, const uint32_t* __restrict__ active, uint32_t nunits,
                       const uint32_t* __restrict__ ubase, const uint32_t* __restrict__ masks,
                       const uint32_t* __restrict__ ids, const uint32_t* __restrict__ ids_int,
                       uint32_t n2, int bands, const uint32_t* __restrict__ cnt_off,
                       uint32_t* __restrict__ outJ, uint2* __restrict__ loc) {
  __shared__ uint32_t idt_sm[kEmWarps][32];
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t nw = gridDim.x * kEmWarps;
  uint32_t u = blockIdx.x * kEmWarps + (threadIdx.x >> 5);
  if (u >= nunits) return;
  uint32_t* idt = idt_sm[threadIdx.x >> 5];
  struct L1 { uint2 un; uint32_t tb; };
  struct L2 { uint32_t idx, idi, msk, acc, nxt; };
  auto load1 = [&](uint32_t uu) -> L1 {              // needs only the unit index
    L1 r; r.un = make_uint2(0u, 0u); r.tb = 0u;
    if (uu < nunits) { const uint32_t uid = active ? active[uu] : uu; r.un = units[uid]; r.tb = ubase[uid]; }
    return r;
  };
  auto load2 = [&](const L1& a) -> L2 {              // needs the descriptor
    L2 r; r.idx = 0u; r.idi = 0u; r.msk = 0u; r.acc = 0u; r.nxt = 0u;
    if (a.un.y) {
      if (lane < a.un.y) r.idx = ids[a.un.x + lane];
      if (lane < min(32u, a.un.y - 1u)) {
        r.idi = ids_int[a.un.x + lane];
        r.acc = cnt_off[a.un.x + lane];
        r.nxt = cnt_off[a.un.x + lane + 1];
      }
      r.msk = masks[(size_t)a.tb * 32 + lane];
    }
    return r;
  };
  // kFillDepth units in flight per warp: descriptors kFillDepth ahead, their ids / masks / offsets
  // kFillDepth - 1 ahead
  L1 a[kFillDepth];
  L2 b[kFillDepth - 1];
#pragma unroll
  for (int q = 0; q < kFillDepth; ++q) a[q] = load1(u + q * nw);
#pragma unroll
  for (int q = 0; q < kFillDepth - 1; ++q) b[q] = load2(a[q]);
  for (; u < nunits; u += nw) {
    const L2 bn = load2(a[kFillDepth - 1]);          // chains of the next units advance one level
    const L1 an = load1(u + kFillDepth * nw);
    const L1 a0 = a[0];
    const L2 b0 = b[0];
    // ---- the current unit
    const uint32_t g0 = a0.un.x, mrem = a0.un.y;
    const uint32_t* __restrict__ idp = ids + g0;
    const uint32_t* __restrict__ mp = masks + (size_t)a0.tb * 32 + lane;
    uint32_t mask = b0.msk, idc = b0.idx, acc = b0.acc;
    if (b0.nxt > acc)                                // where the row kernel finds this group
      loc[(size_t)(g0 / n2) * n2 + b0.idi] = make_uint2(acc, b0.nxt - acc);
    for (uint32_t c0 = 0; c0 < mrem; c0 += 32) {
      uint32_t mask_n = 0, idc_n = 0;                // next tile, in flight during this one
      if (c0 + 32 < mrem) {
        mask_n = mp[(size_t)(c0 + 32)];              // (c0+32)/32 tiles further = (c0+32) words
        if (c0 + 32 + lane < mrem) idc_n = idp[c0 + 32 + lane];
      }
      // the tile's 32 column ids go through shared memory; every lane then walks its own bits (no
      // vote, no shuffle per partner: the loop is divergent, but it is half the instructions)
      __syncwarp();
      idt[lane] = idc;
      __syncwarp();
      while (mask) {
        const int c = __ffs(mask) - 1;
        mask &= mask - 1;
        outJ[acc++] = idt[c];
      }
      mask = mask_n; idc = idc_n;
    }
#pragma unroll
    for (int q = 0; q + 1 < kFillDepth; ++q) a[q] = a[q + 1];
    a[kFillDepth - 1] = an;
#pragma unroll
    for (int q = 0; q + 2 < kFillDepth; ++q) b[q] = b[q + 1];
    b[kFillDepth - 2] = bn;
  }
}

// Small units: ONE THREAD per bucket of at most kSmallMax kept members (bands >= 1).  The thread
// walks the bucket's pairs (row r, column c > r) itself: the row's S values of the earlier bands in
// registers, the column's read chunk by chunk; the same first-band rule as the warp kernels.  No
// mask cache: the fill pass repeats the few compares.  MODE EM_COUNT writes cnt[g] per row record,
// EM_FILL_J appends the partners at the scanned offsets and leaves loc[band][row].
template <int BW, int MODE>
__global__ void __launch_bounds__(128)
small_units_kernel(const uint2* __restrict__ units_s, uint32_t nsmall, const uint32_t* __restrict__ ids,
                   const uint32_t* __restrict__ ids_int, uint32_t n2, const uint32_t* __restrict__ S,
                   uint32_t* __restrict__ cnt_off, uint32_t* __restrict__ outJ, uint2* __restrict__ loc,
                   uint32_t row_lo, uint32_t row_hi) {
  constexpr int SW = 4 * BW;
  const uint32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= nsmall) return;
  const uint2 unit = units_s[u];
  const uint32_t g0 = unit.x, m = unit.y;                 // m kept members, 2 <= m <= kSmallMax
  const int b = (int)(g0 / n2);
  const int nch = (b + 3) >> 2;
  // the bucket's members lie in [first id, last id]: nothing to do outside the range of this call
  if (ids[g0] >= row_hi || ids[g0 + m - 2] < row_lo) return;
  for (uint32_t r = 0; r + 1 < m; ++r) {
    const uint32_t ext = ids[g0 + r];
    if (ext < row_lo || ext >= row_hi) continue;
    const uint32_t row = ids_int[g0 + r];
    uint4 R[BW];
#pragma unroll
    for (int ch = 0; ch < BW; ++ch) {
      if (ch < nch) {
        uint4 v = *reinterpret_cast<const uint4*>(S + (int64_t)row * SW + 4 * ch);
        if (4 * ch + 1 >= b) v.y = kFull;                 // bands >= b never match (no S value is 0xFFFFFFFF)
        if (4 * ch + 2 >= b) v.z = kFull;
        if (4 * ch + 3 >= b) v.w = kFull;
        R[ch] = v;
      }
    }
    uint32_t acc = 0, first = 0;
    if (MODE != EM_COUNT) { acc = cnt_off[g0 + r]; first = acc; }
    for (uint32_t c = r + 1; c < m; ++c) {
      const uint32_t col = ids_int[g0 + c];
      bool dup = false;
#pragma unroll
      for (int ch = 0; ch < BW; ++ch) {
        if (ch < nch) {
          const uint4 v = *reinterpret_cast<const uint4*>(S + (int64_t)col * SW + 4 * ch);
          dup |= (v.x == R[ch].x) | (v.y == R[ch].y) | (v.z == R[ch].z) | (v.w == R[ch].w);
        }
      }
      if (!dup) {
        if (MODE != EM_COUNT) outJ[acc] = ids[g0 + c];
        ++acc;
      }
    }
    if (MODE == EM_COUNT) cnt_off[g0 + r] = acc;
    else if (acc > first) loc[(size_t)b * n2 + row] = make_uint2(first, acc - first);
  }
}

// ---------------------------------------------------------------------------------------------
// a5.3  every row into its slice of the output, in ascending j if asked
// ---------------------------------------------------------------------------------------------
// One warp per INTERNAL row r (rows are visited in band 0's sorted order, i.e. family by family,
// and written to the slice of `out` that belongs to the row's EXTERNAL id: ext_off).  The row's
// partners (external ids) sit in the partner scratch as <= B ascending groups, group b at
// inJ[off[b*n2+r], off[b*n2+r+1]).  The ids of a repertoire carry no structure, so the partners
// of a row are spread evenly between the row's smallest and largest partner: ONE
// most-significant-digit pass over kRsBins equal-width value bins (shared-memory counters)
// groups them, and an element's final place is its bin's start plus the number of smaller
// elements in its own bin (1-2 on average, any number is correct).  The row's output slice (2T
// words) is the scratch: X = words [0,T), Y = words [T,2T).  Passes: gather the groups into X ->
// count per bin -> scan -> group by bin into Y -> rank inside the bin, sorted, back into X ->
// expand X into (i, j) pairs in place, from the top down.
constexpr int kRsWarps = 8;
constexpr int kRsBins = 1024;

__device__ __forceinline__ void
sort_one_row(const uint32_t* __restrict__ inJ, uint2* out, uint32_t gs, uint32_t len, uint32_t row,
             uint32_t obase, bool do_sort, uint32_t* bins, int lane) {
  // lane b holds group b: (gs, len) = its start in inJ and its length (row_group below)
  uint32_t pre = len;                        // inclusive -> exclusive prefix of the group lengths
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t o = __shfl_up_sync(kFull, pre, d);
    if (lane >= d) pre += o;
  }
  const uint32_t T = __shfl_sync(kFull, pre, 31);
  if (T == 0) return;
  pre -= len;
  const uint32_t nonempty = __ballot_sync(kFull, len > 0);
  out += obase;                              // the row's slice of the output
  uint32_t* X = reinterpret_cast<uint32_t*>(out);
  // the groups are small (a few elements each): four are gathered per step, loads first
  auto gather = [&](auto&& put) {
    uint32_t gm = nonempty;
    while (gm) {
      uint32_t s[4], l[4], p[4], v[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        l[k] = 0; s[k] = 0; p[k] = 0;
        if (gm) {
          const int g = __ffs(gm) - 1;
          gm &= gm - 1;
          s[k] = __shfl_sync(kFull, gs, g); l[k] = __shfl_sync(kFull, len, g); p[k] = __shfl_sync(kFull, pre, g);
        }
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) v[k] = (uint32_t)lane < l[k] ? inJ[s[k] + lane] : 0u;
#pragma unroll
      for (int k = 0; k < 4; ++k) if ((uint32_t)lane < l[k]) put(p[k] + lane, v[k]);
#pragma unroll
      for (int k = 0; k < 4; ++k)
        for (uint32_t e = 32 + lane; e < l[k]; e += 32) put(p[k] + e, inJ[s[k] + e]);
    }
  };
  if (__popc(nonempty) == 1 || !do_sort) {   // already ascending, or the grouped order is asked for
    gather([&](uint32_t at, uint32_t x) { out[at] = make_uint2(row, x); });
    return;
  }
  uint32_t lo = kFull, hi = 0;               // value range: every group is ascending
  if (len > 0) { lo = inJ[gs]; hi = inJ[gs + len - 1]; }
  gather([&](uint32_t at, uint32_t x) { X[at] = x; });
  __syncwarp();
  if (T <= 32) {                             // rank by counting inside the warp
    const uint32_t x = (uint32_t)lane < T ? X[lane] : kFull;
    uint32_t rank = 0;
    for (uint32_t s = 0; s < T; ++s) rank += __shfl_sync(kFull, x, s) < x ? 1u : 0u;
    __syncwarp();
    if ((uint32_t)lane < T) out[rank] = make_uint2(row, x);
    return;
  }
  lo = __reduce_min_sync(kFull, lo);
  hi = __reduce_max_sync(kFull, hi);
  // 64, 256 or 1,024 bins by row size (zeroing and scanning the bins is the fixed cost of a row)
  const int psh = T <= 64u ? 1 : T <= 256u ? 3 : 5;          // log2(bins per lane)
  const uint32_t nbins = 32u << psh;
  const float scale = (float)nbins / ((float)(hi - lo) + 1.0f);
  auto bin_of = [&](uint32_t x) -> uint32_t {     // monotone in x, < nbins
    return min(nbins - 1u, (uint32_t)((float)(x - lo) * scale));
  };
  // bin b lives at word b + b/per (per = bins per lane): the lane-major walk of the scan below
  // is then conflict-free
  auto bin_at = [&](uint32_t x) -> uint32_t { const uint32_t b = bin_of(x); return b + (b >> psh); };
  uint32_t* Y = X + T;
  for (uint32_t q = lane; q < nbins + 32u; q += 32) bins[q] = 0u;
  __syncwarp();
  // (every pass loads 4 batches of 32 before it uses them: the passes are latency-bound)
  for (uint32_t t0 = lane; t0 < T; t0 += 128) {
    uint32_t x[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = t0 + 32 * u < T ? X[t0 + 32 * u] : 0u;
#pragma unroll
    for (int u = 0; u < 4; ++u) if (t0 + 32 * u < T) atomicAdd(&bins[bin_at(x[u])], 1u);
  }
  __syncwarp();
  {                                          // exclusive scan of the bin counts
    const int per = 1 << psh;
    uint32_t* mine = bins + lane * (per + 1);
    uint32_t s = 0;
    for (int q = 0; q < per; ++q) s += mine[q];
    uint32_t inc = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t o = __shfl_up_sync(kFull, inc, d);
      if (lane >= d) inc += o;
    }
    uint32_t run = inc - s;
    for (int q = 0; q < per; ++q) { const uint32_t v = mine[q]; mine[q] = run; run += v; }
  }
  __syncwarp();
  for (uint32_t t0 = lane; t0 < T; t0 += 128) {   // group by bin (arrival order inside a bin)
    uint32_t x[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = t0 + 32 * u < T ? X[t0 + 32 * u] : 0u;
#pragma unroll
    for (int u = 0; u < 4; ++u) if (t0 + 32 * u < T) Y[atomicAdd(&bins[bin_at(x[u])], 1u)] = x[u];
  }
  __syncwarp();                              // now bins[b] = end of bin b = start of bin b+1
  for (uint32_t t0 = lane; t0 < T; t0 += 128) {   // rank inside the bin -> sorted, back into X
    uint32_t x[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = t0 + 32 * u < T ? Y[t0 + 32 * u] : 0u;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (t0 + 32 * u < T) {
        const uint32_t b = bin_of(x[u]);
        const uint32_t s = b ? bins[(b - 1) + ((b - 1) >> psh)] : 0u, e = bins[b + (b >> psh)];
        uint32_t rk = s;
        for (uint32_t q = s; q < e; ++q) rk += Y[q] < x[u] ? 1u : 0u;
        X[rk] = x[u];
      }
    }
  }
  __syncwarp();
  // expand in place, top down: pair t lands on words 2t, 2t+1 >= t, i.e. never on an element
  // of a lower batch; inside a batch every load precedes every store
  for (uint32_t t1 = (T + 127) / 128 * 128; t1 > 0; t1 -= 128) {
    const uint32_t t0 = t1 - 128 + lane;
    uint32_t x[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = t0 + 32 * u < T ? X[t0 + 32 * u] : 0u;
    __syncwarp();
#pragma unroll
    for (int u = 0; u < 4; ++u) if (t0 + 32 * u < T) out[t0 + 32 * u] = make_uint2(row, x[u]);
  }
}

constexpr int kRsChunk = 8;

__global__ void __launch_bounds__(kRsWarps * 32, 5)
row_sort_kernel(const uint32_t* __restrict__ off, const uint2* __restrict__ loc, int64_t n2, int bands,
                const uint32_t* __restrict__ ids0, const uint32_t* __restrict__ ext_off,
                bool do_sort, const uint32_t* __restrict__ inJ, uint2* out,
                unsigned long long* __restrict__ next_row, const uint32_t* __restrict__ rowstart,
                uint32_t* __restrict__ delta, uint4* __restrict__ sched, uint32_t row_lo, uint32_t row_hi) {
  __shared__ __align__(16) uint32_t bins_sh[kRsWarps][kRsBins + kRsBins / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  // Rows differ by four orders of magnitude in size: persistent warps fetch rows kRsChunk at a
  // time from a global counter, so no warp idles behind a heavy row of its block.
  for (;;) {
    unsigned long long first = 0;
    if (lane == 0) first = atomicAdd(next_row, (unsigned long long)kRsChunk);
    first = __shfl_sync(kFull, first, 0);
    if ((int64_t)first >= n2) return;
    const int64_t last = min(n2, (int64_t)first + kRsChunk);
    // the loads of row r + 1 (its external id one row earlier still) are issued before row r is
    // worked on: the chain id -> output offset and the group table never stall the sort
    auto row_group = [&](int64_t r) -> uint2 {           // lane b: group b of row r
      uint2 g = make_uint2(0u, 0u);
      if (lane == 0) { g.x = off[r]; g.y = off[r + 1] - g.x; }
      else if (lane < bands) g = loc[(int64_t)lane * n2 + r];
      return g;
    };
    uint32_t i_c = ids0[first];
    uint32_t i_n = (int64_t)first + 1 < last ? ids0[first + 1] : 0u;
    uint2 g_c = row_group((int64_t)first);
    uint32_t eo_c = ext_off[i_c];
    for (int64_t r = (int64_t)first; r < last; ++r) {
      const uint32_t i = i_c, eo = eo_c;     // external id of internal row r, its output offset
      const uint2 g = g_c;
      if (r + 1 < last) {
        i_c = i_n;
        eo_c = ext_off[i_n];
        g_c = row_group(r + 1);
        if (r + 2 < last) i_n = ids0[r + 2];
      }
      if (sched) {
        // the family-ordered chunk schedule of the edit-distance stage (sq_common.cuh): delta[r] =
        // (first pair of row r in the caller's buffer) - rowstart[r]; sched[k] for every chunk k
        // whose first position 32k falls into row r
        const uint32_t b = rowstart[r], e = rowstart[r + 1];
        const uint32_t d = eo - b;
        if (lane == 0) delta[r] = d;
        for (uint32_t k = (b + 31) / 32 + lane; (uint64_t)k * 32 < e; k += 32)
          sched[k] = make_uint4((uint32_t)r, d, e, b);
      }
      if (i >= row_lo && i < row_hi) sort_one_row(inJ, out, g.x, g.y, i, eo, do_sort, bins_sh[w], lane);
      __syncwarp();
    }
  }
}

template <int BW>
int launch_emit(sq_ctx* c, int mode, const uint2* units, const uint32_t* active, uint32_t nunits, const uint32_t* ids,
                const uint32_t* ids_int, uint32_t n2, int bands, const uint32_t* S,
                uint32_t* cnt_off, uint32_t* outJ, const uint32_t* ubase, uint32_t* masks, uint2* loc,
                uint32_t row_lo, uint32_t row_hi) {
  // persistent warps: exactly the resident blocks of every SM, never more warps than units
  int per_sm = 0;
  cudaError_t e;
  if (mode == EM_COUNT)
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, emit_kernel<BW, EM_COUNT>, kEmWarps * 32, 0);
  else
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, emit_kernel<BW, EM_FILL_J>, kEmWarps * 32, 0);
  if (e != cudaSuccess || per_sm < 1) per_sm = 4;
  unsigned g = (unsigned)(c->sm_count * per_sm);
  const unsigned need = (nunits + kEmWarps - 1) / kEmWarps;
  if (g > need) g = need;
  if (mode == EM_COUNT)
    SQ_TIMED(c, SQ_K_EMIT, emit_kernel<BW, EM_COUNT><<<g, kEmWarps * 32, 0, c->stream>>>(
        units, active, nunits, ids, ids_int, n2, bands, S, cnt_off, outJ, ubase, masks, loc, row_lo, row_hi));
  else
    SQ_TIMED(c, SQ_K_EMIT, emit_kernel<BW, EM_FILL_J><<<g, kEmWarps * 32, 0, c->stream>>>(
        units, active, nunits, ids, ids_int, n2, bands, S, cnt_off, outJ, ubase, masks, loc, row_lo, row_hi));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int launch_emit_band0(sq_ctx* c, int mode, const uint2* units0, const uint32_t* active0, uint32_t nunits0,
                      const uint32_t* ids, int bands, uint32_t* cnt_off, uint32_t* outJ,
                      uint32_t row_lo, uint32_t row_hi) {
  const unsigned g = (nunits0 + kEmWarps - 1) / kEmWarps;
  if (mode == EM_COUNT)
    SQ_TIMED(c, SQ_K_EMIT, emit_band0_kernel<EM_COUNT><<<g, kEmWarps * 32, 0, c->stream>>>(
        units0, active0, nunits0, ids, bands, cnt_off, outJ, row_lo, row_hi));
  else
    SQ_TIMED(c, SQ_K_EMIT, emit_band0_kernel<EM_FILL_J><<<g, kEmWarps * 32, 0, c->stream>>>(
        units0, active0, nunits0, ids, bands, cnt_off, outJ, row_lo, row_hi));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int launch_fill_masks(sq_ctx* c, const uint2* units, const uint32_t* active, uint32_t nunits, const uint32_t* ubase,
                      const uint32_t* masks, const uint32_t* ids, const uint32_t* ids_int,
                      uint32_t n2, int bands, const uint32_t* cnt_off, uint32_t* outJ, uint2* loc) {
  unsigned g = (unsigned)c->sm_count * 16u;          // 64 warps per SM, persistent
  const unsigned need = (nunits + kEmWarps - 1) / kEmWarps;
  if (g > need) g = need;
  SQ_TIMED(c, SQ_K_EMIT, emit_fill_masks_kernel<<<g, kEmWarps * 32, 0, c->stream>>>(
      units, active, nunits, ubase, masks, ids, ids_int, n2, bands, cnt_off, outJ, loc));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

// both unit lists, one mode.  `masks` (may be nullptr): the per-tile masks of new pairs, written
// by the count pass and, when present, read by the fill pass instead of repeating the compares.
// (active / active0 = the units of this call's row range, nullptr = all; nunits / nunits0 = their number)
template <int BW>
int launch_small(sq_ctx* c, int mode, const uint2* units_s, uint32_t nsmall, const uint32_t* ids,
                 const uint32_t* ids_int, uint32_t n2, const uint32_t* S, uint32_t* cnt_off, uint32_t* outJ,
                 uint2* loc, uint32_t row_lo, uint32_t row_hi) {
  const unsigned g = (nsmall + 127) / 128;
  if (mode == EM_COUNT)
    SQ_TIMED(c, SQ_K_EMIT, small_units_kernel<BW, EM_COUNT><<<g, 128, 0, c->stream>>>(
        units_s, nsmall, ids, ids_int, n2, S, cnt_off, outJ, loc, row_lo, row_hi));
  else
    SQ_TIMED(c, SQ_K_EMIT, small_units_kernel<BW, EM_FILL_J><<<g, 128, 0, c->stream>>>(
        units_s, nsmall, ids, ids_int, n2, S, cnt_off, outJ, loc, row_lo, row_hi));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int dispatch_emit(sq_ctx* c, int bw, int mode, const uint2* units, const uint32_t* active, uint32_t nunits,
                  const uint2* units0, const uint32_t* active0, uint32_t nunits0, const uint2* units_s,
                  uint32_t nsmall, const uint32_t* ids,
                  const uint32_t* ids_int, uint32_t n2, int bands, const uint32_t* S,
                  uint32_t* cnt_off, uint32_t* outJ, const uint32_t* ubase, uint32_t* masks, uint2* loc,
                  uint32_t row_lo, uint32_t row_hi) {
  int rc = SQ_OK;
  if (nsmall) {
    switch (bw) {
      case 1: rc = launch_small<1>(c, mode, units_s, nsmall, ids, ids_int, n2, S, cnt_off, outJ, loc, row_lo, row_hi); break;
      case 2: rc = launch_small<2>(c, mode, units_s, nsmall, ids, ids_int, n2, S, cnt_off, outJ, loc, row_lo, row_hi); break;
      case 4: rc = launch_small<4>(c, mode, units_s, nsmall, ids, ids_int, n2, S, cnt_off, outJ, loc, row_lo, row_hi); break;
      default: rc = launch_small<8>(c, mode, units_s, nsmall, ids, ids_int, n2, S, cnt_off, outJ, loc, row_lo, row_hi); break;
    }
    if (rc != SQ_OK) return rc;
  }
  if (nunits0) rc = launch_emit_band0(c, mode, units0, active0, nunits0, ids, bands, cnt_off, outJ, row_lo, row_hi);
  if (rc != SQ_OK || nunits == 0) return rc;
  if (mode != EM_COUNT && masks)
    return launch_fill_masks(c, units, active, nunits, ubase, masks, ids, ids_int, n2, bands, cnt_off, outJ, loc);
  switch (bw) {
    case 1: return launch_emit<1>(c, mode, units, active, nunits, ids, ids_int, n2, bands, S, cnt_off, outJ, ubase, masks, loc, row_lo, row_hi);
    case 2: return launch_emit<2>(c, mode, units, active, nunits, ids, ids_int, n2, bands, S, cnt_off, outJ, ubase, masks, loc, row_lo, row_hi);
    case 4: return launch_emit<4>(c, mode, units, active, nunits, ids, ids_int, n2, bands, S, cnt_off, outJ, ubase, masks, loc, row_lo, row_hi);
    default: return launch_emit<8>(c, mode, units, active, nunits, ids, ids_int, n2, bands, S, cnt_off, outJ, ubase, masks, loc, row_lo, row_hi);
  }
}

// the units with at least one row of the id range [row_lo, row_hi): the ids of a bucket ascend, so a
// unit's rows lie between the ids of its first and its last row (order of the list is irrelevant)
__global__ void __launch_bounds__(256)
active_units_kernel(const uint2* __restrict__ units, uint32_t nunits, const uint32_t* __restrict__ ids,
                    uint32_t row_lo, uint32_t row_hi, uint32_t* __restrict__ active,
                    unsigned long long* __restrict__ nactive) {
  const uint32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  bool on = false;
  if (u < nunits) {
    const uint2 un = units[u];
    const uint32_t nrows = min(32u, un.y - 1u);
    on = ids[un.x] < row_hi && ids[un.x + nrows - 1u] >= row_lo;
  }
  const uint32_t m = __ballot_sync(kFull, on);
  if (!m) return;
  const int lane = threadIdx.x & 31;
  unsigned long long base = 0;
  if (lane == 0) base = atomicAdd(nactive, (unsigned long long)__popc(m));
  base = __shfl_sync(kFull, base, 0);
  if (on) active[base + __popc(m & ((1u << lane) - 1u))] = u;
}

// ---------------------------------------------------------------------------------------------
// the schedule of the DP stage in FAMILY-LABEL order
// ---------------------------------------------------------------------------------------------
// The internal row order (band 0's bucket order) keeps the members of one band-0 bucket together, but a
// clonal family is many band-0 buckets -- a member with two or three edits usually sits in a bucket of
// its own -- scattered over the order by their hash keys, while its partners are spread over the whole
// family: the text gathers of such rows miss L2.  So the schedule visits the rows in the order of a
// LABEL: the smallest external id among the row itself and the heads of all buckets it shares (a
// bucket's ids ascend, so its head is its smallest member) -- one round of min-id propagation over the
// buckets.  Almost every member of a family shares some bucket with the family's exact copies of the
// seed, so a family gets one label and its rows become neighbours in the schedule.  Only the schedule
// (a permutation of pair indices) changes; outputs do not.  Config 4: DRAM reads of the DP kernel
// 54.7 -> ~20 GB, DP 27.3 -> 25.2 ms for ~1.0 ms of extra kernels (label: 16 gathers per row; a 3-pass
// sort of 10 M (label, row) records; sizes, scan, schedule entries), step -1.1 ms.
__global__ void __launch_bounds__(256)
sched_label_kernel(const uint32_t* __restrict__ S, int SW, int bands, const uint32_t* __restrict__ vin,
                   int64_t n2, uint64_t* __restrict__ keys, uint32_t* __restrict__ rows) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n2) return;
  uint32_t label = vin[r];                           // band 0: record r is internal row r
  for (int b0 = 0; b0 < bands; b0 += 4) {
    const uint4 v = *reinterpret_cast<const uint4*>(S + r * SW + b0);
    const uint32_t vv[4] = {v.x, v.y, v.z, v.w};
    uint32_t hid[4];
#pragma unroll
    for (int q = 0; q < 4; ++q)                      // (a sentinel: the row shares no bucket in that band)
      hid[q] = (b0 + q < bands && !(vv[q] & 0x80000000u)) ? vin[(int64_t)(b0 + q) * n2 + vv[q]] : 0xFFFFFFFFu;
#pragma unroll
    for (int q = 0; q < 4; ++q) label = min(label, hid[q]);
  }
  keys[r] = label;
  rows[r] = (uint32_t)r;
}

// sizes of the rows in schedule order (rowstart = exclusive scan of the sizes in internal order)
__global__ void __launch_bounds__(256)
sched_sizes_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ rowstart, int64_t n2,
                   uint32_t* __restrict__ sizes) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k > n2) return;
  uint32_t v = 0;
  if (k < n2) { const uint32_t r = order[k]; v = rowstart[r + 1] - rowstart[r]; }
  sizes[k] = v;
}

// delta2[k] and the chunk entries of schedule position k (= internal row order[k]); a warp takes 32
// positions and writes the chunk entries of each of them together
__global__ void __launch_bounds__(256)
sched_write_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ start2, int64_t n2,
                   const uint32_t* __restrict__ ids0, const uint32_t* __restrict__ ext_off,
                   uint32_t* __restrict__ delta2, uint4* __restrict__ sched) {
  const int lane = threadIdx.x & 31;
  const int64_t k = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
  uint32_t b = 0, e = 0, d = 0;
  if (k < n2) {
    b = start2[k]; e = start2[k + 1];
    d = ext_off[ids0[order[k]]] - b;
    delta2[k] = d;
  }
  // rows that hold the first position of at least one chunk
  uint32_t m = __ballot_sync(kFull, k < n2 && (((uint64_t)b + 31) / 32) * 32 < (uint64_t)e);
  while (m) {
    const int l = __ffs(m) - 1;
    m &= m - 1;
    const uint32_t bb = __shfl_sync(kFull, b, l), ee = __shfl_sync(kFull, e, l), dd = __shfl_sync(kFull, d, l);
    const uint32_t kk = (uint32_t)(k - lane + l);
    for (uint64_t c = ((uint64_t)bb + 31) / 32 + lane; c * 32 < ee; c += 32) sched[c] = make_uint4(kk, dd, ee, bb);
  }
}

inline int chunks_for(int bands) { return bands <= 4 ? 1 : bands <= 8 ? 2 : bands <= 16 ? 4 : 8; }

}  // namespace

size_t sq_lsh_scratch_bytes(int64_t n, int bands, int64_t pair_capacity) {
  const size_t nn = (size_t)(n > 0 ? n : 1), B = (size_t)(bands > 0 ? bands : 1);
  const size_t rec = nn * B;
  const size_t sw = 4 * (size_t)chunks_for((int)B);
  size_t s = 0;
  s += 2 * sq_align_up((rec + 4) * 8 + 16);    // keys ping-pong (the unit lists reuse one)
  s += 2 * sq_align_up(rec * 4 + 16);          // ids ping-pong (the internal rows reuse one)
  s += sq_align_up(nn * sw * 4 + 16);          // bucket-id table S
  s += sq_align_up((rec + 2) * 4 + 16);        // per record counts -> offsets
  s += sq_align_up((rec + 2) * 8 + 16);        // loc[band][row]: where the row kernel finds a group
  s += sq_align_up((rec / 2 + 2) * 4 + 16);    // first mask tile of every unit
  s += 4 * sq_align_up((nn + 2) * 4 + 16);     // non-empty flags / ranks; rowidx; ext_off; rowstart
  s += sq_sort_scratch_bytes(n, bands);
  s += sq_align_up((size_t)(pair_capacity > 0 ? pair_capacity : 0) * 4 + 16);   // partners
  s += sq_align_up(rec * 32 + 16);             // mask cache of the count pass (used if it fits)
  s += sq_align_up(((size_t)(pair_capacity > 0 ? pair_capacity : 0) / 32 + 2) * 16 + 16) +
       2 * sq_align_up((nn + 2) * 4 + 16);     // chunk schedule of the edit-distance stage
  s += 2 * sq_align_up((nn + 2) * 8 + 16) + 3 * sq_align_up((nn + 2) * 4 + 16);   // its family-label order
  return s + 4096;
}

// a3, a4, a5.1: band keys -> bucket sort -> bucket scan.  Leaves the sorted records, the bucket-id
// table S and the unit lists in the scratch (c->lsh) for any number of sq_lsh_emit_range calls.
extern "C" int sq_lsh_prepare(sq_ctx* c, const uint32_t* sig, int H, int bands, int rows, int bucket_cap,
                              int64_t* n_raw) {
  if (!c) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  if (n_raw) *n_raw = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (H < 1 || bands < 1 || rows < 1 || bucket_cap < 1 || (int64_t)bands * rows > H) return SQ_ERR_INVALID_ARG;
  if (bands > SQ_MAX_BANDS || H > SQ_MAX_H) return SQ_ERR_UNSUPPORTED;
  const int64_t n = c->n;
  c->last_raw_pairs = 0;
  sq_scratch_reset(c);
  sq_ctx::LshState& L = c->lsh;
  L = sq_ctx::LshState();
  L.n = n; L.bands = bands; L.bw = chunks_for(bands);
  if (n == 0) { L.valid = true; L.mark = c->scratch_top; return SQ_OK; }
  if (!sig) return SQ_ERR_INVALID_ARG;
  if (n * bands >= (1ll << 31)) return SQ_ERR_UNSUPPORTED;

  const size_t rec = (size_t)n * bands;
  const int sw = 4 * L.bw;
  uint64_t* k0 = sq_scratch<uint64_t>(c, rec + 4);     // (+4: the three unit lists end 2 entries past rec)
  uint64_t* k1 = sq_scratch<uint64_t>(c, rec + 4);
  uint32_t* v0 = sq_scratch<uint32_t>(c, rec);
  uint32_t* v1 = sq_scratch<uint32_t>(c, rec);
  uint32_t* S = sq_scratch<uint32_t>(c, (size_t)n * sw);
  uint32_t* cnt = sq_scratch<uint32_t>(c, rec + 2);
  uint32_t* ubase = sq_scratch<uint32_t>(c, rec / 2 + 2);
  uint2* loc = sq_scratch<uint2>(c, rec + 2);
  uint32_t* nonempty = sq_scratch<uint32_t>(c, (size_t)n + 2);
  uint32_t* rowidx = sq_scratch<uint32_t>(c, (size_t)n + 2);
  uint32_t* ext_off = sq_scratch<uint32_t>(c, (size_t)n + 2);
  uint32_t* rowstart = sq_scratch<uint32_t>(c, (size_t)n + 2);
  uint8_t* tmp = sq_scratch<uint8_t>(c, sq_sort_scratch_bytes(n, bands));
  if (!k0 || !k1 || !v0 || !v1 || !S || !cnt || !ubase || !loc || !nonempty || !rowidx || !ext_off || !rowstart || !tmp)
    return SQ_ERR_WORKSPACE;
  cudaStream_t st = c->stream;
  unsigned long long* counters = c->dflags;      // [0] unique, [1] raw, [2] n2, [4] units
  SQ_CUDA(c, cudaMemsetAsync(counters, 0, 128, st));

  // a3: band keys + non-empty flags
  const unsigned gb = (unsigned)((n + 255) / 256);
  if (rows == 4 && (H & 3) == 0 && (reinterpret_cast<uintptr_t>(sig) & 15) == 0)
    SQ_TIMED(c, SQ_K_BANDKEY, band_key4_kernel<<<gb, 256, 0, st>>>(sig, n, H, bands, k0, v0, nonempty));
  else
    SQ_TIMED(c, SQ_K_BANDKEY, band_key_kernel<<<gb, 256, 0, st>>>(sig, n, H, bands, rows, k0, v0, nonempty));
  SQ_LAUNCH_CHECK(c);
  int rc = sq_exclusive_scan_u32(c, nonempty, nonempty, n, reinterpret_cast<uint32_t*>(tmp),
                                 counters + 2);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters + 2, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t n2 = (int64_t)c->pinned[0];
  L.n2 = n2;
  if (n2 < 2) { L.valid = true; L.mark = c->scratch_top; return SQ_OK; }   // no pairs
  uint64_t* kin = k0; uint64_t* kalt = k1; uint32_t* vin = v0; uint32_t* valt = v1;
  if (n2 != n) {
    SQ_TIMED(c, SQ_K_BANDKEY, compact_kernel<<<gb, 256, 0, st>>>(k0, nonempty, n, n2, bands, k1, v1));
    SQ_LAUNCH_CHECK(c);
    kin = k1; kalt = k0; vin = v1; valt = v0;
  }
  // a4: stable radix sort of every band's records by the 64-bit key
  {
    int in_alt = 0;
    const int kb = c->sort_key_bytes;            // top bytes of the key the sort looks at (1..8)
    if (n2 < (1ll << 30)) {
      rc = sq_onesweep_sort(c, kin, kalt, vin, valt, n2, bands, 8 - kb, kb, tmp, &in_alt);
    } else {
      int shifts[8], widths[8];
      for (int p = 0; p < 8; ++p) { shifts[p] = 8 * p; widths[p] = 8; }
      rc = sq_radix_sort(c, kin, kalt, vin, valt, n2, bands, shifts, widths, 8, tmp, &in_alt);
    }
    if (rc != SQ_OK) return rc;
    if (in_alt) { uint64_t* t = kin; kin = kalt; kalt = t; uint32_t* tv = vin; vin = valt; valt = tv; }
    if (n2 < (1ll << 30) && kb < 8) {
      // prefix runs holding several full keys -> in full-key order (the list lives in `cnt`, which
      // is cleared afterwards; a mixed run has >= 2 records, so rec / 2 entries always suffice)
      dim3 gd((unsigned)((n2 + 255) / 256), (unsigned)bands);
      SQ_TIMED(c, SQ_K_SEGMENT, detect_mixed_kernel<<<gd, 256, 0, st>>>(
          kin, n2, 64 - 8 * kb, cnt, counters + 3));
      SQ_LAUNCH_CHECK(c);
      SQ_TIMED(c, SQ_K_SEGMENT, fix_mixed_kernel<<<(unsigned)(c->sm_count * 4), 256, 0, st>>>(
          kin, vin, kalt, valt, n2, 64 - 8 * kb, cnt, counters + 3));
      SQ_LAUNCH_CHECK(c);
    }
  }
  // internal rows: position in band 0's sorted order (band 0's records are vin[0, n2))
  const int64_t total = n2 * bands;
  const unsigned gt = (unsigned)((total + 255) / 256);
  uint32_t* vint = valt;                         // the dead id buffer: internal row of every record
  SQ_CUDA(c, cudaMemsetAsync(rowidx, 0xFF, (size_t)n * 4, st));
  SQ_TIMED(c, SQ_K_SEGMENT, rowidx_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(vin, n2, rowidx));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SEGMENT, translate_kernel<<<gt, 256, 0, st>>>(vin, total, rowidx, vint));
  SQ_LAUNCH_CHECK(c);
  // a5.1: buckets -> S table + unit lists (the unit lists live in the dead key buffer)
  uint2* units = reinterpret_cast<uint2*>(kalt);
  uint2* units0 = units + rec / 2 + 1;           // <= n2/2 units of band 0, <= rec/2 in all
  uint2* units_s = units0 + (size_t)n2 / 2 + 1;  // <= (rec - n2)/2 small units of bands >= 1
  SQ_TIMED(c, SQ_K_SEGMENT, s_prefill_kernel<<<(unsigned)((n2 * (sw / 4) + 255) / 256), 256, 0, st>>>(S, n2, sw));
  SQ_LAUNCH_CHECK(c);
  {
    dim3 grid((unsigned)((n2 + kBsTile - 1) / kBsTile), (unsigned)bands);
    SQ_TIMED(c, SQ_K_SEGMENT, bucket_scan_kernel<<<grid, kBsThreads, 0, st>>>(
        kin, vint, n2, bucket_cap, sw, S, units, units0, units_s, ubase, counters));
    SQ_LAUNCH_CHECK(c);
  }
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters, 128, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  c->last_raw_pairs = (int64_t)c->pinned[1];
  if (n_raw) *n_raw = c->last_raw_pairs;
  L.raw = c->last_raw_pairs;
  L.nunits = (uint32_t)c->pinned[4]; L.nunits0 = (uint32_t)c->pinned[5]; L.ntiles = c->pinned[7];
  L.nsmall = (uint32_t)c->pinned[8]; L.units_s = units_s;
  L.vin = vin; L.vint = vint; L.S = S; L.cnt = cnt; L.ubase = ubase; L.loc = loc; L.rowidx = rowidx;
  L.ext_off = ext_off; L.rowstart = rowstart; L.tmp = tmp; L.units = units; L.units0 = units0;
  // the sorted keys are dead from here on: the lists of a call's active units take their place
  L.active = reinterpret_cast<uint32_t*>(kin);
  L.mark = c->scratch_top;
  L.valid = true;
  return SQ_OK;
}

// a5.2, a5.3 for the rows (external ids) [row_lo, row_hi): count -> offsets -> fill -> every row of the
// range into its slice of pairs_out, ascending (i, j) (or grouped, SQ_LSH_UNORDERED).
extern "C" int sq_lsh_emit_range(sq_ctx* c, int64_t row_lo, int64_t row_hi, int flags, uint32_t* pairs_out,
                                 int64_t capacity, int64_t* n_pairs) {
  if (!c || !n_pairs) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  *n_pairs = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  sq_ctx::LshState& L = c->lsh;
  if (!L.valid || L.n != c->n) return SQ_ERR_NOT_PACKED;          // sq_lsh_prepare has not run (or its scratch is gone)
  if (capacity < 0 || (flags != SQ_LSH_SORTED && flags != SQ_LSH_UNORDERED) || row_lo < 0 || row_hi < row_lo ||
      row_hi > L.n)
    return SQ_ERR_INVALID_ARG;
  if (capacity > 0 && !pairs_out) return SQ_ERR_INVALID_ARG;
  c->scratch_top = L.mark;
  c->sched = nullptr;
  if (L.n2 < 2 || L.nunits + L.nunits0 + L.nsmall == 0 || row_lo == row_hi) return SQ_OK;
  const int64_t n = L.n, n2 = L.n2;
  const int bands = L.bands, bw = L.bw;
  const size_t rec = (size_t)n * bands;
  const int64_t total = n2 * bands;
  const uint32_t lo = (uint32_t)row_lo, hi = (uint32_t)(row_hi > 0xFFFFFFFFll ? 0xFFFFFFFFll : row_hi);
  cudaStream_t st = c->stream;
  unsigned long long* counters = c->dflags;
  uint32_t* cnt = L.cnt; uint2* loc = L.loc;
  uint32_t* tmp32 = reinterpret_cast<uint32_t*>(L.tmp);
  const unsigned gb = (unsigned)((n + 255) / 256);
  int rc;
  // the units that hold a row of the range (all of them for the whole repertoire)
  const bool whole = row_lo == 0 && row_hi == n;
  const uint32_t* active = nullptr; const uint32_t* active0 = nullptr;
  uint32_t nunits = L.nunits, nunits0 = L.nunits0;
  if (!whole) {
    uint32_t* act = L.active;                    // <= rec / 2 units in all; the key buffer holds 2 * rec words
    uint32_t* act0 = act + rec / 2 + 1;
    SQ_CUDA(c, cudaMemsetAsync(counters + 4, 0, 16, st));
    if (nunits) {
      SQ_TIMED(c, SQ_K_SEGMENT, active_units_kernel<<<(nunits + 255) / 256, 256, 0, st>>>(
          L.units, nunits, L.vin, lo, hi, act, counters + 4));
      SQ_LAUNCH_CHECK(c);
    }
    if (nunits0) {
      SQ_TIMED(c, SQ_K_SEGMENT, active_units_kernel<<<(nunits0 + 255) / 256, 256, 0, st>>>(
          L.units0, nunits0, L.vin, lo, hi, act0, counters + 5));
      SQ_LAUNCH_CHECK(c);
    }
    SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters, 64, cudaMemcpyDeviceToHost, st));
    SQ_CUDA(c, cudaStreamSynchronize(st));
    nunits = (uint32_t)c->pinned[4]; nunits0 = (uint32_t)c->pinned[5];
    active = act; active0 = act0;
    if (nunits + nunits0 + L.nsmall == 0) return SQ_OK;
  }
  // mask cache: 32 words per (unit, column tile); optional -- without it pass 2 repeats the compares
  uint32_t* masks = (nunits && L.ntiles) ? sq_scratch<uint32_t>(c, (size_t)L.ntiles * 32) : nullptr;
  // a5.2 pass 1: counts per sorted record -> offsets
  SQ_CUDA(c, cudaMemsetAsync(cnt, 0, (rec + 2) * 4, st));
  rc = dispatch_emit(c, bw, EM_COUNT, L.units, active, nunits, L.units0, active0, nunits0, L.units_s, L.nsmall, L.vin, L.vint, (uint32_t)n2,
                     bands, L.S, cnt, nullptr, L.ubase, masks, loc, lo, hi);
  if (rc != SQ_OK) return rc;
  rc = sq_exclusive_scan_u32(c, cnt, cnt, total + 1, tmp32, counters);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counters, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t uniq = (int64_t)c->pinned[0];
  *n_pairs = uniq;
  if (uniq > capacity) return SQ_ERR_CAPACITY;
  if (uniq >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;   // 32-bit output offsets (per call)
  if (uniq == 0) return SQ_OK;
  // a5.2 pass 2: the new partners of every sorted record into the partner scratch (unit by unit,
  // contiguous); it also leaves loc[band][row] = (start, length) of every non-empty group
  uint32_t* tmpJ = sq_scratch<uint32_t>(c, (size_t)uniq);
  if (!tmpJ) return SQ_ERR_WORKSPACE;
  SQ_CUDA(c, cudaMemsetAsync(loc, 0, (rec + 2) * 8, st));
  rc = dispatch_emit(c, bw, EM_FILL_J, L.units, active, nunits, L.units0, active0, nunits0, L.units_s, L.nsmall, L.vin, L.vint, (uint32_t)n2,
                     bands, L.S, cnt, tmpJ, L.ubase, masks, loc, lo, hi);
  if (rc != SQ_OK) return rc;
  // where every EXTERNAL row starts in the output
  uint32_t* rowstart = L.rowstart; uint32_t* ext_off = L.ext_off;
  SQ_TIMED(c, SQ_K_SEGMENT, row_total_kernel<<<(unsigned)((n2 + 256) / 256), 256, 0, st>>>(cnt, loc, n2, bands, rowstart));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SEGMENT, ext_count_kernel<<<gb, 256, 0, st>>>(L.rowidx, rowstart, n, ext_off));
  SQ_LAUNCH_CHECK(c);
  rc = sq_exclusive_scan_u32(c, ext_off, ext_off, n, tmp32, nullptr);
  if (rc != SQ_OK) return rc;
  rc = sq_exclusive_scan_u32(c, rowstart, rowstart, n2 + 1, tmp32, nullptr);
  if (rc != SQ_OK) return rc;                     // rowstart[r] = first internal position of row r
  // a5.3: every row (sorted if asked) into its slice of the output
  {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, row_sort_kernel, kRsWarps * 32, 0) != cudaSuccess ||
        per_sm < 1)
      per_sm = 2;
    unsigned g = (unsigned)(c->sm_count * per_sm);
    const unsigned need = (unsigned)((n2 + kRsWarps * kRsChunk - 1) / (kRsWarps * kRsChunk));
    if (g > need) g = need;
    SQ_CUDA(c, cudaMemsetAsync(counters + 6, 0, 8, st));
    // family-ordered chunk schedule for sq_edit_distance (a hint; skipped if it does not fit),
    // written by the row kernel on its way
    const size_t nchunks = ((size_t)uniq + 31) / 32;
    uint4* sched = sq_scratch<uint4>(c, nchunks);
    uint32_t* delta = sq_scratch<uint32_t>(c, (size_t)n2 + 1);
    if (!sched || !delta) { sched = nullptr; delta = nullptr; }
    // the schedule in family-label order (optional: without room for its arrays the row kernel writes the
    // schedule in internal row order on its way)
    // -- when the DP stages will follow the schedule: the packed sequences exceed sched_min_bytes (smaller
    // inputs sit in L2 anyway; the graph step, whose criterion is the size of the signatures, then walks
    // the internal row order the row kernel writes on its way)
    const uint32_t* sched_start = rowstart;
    bool by_label = false;
    const bool sched_used = (size_t)c->n * (size_t)c->stride > (size_t)c->sched_min_bytes;
    // (and only for the whole repertoire: the label kernels walk all rows, a call for a slice of the rows --
    // the streamed / sharded entry points make many -- keeps the schedule the row kernel writes for free)
    if (sched && c->sched_by_label && sched_used && whole && n2 < (1ll << 30)) {
      const size_t top = c->scratch_top;
      uint64_t* lk0 = sq_scratch<uint64_t>(c, (size_t)n2 + 2);
      uint64_t* lk1 = sq_scratch<uint64_t>(c, (size_t)n2 + 2);
      uint32_t* lv0 = sq_scratch<uint32_t>(c, (size_t)n2 + 2);
      uint32_t* lv1 = sq_scratch<uint32_t>(c, (size_t)n2 + 2);
      uint32_t* start2 = sq_scratch<uint32_t>(c, (size_t)n2 + 2);
      if (lk0 && lk1 && lv0 && lv1 && start2) {
        const unsigned gr = (unsigned)((n2 + 256) / 256);
        SQ_TIMED(c, SQ_K_SEGMENT, sched_label_kernel<<<gr, 256, 0, st>>>(L.S, 4 * bw, bands, L.vin, n2, lk0, lv0));
        SQ_LAUNCH_CHECK(c);
        int nb = 1;
        while (nb < 4 && (1ll << (8 * nb)) < n) ++nb;              // key bytes that hold the label (an external id)
        int in_alt = 0;
        rc = sq_onesweep_sort(c, lk0, lk1, lv0, lv1, n2, 1, 0, nb, L.tmp, &in_alt);
        if (rc != SQ_OK) return rc;
        const uint32_t* order = in_alt ? lv1 : lv0;
        SQ_TIMED(c, SQ_K_SEGMENT, sched_sizes_kernel<<<gr, 256, 0, st>>>(order, rowstart, n2, start2));
        SQ_LAUNCH_CHECK(c);
        rc = sq_exclusive_scan_u32(c, start2, start2, n2 + 1, tmp32, nullptr);
        if (rc != SQ_OK) return rc;
        SQ_TIMED(c, SQ_K_SEGMENT, sched_write_kernel<<<gr, 256, 0, st>>>(order, start2, n2, L.vin, ext_off, delta, sched));
        SQ_LAUNCH_CHECK(c);
        sched_start = start2;
        by_label = true;
      } else {
        c->scratch_top = top;
      }
    }
    SQ_TIMED(c, SQ_K_ROWSORT, row_sort_kernel<<<g, kRsWarps * 32, 0, st>>>(
        cnt, loc, n2, bands, L.vin, ext_off, flags == SQ_LSH_SORTED, tmpJ, reinterpret_cast<uint2*>(pairs_out),
        counters + 6, rowstart, by_label ? nullptr : delta, by_label ? nullptr : sched, lo, hi));
    SQ_LAUNCH_CHECK(c);
    if (sched) {
      c->sched = sched;
      c->sched_rowstart = sched_start;
      c->sched_delta = delta;
      c->sched_chunks = (int64_t)nchunks;
      c->sched_pairs = pairs_out;
      c->sched_npairs = uniq;
    }
  }
  SQ_CUDA(c, cudaStreamSynchronize(st));
  return SQ_OK;
}

extern "C" int sq_lsh_candidates(sq_ctx* c, const uint32_t* sig, int H, int bands, int rows,
                                 int bucket_cap, int flags, uint32_t* pairs_out, int64_t capacity,
                                 int64_t* n_pairs) {
  if (!c || !n_pairs) return SQ_ERR_INVALID_ARG;
  *n_pairs = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (capacity < 0 || (flags != SQ_LSH_SORTED && flags != SQ_LSH_UNORDERED)) return SQ_ERR_INVALID_ARG;
  if (c->n > 0 && capacity > 0 && !pairs_out) return SQ_ERR_INVALID_ARG;
  int rc = sq_lsh_prepare(c, sig, H, bands, rows, bucket_cap, nullptr);
  if (rc != SQ_OK) return rc;
  return sq_lsh_emit_range(c, 0, c->n, flags, pairs_out, capacity, n_pairs);
}
