// sq_join.cu -- SURVEY.md 8(f) ranks 3-4: the cross-repertoire join and its out-of-core driver.
//
// PAPER.md App. F.1, Eq. 45: a 2-D grid over "the two sequence batches being compared",
// N x M.  sq_all_pairs reads it as a self-join; here the two batches are two packed sets A and B
// (two contexts, same stride and alphabet) and the result is every (i in A, j in B) with
// d(A_i, B_j) <= max_d.  PAPER.md L139-143, Eq. 12: the batch size that keeps a tile inside the
// device memory -- sq_batch_size is that formula, and sq_join_host walks A in row blocks of that
// many cells, streaming each block's hits to the host while the next block is computed, so neither
// the hit list nor the survivor list of the whole rectangle ever has to fit in HBM.
//
//   join_filter_kernel   a block owns 256 columns j and kJoinRows rows i.  Each thread keeps its
//                        column's residue histogram (32 bytes) in registers; the rows' histograms
//                        sit in shared memory and are read as broadcasts.  Bag distance
//                        (L1 of the histograms + |m - n|) / 2 <= d (sq_allpairs.cu) decides
//                        whether the pair can be a hit; survivors are appended with
//                        warp-aggregated atomics.
//   DP                   sq_edit_distance_ab on the survivors (patterns from A, texts from B).
//   hits                 sq_hit_compact, then one radix sort by (i, j).
// A row range whose survivors do not fit their scratch is split in two and redone (host work
// list), so the only hard limit is one row against all of B.
#include "sq_common.cuh"

namespace {

constexpr int kJoinThreads = 256;
constexpr int kJoinRows = 16;

// NW = histogram words that can be non-zero: ceil(alphabet / 4) (5 for the 20 amino acids)
template <int NW>
__global__ void __launch_bounds__(kJoinThreads)
join_filter_kernel(const uint32_t* __restrict__ rhA, const uint32_t* __restrict__ lensA, int64_t row0,
                   int64_t rows, int64_t a_base, const uint32_t* __restrict__ rhB,
                   const uint32_t* __restrict__ lensB, int64_t nB, int max_d, int upper,
                   uint2* __restrict__ surv, unsigned long long scap,
                   unsigned long long* __restrict__ counter) {
  __shared__ uint32_t ha[kJoinRows][8];
  __shared__ int la[kJoinRows];
  const int64_t r0 = row0 + (int64_t)blockIdx.x * kJoinRows;          // first row (index into rhA)
  const int nr = (int)min((int64_t)kJoinRows, row0 + rows - r0);
  const int64_t jbase = (int64_t)blockIdx.y * kJoinThreads;
  // `upper`: columns j <= i never count; skip the block when all of its cells are such
  if (upper && jbase + kJoinThreads <= a_base + r0 + 1) return;
  if (threadIdx.x < (unsigned)(8 * nr)) ha[threadIdx.x >> 3][threadIdx.x & 7] = rhA[r0 * 8 + threadIdx.x];
  if (threadIdx.x >= 128 && threadIdx.x < 128u + (unsigned)nr) la[threadIdx.x - 128] = (int)lensA[r0 + threadIdx.x - 128];
  __syncthreads();
  const int64_t cidx = jbase + threadIdx.x;
  const bool col = cidx < nB;
  uint32_t hb[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  int nl = 0;
  const int64_t j = cidx;
  if (col) {
    const uint4 b0 = reinterpret_cast<const uint4*>(rhB)[cidx * 2];
    const uint4 b1 = reinterpret_cast<const uint4*>(rhB)[cidx * 2 + 1];
    hb[0] = b0.x; hb[1] = b0.y; hb[2] = b0.z; hb[3] = b0.w;
    hb[4] = b1.x; hb[5] = b1.y; hb[6] = b1.z; hb[7] = b1.w;
    nl = (int)lensB[cidx];
  }
  const int lane = threadIdx.x & 31;
  for (int r = 0; r < nr; ++r) {
    const int m = la[r];
    uint32_t l1 = (uint32_t)(m > nl ? m - nl : nl - m);
#pragma unroll
    for (int q = 0; q < NW; ++q) l1 += __vsadu4(ha[r][q], hb[q]);
    const int64_t i = a_base + r0 + r;                                 // row id in A
    const bool pass = col && (int)(l1 >> 1) <= max_d && (!upper || j > i);
    const uint32_t mask = __ballot_sync(0xFFFFFFFFu, pass);
    if (mask) {
      unsigned long long base = 0;
      if (lane == __ffs(mask) - 1) base = atomicAdd(counter, (unsigned long long)__popc(mask));
      base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
      if (pass) {
        const unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
        if (slot < scap) surv[slot] = make_uint2((uint32_t)i, (uint32_t)j);
      }
    }
  }
}

// Both sides in order of length (row r is sequence a_base + permA[r] of A, column c is sequence
// permB[c] of B): since |m - n| <= d, a tile of 16 rows only meets the columns whose length lies in
// [min length of the tile - max_d, max length + max_d] -- a contiguous range of the sorted columns,
// found by two binary searches.  Block (x, y) takes row tile x and every gridDim.y-th column block
// of that range; the rest is the kernel above.
template <int NW>
__global__ void __launch_bounds__(kJoinThreads)
join_filter_ranged_kernel(const uint32_t* __restrict__ rhA, const uint32_t* __restrict__ lensA,
                          const uint32_t* __restrict__ permA, int64_t row0, int64_t rows, int64_t a_base,
                          const uint32_t* __restrict__ rhB, const uint32_t* __restrict__ lensB,
                          const uint32_t* __restrict__ permB, int64_t nB, int max_d,
                          uint2* __restrict__ surv, unsigned long long scap,
                          unsigned long long* __restrict__ counter) {
  __shared__ uint32_t ha[kJoinRows][8];
  __shared__ int la[kJoinRows];
  __shared__ uint32_t ia[kJoinRows];
  __shared__ int64_t crange[2];
  const int64_t r0 = row0 + (int64_t)blockIdx.x * kJoinRows;
  const int nr = (int)min((int64_t)kJoinRows, row0 + rows - r0);
  if (threadIdx.x < (unsigned)(8 * nr)) ha[threadIdx.x >> 3][threadIdx.x & 7] = rhA[r0 * 8 + threadIdx.x];
  if (threadIdx.x >= 128 && threadIdx.x < 128u + (unsigned)nr) {
    la[threadIdx.x - 128] = (int)lensA[r0 + threadIdx.x - 128];
    ia[threadIdx.x - 128] = permA[r0 + threadIdx.x - 128];
  }
  if (threadIdx.x == 255) {
    // rows ascend in length: first column with length >= lo, first with length > hi
    const int lo = (int)lensA[r0] - max_d, hi = (int)lensA[r0 + nr - 1] + max_d;
    int64_t a = 0, b = nB;
    while (a < b) { const int64_t mid = (a + b) >> 1; if ((int)lensB[mid] < lo) a = mid + 1; else b = mid; }
    crange[0] = a;
    b = nB;
    while (a < b) { const int64_t mid = (a + b) >> 1; if ((int)lensB[mid] <= hi) a = mid + 1; else b = mid; }
    crange[1] = a;
  }
  __syncthreads();
  const int64_t c_lo = crange[0] / kJoinThreads * kJoinThreads, c_hi = crange[1];
  const int lane = threadIdx.x & 31;
  for (int64_t jbase = c_lo + (int64_t)blockIdx.y * kJoinThreads; jbase < c_hi;
       jbase += (int64_t)gridDim.y * kJoinThreads) {
    const int64_t cidx = jbase + threadIdx.x;
    const bool col = cidx < c_hi;
    uint32_t hb[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int nl = 0;
    uint32_t j = 0;
    if (col) {
      const uint4 b0 = reinterpret_cast<const uint4*>(rhB)[cidx * 2];
      const uint4 b1 = reinterpret_cast<const uint4*>(rhB)[cidx * 2 + 1];
      hb[0] = b0.x; hb[1] = b0.y; hb[2] = b0.z; hb[3] = b0.w;
      hb[4] = b1.x; hb[5] = b1.y; hb[6] = b1.z; hb[7] = b1.w;
      nl = (int)lensB[cidx];
      j = permB[cidx];
    }
    for (int r = 0; r < nr; ++r) {
      const int m = la[r];
      uint32_t l1 = (uint32_t)(m > nl ? m - nl : nl - m);
#pragma unroll
      for (int q = 0; q < NW; ++q) l1 += __vsadu4(ha[r][q], hb[q]);
      const bool pass = col && (int)(l1 >> 1) <= max_d;
      const uint32_t mask = __ballot_sync(0xFFFFFFFFu, pass);
      if (mask) {
        unsigned long long base = 0;
        if (lane == __ffs(mask) - 1) base = atomicAdd(counter, (unsigned long long)__popc(mask));
        base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
        if (pass) {
          const unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
          if (slot < scap) surv[slot] = make_uint2((uint32_t)a_base + ia[r], j);
        }
      }
    }
  }
}

// columns in order of length: histogram + length of column c = those of sequence perm[c]
__global__ void __launch_bounds__(256)
join_gather_cols_kernel(const uint32_t* __restrict__ rh, const uint32_t* __restrict__ lens,
                        const uint32_t* __restrict__ perm, int64_t n, uint32_t* __restrict__ rh_s,
                        uint32_t* __restrict__ lens_s) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const uint32_t src = perm[c];
  const uint4* in = reinterpret_cast<const uint4*>(rh) + (int64_t)src * 2;
  uint4* out = reinterpret_cast<uint4*>(rh_s) + c * 2;
  out[0] = in[0]; out[1] = in[1];
  lens_s[c] = lens[src];
}

__global__ void __launch_bounds__(256)
join_len_keys_kernel(const uint32_t* __restrict__ lens, int64_t n, uint64_t* __restrict__ keys,
                     uint32_t* __restrict__ vals) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  keys[c] = lens[c];
  vals[c] = (uint32_t)c;
}

inline int bits_for(int64_t n) {
  int b = 1;
  while (b < 32 && (1ll << b) < n) ++b;
  return b;
}

inline size_t join_survivor_cap(int64_t cap) { return 4 * (size_t)(cap > 0 ? cap : 1) + 65536; }

// (rh, lens) of n sequences -> the same in order of length + the permutation, in scratch above the
// current top.  *ok = 0 when the scratch does not hold it (the caller then stays unsorted).
int join_sort_by_length(sq_ctx* c, const uint32_t* rh, const uint32_t* lens, int64_t n,
                        const uint32_t** perm, const uint32_t** rh_s, const uint32_t** lens_s, int* ok) {
  *ok = 0;
  uint64_t* lk = sq_scratch<uint64_t>(c, (size_t)n);
  uint64_t* lk_alt = sq_scratch<uint64_t>(c, (size_t)n);
  uint32_t* lv = sq_scratch<uint32_t>(c, (size_t)n);
  uint32_t* lv_alt = sq_scratch<uint32_t>(c, (size_t)n);
  uint8_t* ltmp = sq_scratch<uint8_t>(c, sq_sort_scratch_bytes(n, 1));
  uint32_t* rhS = sq_scratch<uint32_t>(c, (size_t)n * 8);
  uint32_t* lensS = sq_scratch<uint32_t>(c, (size_t)n);
  if (!lk || !lk_alt || !lv || !lv_alt || !ltmp || !rhS || !lensS) return SQ_OK;
  const unsigned gb = (unsigned)((n + 255) / 256);
  SQ_TIMED(c, SQ_K_ALLPAIRS, join_len_keys_kernel<<<gb, 256, 0, c->stream>>>(lens, n, lk, lv));
  SQ_LAUNCH_CHECK(c);
  const int shifts[1] = {0}, widths[1] = {8};
  int in_alt = 0;
  int rc = sq_radix_sort(c, lk, lk_alt, lv, lv_alt, n, 1, shifts, widths, 1, ltmp, &in_alt);
  if (rc != SQ_OK) return rc;
  const uint32_t* pv = in_alt ? lv_alt : lv;
  SQ_TIMED(c, SQ_K_ALLPAIRS, join_gather_cols_kernel<<<gb, 256, 0, c->stream>>>(rh, lens, pv, n, rhS, lensS));
  SQ_LAUNCH_CHECK(c);
  *perm = pv; *rh_s = rhS; *lens_s = lensS; *ok = 1;
  return SQ_OK;
}

int join_filter_ranged(sq_ctx* c, const uint32_t* rhA, const uint32_t* lensA, const uint32_t* permA, int64_t row0,
                       int64_t rows, int64_t a_base, const uint32_t* rhB, const uint32_t* lensB,
                       const uint32_t* permB, int64_t nB, int max_d, uint2* surv, size_t scap,
                       unsigned long long* counter) {
  if (rows <= 0 || nB <= 0) return SQ_OK;
  const int64_t tiles = (rows + kJoinRows - 1) / kJoinRows;
  // enough blocks to fill the machine, at most one per column block
  int64_t gy = ((int64_t)c->sm_count * 32 + tiles - 1) / tiles;
  const int64_t cblocks = (nB + kJoinThreads - 1) / kJoinThreads;
  if (gy > cblocks) gy = cblocks;
  if (gy > 65535) gy = 65535;
  if (gy < 1) gy = 1;
  dim3 grid((unsigned)tiles, (unsigned)gy);
  const unsigned long long sc = (unsigned long long)scap;
  if (c->alphabet <= 20)
    SQ_TIMED(c, SQ_K_ALLPAIRS, join_filter_ranged_kernel<5><<<grid, kJoinThreads, 0, c->stream>>>(
        rhA, lensA, permA, row0, rows, a_base, rhB, lensB, permB, nB, max_d, surv, sc, counter));
  else
    SQ_TIMED(c, SQ_K_ALLPAIRS, join_filter_ranged_kernel<8><<<grid, kJoinThreads, 0, c->stream>>>(
        rhA, lensA, permA, row0, rows, a_base, rhB, lensB, permB, nB, max_d, surv, sc, counter));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

// Every hit of rows [a_begin, a_end) of A against all of B, sorted by (i, j), into device buffers.
// Scratch is taken above the current top and given back.  Synchronises.
int join_core(sq_ctx* a, const sq_ctx* b, int64_t a_begin, int64_t a_end, int max_d, int flags,
              uint32_t* pairs_out, uint16_t* dist_out, int64_t capacity, int64_t* n_out) {
  *n_out = 0;
  const int64_t rows = a_end - a_begin, nB = b->n;
  if (rows <= 0 || nB <= 0) return SQ_OK;
  if ((nB + kJoinThreads - 1) / kJoinThreads > 65535) return SQ_ERR_UNSUPPORTED;
  if (capacity >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;
  cudaStream_t st = a->stream;
  const size_t top = a->scratch_top;
  struct Restore { sq_ctx* c; size_t t; ~Restore() { c->scratch_top = t; } } restore{a, top};
  const size_t cap = (size_t)(capacity > 0 ? capacity : 1), scap = join_survivor_cap(capacity);
  uint64_t* hp = sq_scratch<uint64_t>(a, cap);
  uint64_t* hp_alt = sq_scratch<uint64_t>(a, cap);
  uint32_t* hd = sq_scratch<uint32_t>(a, cap);
  uint32_t* hd_alt = sq_scratch<uint32_t>(a, cap);
  uint8_t* tmp = sq_scratch<uint8_t>(a, sq_sort_scratch_bytes(capacity, 1));
  uint32_t* rhA = sq_scratch<uint32_t>(a, (size_t)rows * 8);
  uint32_t* lensA = sq_scratch<uint32_t>(a, (size_t)rows);
  uint32_t* rhB = sq_scratch<uint32_t>(a, (size_t)nB * 8);
  uint32_t* lensB = sq_scratch<uint32_t>(a, (size_t)nB);
  uint2* surv = sq_scratch<uint2>(a, scap);
  uint16_t* sdist = sq_scratch<uint16_t>(a, scap);
  uint2* surv2 = sq_scratch<uint2>(a, scap);
  uint8_t* tmp2 = sq_scratch<uint8_t>(a, sq_sort_scratch_bytes((int64_t)scap, 1));
  if (!surv2 || !tmp2 || !hp || !hp_alt || !hd || !hd_alt || !tmp || !rhA || !lensA || !rhB || !lensB || !surv || !sdist)
    return SQ_ERR_WORKSPACE;
  SQ_CUDA(a, cudaMemsetAsync(a->dflags, 0, 64, st));
  int rc = sq_residue_hist(a, a->packed + a_begin * a->stride, a->stride, rows, rhA, lensA);
  if (rc != SQ_OK) return rc;
  rc = sq_residue_hist(a, b->packed, b->stride, nB, rhB, lensB);
  if (rc != SQ_OK) return rc;
  // both sides in order of length (stable radix sort of (length, index), one 8-bit pass): a tile of
  // rows then only meets the columns within max_d of its lengths.  Not for SQ_JOIN_UPPER, whose
  // blocks below the diagonal are skipped by index instead; without the scratch: unsorted.
  const uint32_t* permA = nullptr; const uint32_t* permB = nullptr;
  const uint32_t* rhR = rhA; const uint32_t* lensR = lensA;
  const uint32_t* rhC = rhB; const uint32_t* lensC = lensB;
  if (!(flags & SQ_JOIN_UPPER) && nB >= 4096) {
    const uint32_t *pa = nullptr, *ra = nullptr, *la_ = nullptr, *pb = nullptr, *rb = nullptr, *lb_ = nullptr;
    int ok = 0;
    rc = join_sort_by_length(a, rhA, lensA, rows, &pa, &ra, &la_, &ok);
    if (rc != SQ_OK) return rc;
    if (ok) {
      rc = join_sort_by_length(a, rhB, lensB, nB, &pb, &rb, &lb_, &ok);
      if (rc != SQ_OK) return rc;
    }
    if (ok) { permA = pa; rhR = ra; lensR = la_; permB = pb; rhC = rb; lensC = lb_; }
  }
  // host work list of row ranges (relative to a_begin); a range whose survivors overflow is halved
  int64_t stack_lo[80], stack_n[80];
  int sp = 0;
  stack_lo[0] = 0; stack_n[0] = rows; sp = 1;
  while (sp > 0) {
    --sp;
    const int64_t lo = stack_lo[sp], cnt = stack_n[sp];
    SQ_CUDA(a, cudaMemsetAsync(a->dflags + 1, 0, 8, st));
    if (permA)
      rc = join_filter_ranged(a, rhR, lensR, permA, lo, cnt, a_begin, rhC, lensC, permB, nB, max_d, surv, scap,
                              a->dflags + 1);
    else
      rc = sq_bag_filter(a, rhA, lensA, lo, cnt, a_begin, rhB, lensB, nB, max_d, (flags & SQ_JOIN_UPPER) ? 1 : 0,
                         surv, scap, a->dflags + 1);
    if (rc != SQ_OK) return rc;
    SQ_CUDA(a, cudaMemcpyAsync(a->pinned, a->dflags + 1, 8, cudaMemcpyDeviceToHost, st));
    SQ_CUDA(a, cudaStreamSynchronize(st));
    const int64_t ns = (int64_t)a->pinned[0];
    if ((size_t)ns > scap) {
      if (cnt == 1 || sp + 2 > 80) return SQ_ERR_WORKSPACE;    // one row against B does not fit
      const int64_t h = cnt / 2;
      stack_lo[sp] = lo + h; stack_n[sp] = cnt - h; ++sp;         // second half later,
      stack_lo[sp] = lo; stack_n[sp] = h; ++sp;                   // first half next
      continue;
    }
    if (ns == 0) continue;
    // (long sequences: grouping by i and the banded shared-Peq kernel -- sq_edit.cu)
    const uint2* live = surv;
    int64_t nlive = ns;
    rc = sq_survivor_distances(a, b->packed, nB, b->max_len, surv, ns, max_d, surv2, tmp2, sdist, &live, &nlive);
    if (rc != SQ_OK) return rc;
    if (nlive == 0) continue;
    rc = sq_hit_compact(a, live, sdist, nlive, max_d, hp, hd, capacity, a->dflags);
    if (rc != SQ_OK) return rc;
  }
  SQ_CUDA(a, cudaMemcpyAsync(a->pinned, a->dflags, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(a, cudaStreamSynchronize(st));
  const int64_t hits = (int64_t)a->pinned[0];
  *n_out = hits;
  if (hits > capacity) return SQ_ERR_CAPACITY;
  if (hits == 0) return SQ_OK;
  // order by (i, j): LSD passes over the j field (bits 32..) then the i field (bits 0..)
  int shifts[8], widths[8], q = 0;
  const int nbits[2] = {bits_for(nB), bits_for(a->n)};
  for (int f = 0; f < 2; ++f)
    for (int p = 0; p < (nbits[f] + 7) / 8; ++p) {
      shifts[q] = (f == 0 ? 32 : 0) + 8 * p;
      widths[q] = (nbits[f] - 8 * p) >= 8 ? 8 : (nbits[f] - 8 * p);
      ++q;
    }
  int in_alt = 0;
  rc = sq_radix_sort(a, hp, hp_alt, hd, hd_alt, hits, 1, shifts, widths, q, tmp, &in_alt);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(a, cudaMemcpyAsync(pairs_out, in_alt ? hp_alt : hp, (size_t)hits * 8, cudaMemcpyDeviceToDevice, st));
  rc = sq_narrow_dist(a, in_alt ? hd_alt : hd, hits, dist_out);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(a, cudaStreamSynchronize(st));
  return SQ_OK;
}

int join_check(const sq_ctx* a, const sq_ctx* b, int max_d) {
  if (!a || !b) return SQ_ERR_INVALID_ARG;
  if (a->n < 0 || b->n < 0) return SQ_ERR_NOT_PACKED;
  if (a->device != b->device || a->stride != b->stride || a->alphabet != b->alphabet || a->alphabet > 32)
    return SQ_ERR_INVALID_ARG;
  if (max_d < 0) return SQ_ERR_INVALID_ARG;
  return SQ_OK;
}

}  // namespace

// rows [row0, row0 + rows) of rhA (row r is sequence a_base + r of A) against all nB columns of rhB:
// the cells whose bag distance allows d <= max_d are appended to surv (count in *counter)
int sq_bag_filter(sq_ctx* c, const uint32_t* rhA, const uint32_t* lensA, int64_t row0, int64_t rows,
                  int64_t a_base, const uint32_t* rhB, const uint32_t* lensB, int64_t nB, int max_d,
                  int upper, uint2* surv, size_t scap, unsigned long long* counter) {
  if (rows <= 0 || nB <= 0) return SQ_OK;
  if ((nB + kJoinThreads - 1) / kJoinThreads > 65535) return SQ_ERR_UNSUPPORTED;
  dim3 grid((unsigned)((rows + kJoinRows - 1) / kJoinRows), (unsigned)((nB + kJoinThreads - 1) / kJoinThreads));
  const unsigned long long sc = (unsigned long long)scap;
  if (c->alphabet <= 20)
    SQ_TIMED(c, SQ_K_ALLPAIRS, join_filter_kernel<5><<<grid, kJoinThreads, 0, c->stream>>>(
        rhA, lensA, row0, rows, a_base, rhB, lensB, nB, max_d, upper, surv, sc, counter));
  else
    SQ_TIMED(c, SQ_K_ALLPAIRS, join_filter_kernel<8><<<grid, kJoinThreads, 0, c->stream>>>(
        rhA, lensA, row0, rows, a_base, rhB, lensB, nB, max_d, upper, surv, sc, counter));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

size_t sq_join_scratch_bytes(int64_t rows, int64_t n_b, int64_t pair_capacity) {
  const size_t cap = (size_t)(pair_capacity > 0 ? pair_capacity : 1), scap = join_survivor_cap(pair_capacity);
  const size_t r = (size_t)(rows > 0 ? rows : 1), nb = (size_t)(n_b > 0 ? n_b : 1);
  return 2 * sq_align_up(cap * 8 + 16) + 2 * sq_align_up(cap * 4 + 16) + sq_sort_scratch_bytes(pair_capacity, 1) +
         sq_align_up(r * 32 + 16) + sq_align_up(r * 4 + 16) + sq_align_up(nb * 32 + 16) + sq_align_up(nb * 4 + 16) +
         2 * sq_align_up(scap * 8 + 16) + sq_align_up(scap * 2 + 16) + sq_sort_scratch_bytes((int64_t)scap, 1) +
         2 * (sq_align_up(cap * 8 + 16) + sq_align_up(cap * 2 + 16)) +          // sq_join_host staging
         2 * sq_align_up(nb * 8 + 16) + 3 * sq_align_up(nb * 4 + 16) + sq_align_up(nb * 32 + 16) +
         sq_sort_scratch_bytes(n_b, 1) +                                         // columns by length
         2 * sq_align_up(r * 8 + 16) + 3 * sq_align_up(r * 4 + 16) + sq_align_up(r * 32 + 16) +
         sq_sort_scratch_bytes(rows, 1) + 4096;                                  // rows by length
}

extern "C" int64_t sq_batch_size(int64_t n_seqs, uint64_t avail_bytes, uint32_t c, uint32_t l_max) {
  if (n_seqs < 0 || c == 0 || l_max == 0) return -1;
  const uint64_t x = avail_bytes / ((uint64_t)c * (uint64_t)l_max);
  // integer square root: the largest s with s*s <= x
  // (the floating-point root is only a starting guess; 128-bit products so that s near 2^32 is safe)
  uint64_t s = (uint64_t)sqrt((double)x);
  if (s > 0xFFFFFFFFull) s = 0xFFFFFFFFull;
  while ((unsigned __int128)s * s > x) --s;
  while ((unsigned __int128)(s + 1) * (s + 1) <= x) ++s;
  const int64_t bsz = (int64_t)(s > 32 ? s : 32);
  return n_seqs < bsz ? n_seqs : bsz;
}

extern "C" int sq_join(sq_ctx* a, const sq_ctx* b, int64_t a_begin, int64_t a_end, int max_d, int flags,
                       uint32_t* pairs_out, uint16_t* dist_out, int64_t capacity, int64_t* n_out) {
  if (!n_out) return SQ_ERR_INVALID_ARG;
  *n_out = 0;
  int rc = join_check(a, b, max_d);
  if (rc != SQ_OK) return rc;
  SqDeviceGuard guard(a);
  if (a_begin < 0 || a_end < a_begin || a_end > a->n || capacity < 0) return SQ_ERR_INVALID_ARG;
  if (capacity > 0 && (!pairs_out || !dist_out)) return SQ_ERR_INVALID_ARG;
  if (max_d > 65534) max_d = 65534;
  sq_scratch_reset(a);
  return join_core(a, b, a_begin, a_end, max_d, flags, pairs_out, dist_out, capacity, n_out);
}

extern "C" int sq_join_host(sq_ctx* a, const sq_ctx* b, int max_d, int flags, int64_t batch_rows,
                            int64_t block_capacity, uint32_t* pairs_host, uint16_t* dist_host,
                            int64_t capacity, int64_t* n_out) {
  if (!n_out) return SQ_ERR_INVALID_ARG;
  *n_out = 0;
  int rc = join_check(a, b, max_d);
  if (rc != SQ_OK) return rc;
  SqDeviceGuard guard(a);
  if (capacity < 0 || block_capacity < 1) return SQ_ERR_INVALID_ARG;
  if (capacity > 0 && (!pairs_host || !dist_host)) return SQ_ERR_INVALID_ARG;
  if (max_d > 65534) max_d = 65534;
  const int64_t nA = a->n, nB = b->n;
  if (nA == 0 || nB == 0) return SQ_OK;
  sq_scratch_reset(a);
  uint32_t* dp[2]; uint16_t* dd[2];
  for (int s = 0; s < 2; ++s) {
    dp[s] = sq_scratch<uint32_t>(a, (size_t)block_capacity * 2);
    dd[s] = sq_scratch<uint16_t>(a, (size_t)block_capacity);
    if (!dp[s] || !dd[s]) return SQ_ERR_WORKSPACE;
  }
  if (batch_rows <= 0) {
    // Eq. 12 with c = 1: a tile of B x B cells; a block of rows x n_b holds the same number of cells
    const int64_t B = sq_batch_size(nA > nB ? nA : nB, (uint64_t)(a->ws_bytes - a->scratch_top), 1,
                                    (uint32_t)(a->max_len > 0 ? a->max_len : 1));
    batch_rows = (int64_t)(((__int128)B * B) / nB);
  }
  if (batch_rows < 1) batch_rows = 1;
  if (batch_rows > nA) batch_rows = nA;
  cudaEvent_t done[2];
  for (int s = 0; s < 2; ++s) SQ_CUDA(a, cudaEventCreateWithFlags(&done[s], cudaEventDisableTiming));
  struct Ev { cudaEvent_t* e; ~Ev() { cudaEventDestroy(e[0]); cudaEventDestroy(e[1]); } } ev{done};
  bool used[2] = {false, false};
  int64_t total = 0, lo = 0, step = batch_rows;
  int slot = 0;
  int result = SQ_OK;
  while (lo < nA) {
    const int64_t hi = lo + step < nA ? lo + step : nA;
    if (used[slot]) SQ_CUDA(a, cudaEventSynchronize(done[slot]));      // its last copy has left
    int64_t hits = 0;
    rc = join_core(a, b, lo, hi, max_d, flags, dp[slot], dd[slot], block_capacity, &hits);
    if (rc == SQ_ERR_CAPACITY || rc == SQ_ERR_WORKSPACE) {
      if (hi - lo == 1) { result = rc; break; }
      step = (hi - lo) / 2;                                            // smaller blocks from here on
      continue;
    }
    if (rc != SQ_OK) { result = rc; break; }
    if (hits > 0 && total + hits <= capacity) {
      // the block is complete on a->stream (join_core synchronises): ship it beside the next block
      SQ_CUDA(a, cudaMemcpyAsync(pairs_host + 2 * total, dp[slot], (size_t)hits * 8, cudaMemcpyDeviceToHost,
                                 a->copy_stream));
      SQ_CUDA(a, cudaMemcpyAsync(dist_host + total, dd[slot], (size_t)hits * 2, cudaMemcpyDeviceToHost,
                                 a->copy_stream));
      SQ_CUDA(a, cudaEventRecord(done[slot], a->copy_stream));
      used[slot] = true;
      slot ^= 1;
    }
    total += hits;
    lo = hi;
  }
  SQ_CUDA(a, cudaStreamSynchronize(a->copy_stream));
  sq_scratch_reset(a);
  if (result != SQ_OK) return result;
  *n_out = total;
  return total > capacity ? SQ_ERR_CAPACITY : SQ_OK;
}
