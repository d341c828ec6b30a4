// sq_allpairs.cu -- step a7: exhaustive tile path over all i<j (App. F.1,
// Eq. 45: a 2-D grid over two sequence batches, here the self-join's upper triangle).
//
// A block owns one row i and a run of 256 columns j.  The row's Peq table is built ONCE per
// block, cooperatively (thread x sets the bit of position x with a shared-memory atomicOr), and
// shared by all 256 threads: "frequently accessed sequence segments are cached in
// shared memory".  Character stride is odd, so lanes reading different residues hit different
// banks and lanes reading the same residue are a broadcast.  Each thread then streams its own
// column sequence through the Myers/Hyyro column step (sq_dp.cuh).
//   max_d <  0: every distance is written to the condensed upper triangle.
//   max_d >= 0: length filter + early exit; hits are appended with warp-aggregated atomics and
//               then radix-sorted by (i,j) with the distance as payload -> deterministic order.
#include "sq_common.cuh"
#include "sq_dp.cuh"

namespace {

constexpr int kApThreads = 256;

template <int W>
__global__ void __launch_bounds__(kApThreads)
all_pairs_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n, int alphabet, int max_d,
                 uint16_t* __restrict__ dist_full, uint64_t* __restrict__ hit_pairs,
                 uint32_t* __restrict__ hit_dist, unsigned long long capacity,
                 unsigned long long* __restrict__ counter) {
  constexpr int CS = W | 1;                       // odd character stride: bank-conflict free
  __shared__ uint32_t peq[32 * CS];
  const int64_t i = blockIdx.x;
  const int64_t jbase = (int64_t)blockIdx.y * kApThreads;
  if (jbase + kApThreads <= i + 1) return;        // whole block below / on the diagonal
  const uint8_t* rowA = packed + i * stride;
  const int m = rowA[stride - 1];
  for (int t = threadIdx.x; t < 32 * CS; t += kApThreads) peq[t] = 0u;
  __syncthreads();
  if ((int)threadIdx.x < m) {
    const uint32_t ch = rowA[threadIdx.x];
    atomicOr(&peq[ch * CS + (threadIdx.x >> 5)], 1u << (threadIdx.x & 31));
  }
  __syncthreads();
  const int64_t j = jbase + threadIdx.x;
  const bool active = j > i && j < n;
  int d = 0;
  if (active) {
    const uint8_t* rowB = packed + j * stride;
    const int nlen = rowB[stride - 1];
    const int diff = m > nlen ? m - nlen : nlen - m;
    if (max_d >= 0 && diff > max_d) d = max_d + 1;
    else if (m == 0) d = nlen;
    else if (nlen == 0) d = m;
    else d = sq_myers<W>(peq, CS, 1, m, rowB, nlen, max_d);
    if (max_d >= 0 && d > max_d) d = max_d + 1;
  }
  if (max_d < 0) {
    if (active) dist_full[i * (2 * n - i - 1) / 2 + (j - i - 1)] = (uint16_t)d;
    return;
  }
  const bool hit = active && d <= max_d;
  const uint32_t mask = __ballot_sync(0xFFFFFFFFu, hit);
  if (mask) {
    const int lane = threadIdx.x & 31;
    unsigned long long base = 0;
    if (lane == __ffs(mask) - 1) base = atomicAdd(counter, (unsigned long long)__popc(mask));
    base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
    if (hit) {
      const unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
      if (slot < capacity) {
        hit_pairs[slot] = (uint64_t)(uint32_t)i | ((uint64_t)(uint32_t)j << 32);
        hit_dist[slot] = (uint32_t)d;
      }
    }
  }
}


// ---- thresholded path, phase 1: the bag-distance filter -----------------------------------------
// d(a, b) >= bag(a, b) = max(|A minus B|, |B minus A|) over the residue multisets = (L1 + |m - n|) / 2
// with L1 the L1 distance of the residue histograms: an edit changes one count by one (indel) or
// two counts by one each (substitution).  A pair whose bag distance exceeds max_d cannot be a hit,
// so it is dropped before any DP.  The histograms (<= 32 residues, one byte each: 8 words) are
// compared with byte-wise sum-of-absolute-differences instructions (sq_join.cu: sq_bag_filter).
__global__ void __launch_bounds__(256)
residue_hist_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n,
                    uint32_t* __restrict__ rh, uint32_t* __restrict__ lens) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t* __restrict__ row = reinterpret_cast<const uint32_t*>(packed + i * stride);
  const int nw = stride >> 2;
  const uint32_t lastw = row[nw - 1];
  lens[i] = lastw >> 24;
  uint32_t h[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int wi = 0; wi < nw; ++wi) {
    uint32_t word = row[wi];
    if (wi == nw - 1) word |= 0xFF000000u;                 // the length byte is not a residue
    if (word == 0xFFFFFFFFu) continue;                     // padding only
#pragma unroll
    for (int c = 0; c < 32; ++c) {
      const uint32_t eq = __vcmpeq4(word, (uint32_t)c * 0x01010101u);   // 0xFF per equal byte
      h[c >> 2] += (__popc(eq) >> 3) << (8 * (c & 3));
    }
  }
#pragma unroll
  for (int q = 0; q < 8; ++q) rh[i * 8 + q] = h[q];
}

// phase 3: the survivors that are hits, as (i | j << 32, d) records for the final ordering
__global__ void __launch_bounds__(256)
hit_compact_kernel(const uint2* __restrict__ surv, const uint16_t* __restrict__ sdist, int64_t ns,
                   int max_d, uint64_t* __restrict__ hit_pairs, uint32_t* __restrict__ hit_dist,
                   unsigned long long capacity, unsigned long long* __restrict__ counter) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int d = p < ns ? (int)sdist[p] : 0xFFFF;
  const bool hit = p < ns && d <= max_d;
  const uint32_t mask = __ballot_sync(0xFFFFFFFFu, hit);
  if (mask) {
    const int lane = threadIdx.x & 31;
    unsigned long long base = 0;
    if (lane == __ffs(mask) - 1) base = atomicAdd(counter, (unsigned long long)__popc(mask));
    base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
    if (hit) {
      const unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
      if (slot < capacity) {
        const uint2 pr = surv[p];
        hit_pairs[slot] = (uint64_t)pr.x | ((uint64_t)pr.y << 32);
        hit_dist[slot] = (uint32_t)d;
      }
    }
  }
}

__global__ void narrow_dist_kernel(const uint32_t* __restrict__ in, int64_t n,
                                   uint16_t* __restrict__ out) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) out[p] = (uint16_t)in[p];
}

template <int W>
int launch_all_pairs(sq_ctx* c, int max_d, uint16_t* dist_full, uint64_t* hp, uint32_t* hd,
                     int64_t capacity) {
  const int64_t n = c->n;
  dim3 grid((unsigned)n, (unsigned)((n + kApThreads - 1) / kApThreads));
  SQ_TIMED(c, SQ_K_ALLPAIRS, all_pairs_kernel<W><<<grid, kApThreads, 0, c->stream>>>(
      c->packed, c->stride, n, c->alphabet, max_d, dist_full, hp, hd,
      (unsigned long long)capacity, c->dflags));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

inline int bits_for(int64_t n) {
  int b = 1;
  while (b < 32 && (1ll << b) < n) ++b;
  return b;
}

}  // namespace

// launchers shared with sq_join.cu
int sq_residue_hist(sq_ctx* c, const uint8_t* packed, int stride, int64_t n, uint32_t* rh, uint32_t* lens) {
  if (n <= 0) return SQ_OK;
  SQ_TIMED(c, SQ_K_ALLPAIRS, residue_hist_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(
      packed, stride, n, rh, lens));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int sq_hit_compact(sq_ctx* c, const uint2* surv, const uint16_t* sdist, int64_t ns, int max_d,
                   uint64_t* hit_pairs, uint32_t* hit_dist, int64_t capacity, unsigned long long* counter) {
  if (ns <= 0) return SQ_OK;
  SQ_TIMED(c, SQ_K_ALLPAIRS, hit_compact_kernel<<<(unsigned)((ns + 255) / 256), 256, 0, c->stream>>>(
      surv, sdist, ns, max_d, hit_pairs, hit_dist, (unsigned long long)capacity, counter));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int sq_narrow_dist(sq_ctx* c, const uint32_t* in, int64_t n, uint16_t* out) {
  if (n <= 0) return SQ_OK;
  SQ_TIMED(c, SQ_K_MISC, narrow_dist_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(in, n, out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

// survivors of the bag-distance filter the scratch is sized for (more -> the fused kernel runs)
static inline size_t sq_survivor_cap(int64_t pair_capacity) {
  return 4 * (size_t)(pair_capacity > 0 ? pair_capacity : 1) + 65536;
}

size_t sq_allpairs_scratch_bytes(int64_t n, int64_t pair_capacity) {
  size_t cap = (size_t)(pair_capacity > 0 ? pair_capacity : 1);
  size_t nn = (size_t)(n > 0 ? n : 1), scap = sq_survivor_cap(pair_capacity);
  return 2 * sq_align_up(cap * 8 + 16) + 2 * sq_align_up(cap * 4 + 16) +
         sq_sort_scratch_bytes(pair_capacity, 1) +
         sq_align_up(nn * 32 + 16) + sq_align_up(nn * 4 + 16) +          // histograms, lengths
         2 * sq_align_up(scap * 8 + 16) + sq_align_up(scap * 2 + 16) +        // survivors (x2), distances
         sq_sort_scratch_bytes((int64_t)scap, 1) + 4096;
}

extern "C" int sq_all_pairs(sq_ctx* c, int max_d, uint32_t* pairs_out, uint16_t* dist_out,
                            int64_t capacity, int64_t* n_out) {
  if (!c || !n_out) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  *n_out = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  const int64_t n = c->n;
  if (capacity < 0) return SQ_ERR_INVALID_ARG;
  if (n < 2) return SQ_OK;
  if ((n + kApThreads - 1) / kApThreads > 65535) return SQ_ERR_UNSUPPORTED;
  if (max_d > 65534) max_d = -1;
  const int words = (c->max_len + 31) / 32;
  const int64_t npairs = n * (n - 1) / 2;
  cudaStream_t st = c->stream;
  uint64_t* hp = nullptr; uint64_t* hp_alt = nullptr; uint32_t* hd = nullptr; uint32_t* hd_alt = nullptr;
  uint8_t* tmp = nullptr;
  if (max_d < 0) {
    if (!dist_out) return SQ_ERR_INVALID_ARG;
    *n_out = npairs;
    if (capacity < npairs) return SQ_ERR_CAPACITY;
  } else {
    if (capacity >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;
    if (capacity > 0 && (!pairs_out || !dist_out)) return SQ_ERR_INVALID_ARG;
    sq_scratch_reset(c);
    const size_t cap = (size_t)(capacity > 0 ? capacity : 1);
    hp = sq_scratch<uint64_t>(c, cap);
    hp_alt = sq_scratch<uint64_t>(c, cap);
    hd = sq_scratch<uint32_t>(c, cap);
    hd_alt = sq_scratch<uint32_t>(c, cap);
    tmp = sq_scratch<uint8_t>(c, sq_sort_scratch_bytes(capacity, 1));
    if (!hp || !hp_alt || !hd || !hd_alt || !tmp) return SQ_ERR_WORKSPACE;
    SQ_CUDA(c, cudaMemsetAsync(c->dflags, 0, 64, st));
  }
  int rc;
  bool filtered = false;
  if (max_d >= 0) {
    // phases 1-3: bag-distance filter -> DP on the survivors only -> hits.  If the survivors do
    // not fit their scratch, the fused kernel below does the whole job instead.
    const size_t scap = sq_survivor_cap(capacity);
    uint32_t* rh = sq_scratch<uint32_t>(c, (size_t)n * 8);
    uint32_t* lens = sq_scratch<uint32_t>(c, (size_t)n);
    uint2* surv = sq_scratch<uint2>(c, scap);
    uint16_t* sdist = sq_scratch<uint16_t>(c, scap);
    uint2* surv2 = sq_scratch<uint2>(c, scap);
    uint8_t* tmp2 = sq_scratch<uint8_t>(c, sq_sort_scratch_bytes((int64_t)scap, 1));
    if (rh && lens && surv && sdist && surv2 && tmp2 && c->alphabet <= 32) {
      SQ_TIMED(c, SQ_K_ALLPAIRS, residue_hist_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(
          c->packed, c->stride, n, rh, lens));
      SQ_LAUNCH_CHECK(c);
      // (the filter kernel is the join's, sq_join.cu: the column's histogram in registers, 16 rows'
      // histograms in shared memory; blocks below the diagonal return at once)
      rc = sq_bag_filter(c, rh, lens, 0, n, 0, rh, lens, n, max_d, 1, surv, scap, c->dflags + 1);
      if (rc != SQ_OK) return rc;
      SQ_CUDA(c, cudaMemcpyAsync(c->pinned, c->dflags + 1, 8, cudaMemcpyDeviceToHost, st));
      SQ_CUDA(c, cudaStreamSynchronize(st));
      const int64_t ns = (int64_t)c->pinned[0];
      c->last_raw_pairs = ns;                    // survivors of the filter (sq_last_raw_pairs)
      if ((size_t)ns <= scap) {
        filtered = true;
        if (ns > 0) {
          // (long sequences: grouping by i and the banded shared-Peq kernel -- sq_edit.cu)
          const uint2* live = surv;
          int64_t nlive = ns;
          rc = sq_survivor_distances(c, c->packed, n, c->max_len, surv, ns, max_d, surv2, tmp2, sdist, &live,
                                     &nlive);
          if (rc != SQ_OK) return rc;
          if (nlive > 0) {
            SQ_TIMED(c, SQ_K_ALLPAIRS, hit_compact_kernel<<<(unsigned)((nlive + 255) / 256), 256, 0, st>>>(
                live, sdist, nlive, max_d, hp, hd, (unsigned long long)capacity, c->dflags));
            SQ_LAUNCH_CHECK(c);
          }
        }
      }
    }
  }
  if (filtered) rc = SQ_OK;
  else if (words <= 1) rc = launch_all_pairs<1>(c, max_d, dist_out, hp, hd, capacity);
  else if (words <= 2) rc = launch_all_pairs<2>(c, max_d, dist_out, hp, hd, capacity);
  else if (words <= 4) rc = launch_all_pairs<4>(c, max_d, dist_out, hp, hd, capacity);
  else if (words <= 5) rc = launch_all_pairs<5>(c, max_d, dist_out, hp, hd, capacity);
  else if (words <= 8) rc = launch_all_pairs<8>(c, max_d, dist_out, hp, hd, capacity);
  else rc = SQ_ERR_UNSUPPORTED;
  if (rc != SQ_OK) return rc;
  if (max_d < 0) {
    SQ_CUDA(c, cudaStreamSynchronize(st));
    return SQ_OK;
  }
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, c->dflags, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t hits = (int64_t)c->pinned[0];
  *n_out = hits;
  if (hits > capacity) return SQ_ERR_CAPACITY;
  if (hits == 0) return SQ_OK;
  // order the hits by (i, j): LSD radix sort on the j field then the i field, payload = distance
  const int nb = bits_for(n), per_field = (nb + 7) / 8;
  int shifts[8], widths[8], q = 0;
  for (int f = 0; f < 2; ++f)
    for (int p = 0; p < per_field; ++p) {
      shifts[q] = (f == 0 ? 32 : 0) + 8 * p;
      widths[q] = (nb - 8 * p) >= 8 ? 8 : (nb - 8 * p);
      ++q;
    }
  int in_alt = 0;
  rc = sq_radix_sort(c, hp, hp_alt, hd, hd_alt, hits, 1, shifts, widths, q, tmp, &in_alt);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(pairs_out, in_alt ? hp_alt : hp, (size_t)hits * 8,
                             cudaMemcpyDeviceToDevice, st));
  SQ_TIMED(c, SQ_K_MISC, narrow_dist_kernel<<<(unsigned)((hits + 255) / 256), 256, 0, st>>>(
      in_alt ? hd_alt : hd, hits, dist_out));
  SQ_LAUNCH_CHECK(c);
  SQ_CUDA(c, cudaStreamSynchronize(st));
  return SQ_OK;
}
