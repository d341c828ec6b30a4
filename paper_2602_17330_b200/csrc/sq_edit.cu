// sq_edit.cu -- step a6: batched exact Levenshtein distance on an explicit pair list
// (App. F.3: "for each sequence pair processed by an individual thread",
// recurrence Eq. 46).  One thread per pair, Myers/Hyyro bit-parallel DP (sq_dp.cuh) instead of
// the paper's cell-by-cell DP; 32-bit words, W = ceil(max_len/32) words per column.
#include "sq_common.cuh"
#include "sq_dp.cuh"

namespace {

template <int W, bool BANDED>
__global__ void edit_pairs_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n,
                                  const uint8_t* __restrict__ packedB, int64_t nB,
                                  const uint2* __restrict__ pairs, int64_t n_pairs, int max_d,
                                  int alphabet, uint16_t* __restrict__ dist) {
  extern __shared__ uint32_t peq_smem[];
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_pairs) return;
  const uint2 pr = pairs[p];
  if (pr.x >= (uint64_t)n || pr.y >= (uint64_t)nB) { dist[p] = 0xFFFFu; return; }
  const int d = sq_pair_distance<W, BANDED>(packed + (int64_t)pr.x * stride, packedB + (int64_t)pr.y * stride,
                                    stride, alphabet, max_d, peq_smem + threadIdx.x, blockDim.x);
  dist[p] = (uint16_t)d;
}


// ---- single-word fast path: every sequence fits one 32-bit word (max_len <= 31) ---------------
// A warp takes 32 consecutive pairs.  sq_lsh_candidates emits pairs grouped by i, so the lanes
// of a warp share a few distinct patterns i ("runs"): the Peq table of every run is built ONCE,
// cooperatively (lane x holds residue x of the pattern; match.any gives the bit mask of every
// residue in one instruction), and kept in shared memory [run][33] (odd stride: lanes of
// different runs hit different banks, lanes of one run reading one residue are a broadcast).
// Each lane then streams its own text j (one or two 16-byte loads, held in registers) through
// the Myers/Hyyro column step; the distance is read off the final vertical deltas:
// D[m][n] = n + popc(Pv) - popc(Mv) over the m pattern bits, so no score is tracked per column.
constexpr int kEdWarps = 8;
constexpr int kEdRuns = 8;      // Peq tables resident per warp

// SCHED: warp k takes positions [32k, 32k+32) of the family-ordered schedule left by
// sq_lsh_candidates (sq_common.cuh) instead of pairs [32k, 32k+32): consecutive warps then work
// on rows of the same family, whose partners are the same few sequences -- the text gathers hit
// L2.  The schedule only permutes the pair indices; every pair is still read from `pairs`.
template <int STRIDE, bool SCHED>
__global__ void __launch_bounds__(kEdWarps * 32, 5)
edit_pairs_w1_kernel(const uint8_t* __restrict__ packed, int64_t n,
                     const uint8_t* __restrict__ packedB, int64_t nB, const uint2* __restrict__ pairs,
                     int64_t n_pairs, int max_d, uint16_t* __restrict__ dist,
                     const uint4* __restrict__ sched, const uint32_t* __restrict__ rowstart,
                     const uint32_t* __restrict__ delta) {
  constexpr int WORDS = STRIDE / 4;
  __shared__ uint32_t peq_sm[kEdWarps][kEdRuns * 33];
  __shared__ uint32_t mlen_sm[kEdWarps][kEdRuns];
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t wk = (int64_t)blockIdx.x * kEdWarps + w;
  int64_t p = wk * 32 + lane;
  bool valid = p < n_pairs;
  if (SCHED && valid) {
    const uint4 ch = sched[wk];                       // (first row, its delta, end of that row)
    const uint32_t q = (uint32_t)p;
    if (q < ch.z) p = (int64_t)(uint32_t)(ch.y + q);
    else {
      uint32_t r = ch.x + 1;
      while (q >= rowstart[r + 1]) ++r;               // empty rows are stepped over
      p = (int64_t)(uint32_t)(delta[r] + q);
    }
  }
  uint2 pr = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
  if (valid) pr = pairs[p];
  const bool inrange = valid && pr.x < (uint64_t)n && pr.y < (uint64_t)nB;
  const uint32_t i = inrange ? pr.x : 0xFFFFFFFFu;
  // the text is independent of the runs: issue its load first
  uint32_t tw[WORDS];
  {
    const uint4* rowB = reinterpret_cast<const uint4*>(packedB + (int64_t)(inrange ? pr.y : 0u) * STRIDE);
#pragma unroll
    for (int q = 0; q < WORDS / 4; ++q) {
      const uint4 v = inrange ? rowB[q] : make_uint4(0, 0, 0, 0);
      tw[4 * q] = v.x; tw[4 * q + 1] = v.y; tw[4 * q + 2] = v.z; tw[4 * q + 3] = v.w;
    }
  }
  // runs of equal i
  const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, i, 1);
  const bool head = lane == 0 || i != prev;
  const uint32_t hm = __ballot_sync(0xFFFFFFFFu, head);
  const uint32_t run = __popc(hm & (0xFFFFFFFFu >> (31 - lane))) - 1;
  const int nruns = __popc(hm);
  uint32_t* peq = peq_sm[w];
  uint32_t rem = hm;
  const int nlen = (int)(tw[WORDS - 1] >> 24);
  int d = 0;
  // kEdRuns Peq tables fit at a time; a warp with more runs (many tiny rows) takes several rounds
#pragma unroll 1
  for (int rbase = 0; rbase < nruns; rbase += kEdRuns) {
    const int nr = min(kEdRuns, nruns - rbase);
    __syncwarp();
#pragma unroll 1
    for (int r = 0; r < nr; ++r) {
      const int hl = __ffs(rem) - 1;
      rem &= rem - 1;
      const uint32_t ir = __shfl_sync(0xFFFFFFFFu, i, hl);
      uint32_t ch = 0xFFu;
      if (ir != 0xFFFFFFFFu && lane < (uint32_t)STRIDE) ch = packed[(int64_t)ir * STRIDE + lane];
      const uint32_t m = ir != 0xFFFFFFFFu ? __shfl_sync(0xFFFFFFFFu, ch, STRIDE - 1) : 0u;
      peq[r * 33 + lane] = 0u;
      __syncwarp();
      const uint32_t mm = __match_any_sync(0xFFFFFFFFu, ch);
      if (lane < m) peq[r * 33 + ch] = mm & ((1u << m) - 1u);     // m <= 31
      if (lane == 0) mlen_sm[w][r] = m;
    }
    __syncwarp();
    if (!inrange || (int)run < rbase || (int)run >= rbase + nr) continue;
    const int m = (int)mlen_sm[w][run - rbase];
    const int diff = m > nlen ? m - nlen : nlen - m;
    if (max_d >= 0 && diff > max_d) d = max_d + 1;
    else if (m == 0) d = nlen;
    else if (nlen == 0) d = m;
    else {
      // byte address of this run's table in shared memory: one multiply-add per column gives the
      // address of Peq[residue], and (Ph << 1) | 1 is one multiply-add as well (both FMA pipe)
      const uint32_t pq = (uint32_t)__cvta_generic_to_shared(peq + (run - rbase) * 33);
      uint32_t Pv = 0xFFFFFFFFu, Mv = 0u;
#pragma unroll
      for (int wi = 0; wi < WORDS; ++wi) {
        if (4 * wi < nlen) {
          const uint32_t word = tw[wi];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            if (4 * wi + q < nlen) {
              uint32_t Eq;
              // (not volatile, so the loads of a word can be issued ahead of the DP chain; the
              // dummy input m -- read from shared memory after the warp barrier -- keeps them
              // behind the barrier that publishes the table)
              asm("ld.shared.u32 %0, [%1];" : "=r"(Eq) : "r"(((word >> (8 * q)) & 0xFFu) * 4u + pq), "r"(m));
              const uint32_t Xv = Eq | Mv;
              const uint32_t Xh = (((Eq & Pv) + Pv) ^ Pv) | Eq;
              uint32_t Ph = Mv | ~(Xh | Pv);
              uint32_t Mh = Pv & Xh;
              asm("mad.lo.u32 %0, %0, 2, 1;" : "+r"(Ph));
              Mh <<= 1;
              Pv = Mh | ~(Xv | Ph);
              Mv = Ph & Xv;
            }
          }
        }
      }
      const uint32_t mask = (1u << m) - 1u;                        // m <= 31
      d = nlen + __popc(Pv & mask) - __popc(Mv & mask);
    }
  }
  if (!valid) return;
  if (!inrange) { dist[p] = 0xFFFFu; return; }
  if (max_d >= 0 && d > max_d) d = max_d + 1;
  dist[p] = (uint16_t)d;
}

template <int STRIDE>
int launch_edit_w1(sq_ctx* c, const uint8_t* packedB, int64_t nB, const uint32_t* pairs, int64_t n_pairs,
                   int max_d, uint16_t* dist_out) {
  const int64_t per_block = kEdWarps * 32;
  // the schedule pays off only when the packed sequences do not fit the L2 anyway
  const bool big = (size_t)c->n * (size_t)c->stride > ((size_t)96 << 20);
  if (packedB == c->packed && big && c->sched && c->sched_pairs == pairs && c->sched_npairs == n_pairs && c->sched_chunks > 0) {
    const int64_t blocks = (c->sched_chunks + kEdWarps - 1) / kEdWarps;
    SQ_TIMED(c, SQ_K_EDIT, edit_pairs_w1_kernel<STRIDE, true><<<(unsigned)blocks, kEdWarps * 32, 0, c->stream>>>(
        c->packed, c->n, c->packed, c->n, reinterpret_cast<const uint2*>(pairs), n_pairs, max_d, dist_out,
        c->sched, c->sched_rowstart, c->sched_delta));
    SQ_LAUNCH_CHECK(c);
    return SQ_OK;
  }
  const int64_t blocks = (n_pairs + per_block - 1) / per_block;
  SQ_TIMED(c, SQ_K_EDIT, edit_pairs_w1_kernel<STRIDE, false><<<(unsigned)blocks, kEdWarps * 32, 0, c->stream>>>(
      c->packed, c->n, packedB, nB, reinterpret_cast<const uint2*>(pairs), n_pairs, max_d, dist_out, nullptr,
      nullptr, nullptr));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

template <int W, bool BANDED>
int launch_edit_wb(sq_ctx* c, const uint8_t* packedB, int64_t nB, const uint32_t* pairs, int64_t n_pairs,
                   int max_d, uint16_t* dist_out) {
  const int threads = W <= 2 ? 256 : 128;
  const size_t smem = (size_t)c->alphabet * W * threads * sizeof(uint32_t);
  if (smem > 48 * 1024)
    SQ_CUDA(c, cudaFuncSetAttribute(edit_pairs_kernel<W, BANDED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)smem));
  const int64_t blocks = (n_pairs + threads - 1) / threads;
  SQ_TIMED(c, SQ_K_EDIT, edit_pairs_kernel<W, BANDED><<<(unsigned)blocks, threads, smem, c->stream>>>(
      c->packed, c->stride, c->n, packedB, nB, reinterpret_cast<const uint2*>(pairs), n_pairs, max_d,
      c->alphabet, dist_out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

template <int W>
int launch_edit(sq_ctx* c, const uint8_t* packedB, int64_t nB, const uint32_t* pairs, int64_t n_pairs,
                int max_d, uint16_t* dist_out, bool banded) {
  // the band only pays when it is narrower than the words
  if (banded && W > 1 && max_d >= 0 && 2 * max_d + 1 < 32 * (W - 1))
    return launch_edit_wb<W, true>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  return launch_edit_wb<W, false>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
}

// ---- long sequences under a threshold: a cheap look at the first columns ----------------------
// Every alignment path leaves column C through some cell (x, C), and from there to (m, n) it
// costs at least |(m - x) - (n - C)|, so  D[m][n] >= min_x ( D[x][C] + |(m - x) - (n - C)| ).
// Rows x > 64 of column C have D >= x - C > max_d when C < 64 - max_d, so the minimum over the
// rows of the first two words decides: if it exceeds max_d the pair cannot be a hit and the full
// multi-word DP (4-8 words x 100+ columns) is never run for it.  One thread per pair, a two-word
// Myers/Hyyro column for C columns, then one walk down the column.  Pairs that may still be hits
// are compacted (warp-aggregated append) for the full kernel.
constexpr int kPfThreads = 256;

__global__ void __launch_bounds__(kPfThreads)
dp_prefilter_kernel(const uint8_t* __restrict__ packedA, const uint8_t* __restrict__ packedB, int stride,
                    int64_t nA, int64_t nB, const uint2* __restrict__ surv, int64_t ns, int max_d,
                    int alphabet, int C, uint2* __restrict__ alive_out,
                    unsigned long long* __restrict__ counter) {
  extern __shared__ uint32_t peq_smem[];               // [alphabet][2][kPfThreads]
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = p < ns;
  bool alive = valid;
  uint2 pr = make_uint2(0u, 0u);
  if (valid) {
    pr = surv[p];
    if (pr.x < (uint64_t)nA && pr.y < (uint64_t)nB) {
      const uint8_t* rowA = packedA + (int64_t)pr.x * stride;
      const uint8_t* rowB = packedB + (int64_t)pr.y * stride;
      const int m = rowA[stride - 1], n = rowB[stride - 1];
      if (n >= C && m >= 1) {
        const int mr = m < 64 ? m : 64;                // pattern rows held in the two words
        uint32_t* peq = peq_smem + threadIdx.x;
        sq_peq_build<2>(rowA, mr, alphabet, peq, kPfThreads);
        uint32_t Pv0 = 0xFFFFFFFFu, Pv1 = 0xFFFFFFFFu, Mv0 = 0u, Mv1 = 0u;
        const uint32_t* b32 = reinterpret_cast<const uint32_t*>(rowB);
        for (int y0 = 0; y0 < C; y0 += 4) {
          const uint32_t word = b32[y0 >> 2];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            if (y0 + q < C) {
              const uint32_t ch = (word >> (8 * q)) & 0xFFu;
              const uint32_t Eq0 = peq[(ch * 2) * kPfThreads], Eq1 = peq[(ch * 2 + 1) * kPfThreads];
              // word 0
              const uint32_t Xv0 = Eq0 | Mv0;
              const uint64_t s0 = (uint64_t)(Eq0 & Pv0) + (uint64_t)Pv0;
              const uint32_t Xh0 = ((uint32_t)s0 ^ Pv0) | Eq0;
              uint32_t Ph0 = Mv0 | ~(Xh0 | Pv0), Mh0 = Pv0 & Xh0;
              const uint32_t pc = Ph0 >> 31, mc = Mh0 >> 31;
              Ph0 = (Ph0 << 1) | 1u; Mh0 <<= 1;
              Pv0 = Mh0 | ~(Xv0 | Ph0); Mv0 = Ph0 & Xv0;
              // word 1 (carry of the addition and of the two shifts comes from word 0)
              const uint32_t Xv1 = Eq1 | Mv1;
              const uint32_t s1 = (Eq1 & Pv1) + Pv1 + (uint32_t)(s0 >> 32);
              const uint32_t Xh1 = (s1 ^ Pv1) | Eq1;
              uint32_t Ph1 = Mv1 | ~(Xh1 | Pv1), Mh1 = Pv1 & Xh1;
              Ph1 = (Ph1 << 1) | pc; Mh1 = (Mh1 << 1) | mc;
              Pv1 = Mh1 | ~(Xv1 | Ph1); Mv1 = Ph1 & Xv1;
            }
          }
        }
        // walk down column C: D[0][C] = C
        const int rem_n = n - C;
        int D = C;
        int best = D + (m > rem_n ? m - rem_n : rem_n - m);
        const int xmax = mr < C + max_d ? mr : C + max_d;      // deeper rows have D > max_d
        const uint64_t Pv = (uint64_t)Pv0 | ((uint64_t)Pv1 << 32), Mv = (uint64_t)Mv0 | ((uint64_t)Mv1 << 32);
        for (int x = 1; x <= xmax; ++x) {
          D += (int)((Pv >> (x - 1)) & 1ull) - (int)((Mv >> (x - 1)) & 1ull);
          const int rm = m - x;
          const int cand = D + (rm > rem_n ? rm - rem_n : rem_n - rm);
          best = cand < best ? cand : best;
        }
        alive = best <= max_d;
      }
    }
  }
  const uint32_t mask = __ballot_sync(0xFFFFFFFFu, alive);
  if (mask) {
    const int lane = threadIdx.x & 31;
    unsigned long long base = 0;
    if (lane == __ffs(mask) - 1) base = atomicAdd(counter, (unsigned long long)__popc(mask));
    base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
    if (alive) alive_out[base + __popc(mask & ((1u << lane) - 1u))] = pr;
  }
}

}  // namespace

// pairs (i, j): i indexes the context's own pack, j indexes `packedB` (nB slots of the same stride
// and alphabet, at most max_len_b residues each); packedB == c->packed is the ordinary self case
int sq_edit_distance_ab(sq_ctx* c, const uint8_t* packedB, int64_t nB, int max_len_b,
                        const uint32_t* pairs, int64_t n_pairs, int max_d, uint16_t* dist_out,
                        bool banded) {
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (n_pairs < 0) return SQ_ERR_INVALID_ARG;
  if (n_pairs == 0) return SQ_OK;
  if (!pairs || !dist_out || !packedB) return SQ_ERR_INVALID_ARG;
  if (n_pairs >= (1ll << 31) * 128) return SQ_ERR_UNSUPPORTED;
  if (max_d > 65534) max_d = -1;
  if (c->stride == 16) return launch_edit_w1<16>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  if (c->stride == 32) return launch_edit_w1<32>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  const int ml = c->max_len > max_len_b ? c->max_len : max_len_b;
  const int words = (ml + 31) / 32;
  if (words <= 1) return launch_edit<1>(c, packedB, nB, pairs, n_pairs, max_d, dist_out, banded);
  if (words <= 2) return launch_edit<2>(c, packedB, nB, pairs, n_pairs, max_d, dist_out, banded);
  if (words <= 4) return launch_edit<4>(c, packedB, nB, pairs, n_pairs, max_d, dist_out, banded);
  if (words <= 5) return launch_edit<5>(c, packedB, nB, pairs, n_pairs, max_d, dist_out, banded);
  if (words <= 8) return launch_edit<8>(c, packedB, nB, pairs, n_pairs, max_d, dist_out, banded);
  return SQ_ERR_UNSUPPORTED;
}

// Survivors of a coarse filter -> those that can still be within max_d (see dp_prefilter_kernel).
// Returns 1 through *applied when the look-ahead ran (alive pairs in alive_out, their number in
// *counter on the device), 0 when it does not apply (short sequences, large max_d).
int sq_dp_prefilter(sq_ctx* c, const uint8_t* packedB, int64_t nB, int max_len_b, const uint2* surv,
                    int64_t ns, int max_d, uint2* alive_out, unsigned long long* counter, int* applied) {
  *applied = 0;
  const int ml = c->max_len > max_len_b ? c->max_len : max_len_b;
  if (ml <= 64 || max_d < 0 || max_d > 31 || ns <= 0) return SQ_OK;
  const int C = 64 - max_d - 1 < 48 ? 64 - max_d - 1 : 48;
  const size_t smem = (size_t)c->alphabet * 2 * kPfThreads * sizeof(uint32_t);
  if (smem > 48 * 1024)
    SQ_CUDA(c, cudaFuncSetAttribute(dp_prefilter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  SQ_TIMED(c, SQ_K_EDIT, dp_prefilter_kernel<<<(unsigned)((ns + kPfThreads - 1) / kPfThreads), kPfThreads, smem, c->stream>>>(
      c->packed, packedB, c->stride, c->n, nB, surv, ns, max_d, c->alphabet, C, alive_out, counter));
  SQ_LAUNCH_CHECK(c);
  *applied = 1;
  return SQ_OK;
}

int sq_edit_distance_impl(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                          uint16_t* dist_out) {
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  return sq_edit_distance_ab(c, c->packed, c->n, c->max_len, pairs, n_pairs, max_d, dist_out, false);
}
