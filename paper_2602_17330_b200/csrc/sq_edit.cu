// sq_edit.cu -- step a6: batched exact Levenshtein distance on an explicit pair list
// (App. F.3: "for each sequence pair processed by an individual thread",
// recurrence Eq. 46).  One thread per pair, Myers/Hyyro bit-parallel DP (sq_dp.cuh) instead of
// the paper's cell-by-cell DP; 32-bit words, W = ceil(max_len/32) words per column.
#include "sq_common.cuh"
#include "sq_dp.cuh"

namespace {

template <int W>
__global__ void edit_pairs_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n,
                                  const uint8_t* __restrict__ packedB, int64_t nB,
                                  const uint2* __restrict__ pairs, int64_t n_pairs, int max_d,
                                  int alphabet, uint16_t* __restrict__ dist) {
  extern __shared__ uint32_t peq_smem[];
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_pairs) return;
  const uint2 pr = pairs[p];
  if (pr.x >= (uint64_t)n || pr.y >= (uint64_t)nB) { dist[p] = 0xFFFFu; return; }
  const int d = sq_pair_distance<W>(packed + (int64_t)pr.x * stride, packedB + (int64_t)pr.y * stride,
                                    stride, alphabet, max_d, peq_smem + threadIdx.x, blockDim.x);
  dist[p] = (uint16_t)d;
}


// ---- single-word fast path: every sequence fits one 32-bit word (max_len <= 31) ---------------
// A warp takes 32 consecutive pairs.  sq_lsh_candidates emits pairs grouped by i, so the lanes
// of a warp share a few distinct patterns i ("runs"): the Peq table of every run is built ONCE,
// cooperatively (lane x holds residue x of the pattern; match.any gives the bit mask of every
// residue in one instruction), and kept in shared memory [run][33] (odd stride: lanes of
// different runs hit different banks, lanes of one run reading one residue are a broadcast).
// Each lane then streams its own text j through the Myers/Hyyro column step.  The text slot arrives
// by one 256-bit load and is PARKED IN SHARED MEMORY, word-interleaved [word][lane]: a column reads
// its residue with one conflict-free LDS.U8 and turns it into the table address with one
// multiply-add (FMA pipe) -- no shift / mask on the ALU pipe, which is the pipe that bounds the
// loop, and no 32 pre-extracted residues in registers (47 -> 31 registers: 64 resident warps per SM
// instead of 40).  Round 2: 36.2 -> 29.5 ms at config 4.  The distance is read off the final vertical deltas:
// D[m][n] = n + popc(Pv) - popc(Mv) over the m pattern bits, so no score is tracked per column.
constexpr int kEdWarps = 2;     // small blocks: a warp's time varies (runs, text lengths, load chain), and a
                                // block holds its slot until its slowest warp is done (8 -> 2 warps: -5 %)
constexpr int kEdRuns = 8;      // Peq tables resident per warp

// SCHED: warp k takes positions [32k, 32k+32) of the family-ordered schedule left by
// sq_lsh_candidates (sq_common.cuh) instead of pairs [32k, 32k+32): consecutive warps then work
// on rows of the same family, whose partners are the same few sequences -- the text gathers hit
// L2.  The schedule only permutes the pair indices; every pair is still read from `pairs`.
// One column of the single-word chain on the fast path (below).  Every column is entered by the
// warp-uniform indexed jump, i.e. it is a basic block of its own and the assembler moves no load
// across its border -- so the loads are pipelined by hand: column U computes on the table word
// fetched by column U - 1, fetches the word of column U + 1 (address = one multiply-add on the
// FMA pipe) and the residue of column U + 2 (LDS.U8 at a compile-time offset).  13 instructions:
// 2 shared loads, 7 logic ops (ALU pipe), the address, the add and the two shifts as multiply-adds
// (FMA pipe); no branch, no predicate.  Even columns compute on EqA and fetch into EqB, odd ones the
// other way round (no register move).
#define SQ_W1_COL(U, Eq, EqN)                                                                            \
  {                                                                                               \
    if ((U) + 1 < NCOL) {                                                                         \
      uint32_t ad;                                                                                \
      asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(ad) : "r"(resN), "r"(four), "r"(pq));              \
      asm("ld.shared.u32 %0, [%1];" : "=r"(EqN) : "r"(ad), "r"(ones));                           \
    }                                                                                             \
    if ((U) + 2 < NCOL) asm("ld.shared.u8 %0, [%1+" #U "+2];" : "=r"(resN) : "r"(tbase), "r"(ones)); \
    const uint32_t Xv = Eq | Mv;                                                                  \
    const uint32_t Xh = (((Eq & Pv) + Pv) ^ Pv) | Eq;                                             \
    uint32_t Ph = Mv | ~(Xh | Pv);                                                                \
    uint32_t Mh = Pv & Xh;                                                                        \
    asm("mad.lo.u32 %0, %0, %1, %2;" : "+r"(Ph) : "r"(two), "r"(one));                           \
    Mh <<= 1;                                                                                     \
    Pv = Mh | ~(Xv | Ph);                                                                         \
    Mv = Ph & Xv;                                                                                 \
  }

// the unrolled chain of a 32-byte / 16-byte slot, entered at column NCOL - L
#define SQ_W1_CHAIN31(L) \
  switch (L) { \
    case 31: SQ_W1_COL(0, EqA, EqB) \
    case 30: SQ_W1_COL(1, EqB, EqA) \
    case 29: SQ_W1_COL(2, EqA, EqB) \
    case 28: SQ_W1_COL(3, EqB, EqA) \
    case 27: SQ_W1_COL(4, EqA, EqB) \
    case 26: SQ_W1_COL(5, EqB, EqA) \
    case 25: SQ_W1_COL(6, EqA, EqB) \
    case 24: SQ_W1_COL(7, EqB, EqA) \
    case 23: SQ_W1_COL(8, EqA, EqB) \
    case 22: SQ_W1_COL(9, EqB, EqA) \
    case 21: SQ_W1_COL(10, EqA, EqB) \
    case 20: SQ_W1_COL(11, EqB, EqA) \
    case 19: SQ_W1_COL(12, EqA, EqB) \
    case 18: SQ_W1_COL(13, EqB, EqA) \
    case 17: SQ_W1_COL(14, EqA, EqB) \
    case 16: SQ_W1_COL(15, EqB, EqA) \
    case 15: SQ_W1_COL(16, EqA, EqB) \
    case 14: SQ_W1_COL(17, EqB, EqA) \
    case 13: SQ_W1_COL(18, EqA, EqB) \
    case 12: SQ_W1_COL(19, EqB, EqA) \
    case 11: SQ_W1_COL(20, EqA, EqB) \
    case 10: SQ_W1_COL(21, EqB, EqA) \
    case 9: SQ_W1_COL(22, EqA, EqB) \
    case 8: SQ_W1_COL(23, EqB, EqA) \
    case 7: SQ_W1_COL(24, EqA, EqB) \
    case 6: SQ_W1_COL(25, EqB, EqA) \
    case 5: SQ_W1_COL(26, EqA, EqB) \
    case 4: SQ_W1_COL(27, EqB, EqA) \
    case 3: SQ_W1_COL(28, EqA, EqB) \
    case 2: SQ_W1_COL(29, EqB, EqA) \
    case 1: SQ_W1_COL(30, EqA, EqB) \
    default: break; \
  }
#define SQ_W1_CHAIN15(L) \
  switch (L) { \
    case 15: SQ_W1_COL(0, EqA, EqB) \
    case 14: SQ_W1_COL(1, EqB, EqA) \
    case 13: SQ_W1_COL(2, EqA, EqB) \
    case 12: SQ_W1_COL(3, EqB, EqA) \
    case 11: SQ_W1_COL(4, EqA, EqB) \
    case 10: SQ_W1_COL(5, EqB, EqA) \
    case 9: SQ_W1_COL(6, EqA, EqB) \
    case 8: SQ_W1_COL(7, EqB, EqA) \
    case 7: SQ_W1_COL(8, EqA, EqB) \
    case 6: SQ_W1_COL(9, EqB, EqA) \
    case 5: SQ_W1_COL(10, EqA, EqB) \
    case 4: SQ_W1_COL(11, EqB, EqA) \
    case 3: SQ_W1_COL(12, EqA, EqB) \
    case 2: SQ_W1_COL(13, EqB, EqA) \
    case 1: SQ_W1_COL(14, EqA, EqB) \
    default: break; \
  }

template <int STRIDE, bool SCHED>
__global__ void __launch_bounds__(kEdWarps * 32, 64 / kEdWarps)
edit_pairs_w1_kernel(const uint8_t* __restrict__ packed, int64_t n,
                     const uint8_t* __restrict__ packedB, int64_t nB, const uint2* __restrict__ pairs,
                     int64_t n_pairs, int max_d, uint16_t* __restrict__ dist,
                     const uint4* __restrict__ sched, const uint32_t* __restrict__ rowstart,
                     const uint32_t* __restrict__ delta) {
  constexpr int WORDS = STRIDE / 4;
  constexpr int NCOL = STRIDE - 1;                 // longest text of a slot
  constexpr int LSTR = STRIDE + 4;                 // byte stride of a lane's text on the fast path (odd word count)
  __shared__ uint32_t peq_sm[kEdWarps][kEdRuns * 33];
  __shared__ uint32_t mlen_sm[kEdWarps][kEdRuns];
  // the lanes' texts: [word][lane] on the general path, byte-linear [lane][LSTR] on the fast path
  __shared__ __align__(16) uint32_t text_raw[kEdWarps][32 * LSTR / 4];
  static_assert(sizeof(uint32_t) * (STRIDE / 4) * 32 <= sizeof(text_raw[0]), "text area");
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t (*text_sm)[32] = reinterpret_cast<uint32_t (*)[32]>(&text_raw[w][0]);
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
    if (WORDS == 8) {
      // a CDR3 slot is one 32-byte sector: one 256-bit load (LDG.E.256) instead of two 128-bit ones
#pragma unroll
      for (int q = 0; q < WORDS; ++q) tw[q] = 0u;
      if (inrange)
        asm("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
            : "=r"(tw[0]), "=r"(tw[1]), "=r"(tw[2]), "=r"(tw[3]), "=r"(tw[WORDS - 4]), "=r"(tw[WORDS - 3]),
              "=r"(tw[WORDS - 2]), "=r"(tw[WORDS - 1])
            : "l"(rowB));
    } else {
#pragma unroll
      for (int q = 0; q < WORDS / 4; ++q) {
        const uint4 v = inrange ? rowB[q] : make_uint4(0, 0, 0, 0);
        tw[4 * q] = v.x; tw[4 * q + 1] = v.y; tw[4 * q + 2] = v.z; tw[4 * q + 3] = v.w;
      }
    }
  }
  const int nlen = (int)(tw[WORDS - 1] >> 24);
  // ---- fast path: the 32 pairs share ONE pattern (the common case: a row has 161 partners on
  // average at config 4, and the pairs arrive grouped by i).  One table, no run loop; and NO
  // per-column exit: a column whose table word is all ones (every position "matches") moves the whole
  // state up by one bit -- Pv' = Pv << 1, Mv' = Mv << 1 | 1 -- so a lane whose text has ended keeps
  // feeding its slot's pad bytes (0xFF -> table word 255 = ~0) until the warp's longest text is done,
  // and reads D[m][n] from bits [q, q + m) of the final deltas, q = the number of pad columns it ran.
  // That needs m + q <= 32 for every lane that passes the length filter (checked, else the general
  // path below).  The texts are stored byte-linear per lane, so that the warp can ENTER the unrolled
  // chain at column NCOL - Lmax (one warp-uniform indexed jump) and all lanes read "their residue
  // U - (NCOL - Lmax)" at a compile-time offset U of a per-lane base.
  {
    int same;
    __match_all_sync(0xFFFFFFFFu, i, &same);
    if (same && i != 0xFFFFFFFFu) {                   // (i == 0xFFFFFFFF: some lane invalid or out of range)
      uint32_t* peq = peq_sm[w];
      uint32_t chb = 0xFFu;
      if (lane < (uint32_t)STRIDE) chb = packed[(int64_t)i * STRIDE + lane];
      peq[lane] = 0u;
      if (lane == 0) peq[255] = 0xFFFFFFFFu;          // inside the warp's own kEdRuns * 33 words
      const int m = (int)__shfl_sync(0xFFFFFFFFu, chb, STRIDE - 1);
      const uint32_t maskm = (1u << m) - 1u;          // m <= 31
      __syncwarp();
      const uint32_t mm = __match_any_sync(0xFFFFFFFFu, chb);
      if ((int)lane < m) peq[chb] = mm & maskm;
      uint8_t* trow = reinterpret_cast<uint8_t*>(&text_raw[w][0]) + lane * LSTR;
#pragma unroll
      for (int q = 0; q < WORDS; ++q) reinterpret_cast<uint32_t*>(trow)[q] = tw[q];
      const int diff = m > nlen ? m - nlen : nlen - m;
      const bool pass = max_d < 0 || diff <= max_d;
      const int Lmax = __reduce_max_sync(0xFFFFFFFFu, pass ? nlen : 0);
      const int Lmin = __reduce_min_sync(0xFFFFFFFFu, pass ? nlen : NCOL);
      if (m + Lmax - Lmin <= 32) {
        __syncwarp();
        const uint32_t pq = (uint32_t)__cvta_generic_to_shared(peq);
        const uint32_t tbase = (uint32_t)__cvta_generic_to_shared(trow) - (uint32_t)(NCOL - Lmax);
        const uint32_t two = blockDim.x / (kEdWarps * 16), one = blockDim.x / (kEdWarps * 32);
        const uint32_t four = blockDim.x / (kEdWarps * 8);
        // (the chain's loads are not volatile, so that they can be issued ahead of the dependent logic
        // chain; their dummy input `ones` -- read from shared memory behind the warp barrier that
        // publishes table and texts -- keeps them behind that barrier)
        uint32_t ones;
        asm volatile("ld.shared.u32 %0, [%1+1020];" : "=r"(ones) : "r"(pq) : "memory");
        uint32_t Pv = ones, Mv = 0u;
        // residue 0 -> its table word, residue 1: what the first column of the chain expects
        uint32_t resN, EqA, EqB;
        {
          const uint32_t t0 = (uint32_t)__cvta_generic_to_shared(trow);
          uint32_t r0, ad;
          asm("ld.shared.u8 %0, [%1];" : "=r"(r0) : "r"(t0), "r"(ones));
          asm("ld.shared.u8 %0, [%1+1];" : "=r"(resN) : "r"(t0), "r"(ones));
          asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(ad) : "r"(r0), "r"(four), "r"(pq));
          // (the entry column may be an even or an odd one: the word is fetched into both registers)
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(EqA) : "r"(ad), "r"(ones));
          asm volatile("ld.shared.u32 %0, [%1];" : "=r"(EqB) : "r"(ad), "r"(ones));
        }
        if (STRIDE == 32) { SQ_W1_CHAIN31(Lmax) } else { SQ_W1_CHAIN15(Lmax) }
        const uint32_t mask = maskm << ((Lmax - nlen) & 31);       // (a lane that failed the filter: unused)
        int d = nlen + __popc(Pv & mask) - __popc(Mv & mask);
        if (!pass || (max_d >= 0 && d > max_d)) d = max_d + 1;
        dist[p] = (uint16_t)d;
        return;
      }
      __syncwarp();                                    // the general path reuses the shared arrays
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
#pragma unroll
  for (int q = 0; q < WORDS; ++q) text_sm[q][lane] = tw[q];
  // byte y of this lane's text is at tb + (y / 4) * 128 + y % 4 (a compile-time offset per column)
  const uint32_t tb = (uint32_t)__cvta_generic_to_shared(&text_sm[0][lane]);
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
      // 2 and 1 as run-time values (the block has kEdWarps * 32 threads): with literals the assembler turns
      // the multiply-add into a shift-add on the ALU pipe, which is the pipe that bounds this loop
      const uint32_t two = blockDim.x / (kEdWarps * 16), one = blockDim.x / (kEdWarps * 32);
      const uint32_t four = blockDim.x / (kEdWarps * 8);
      uint32_t Pv = 0xFFFFFFFFu, Mv = 0u;
      // one exit per column and ONE reconvergence point behind the loop: a lane whose text has ended
      // leaves the chain and never rejoins it, so the columns need no reconvergence of their own
      // (15 instead of 17 instructions per column: 29.5 -> 28.7 ms)
#pragma unroll
      for (int y = 0; y < STRIDE - 1; ++y) {
        if (y >= nlen) break;
        uint32_t res, ad, Eq;
        // (not volatile, so the loads can be issued ahead of the DP chain; the dummy input m -- read
        // from shared memory after the warp barrier -- keeps them behind the barrier that publishes
        // the table and the texts)
        asm("ld.shared.u8 %0, [%1];" : "=r"(res) : "r"(tb + (uint32_t)((y >> 2) * 128 + (y & 3))), "r"(m));
        asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(ad) : "r"(res), "r"(four), "r"(pq));
        asm("ld.shared.u32 %0, [%1];" : "=r"(Eq) : "r"(ad), "r"(m));
        const uint32_t Xv = Eq | Mv;
        const uint32_t Xh = (((Eq & Pv) + Pv) ^ Pv) | Eq;
        uint32_t Ph = Mv | ~(Xh | Pv);
        uint32_t Mh = Pv & Xh;
        asm("mad.lo.u32 %0, %0, %1, %2;" : "+r"(Ph) : "r"(two), "r"(one));
        Mh <<= 1;
        Pv = Mh | ~(Xv | Ph);
        Mv = Ph & Xv;
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
  const bool big = (size_t)c->n * (size_t)c->stride > (size_t)c->sched_min_bytes;
  const bool use_sched = packedB == c->packed && big && c->sched && c->sched_pairs == pairs &&
                         c->sched_npairs == n_pairs && c->sched_chunks > 0;
  if (use_sched) {
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

// The one-pattern column chain ALONE: tables and texts resident in shared memory (synthetic contents), no
// global memory, every scheduler full.  What it reaches is the ceiling of this formulation of the column
// step (the register file feeds the ALU and the FMA pipe ~1.8 operand vectors per cycle);
// sq_dp_chain_peak reports it in lane-columns per second.
__global__ void __launch_bounds__(kEdWarps * 32, 64 / kEdWarps)
edit_chain_probe_kernel(int iters, int Lmax, uint32_t* __restrict__ sink) {
  constexpr int NCOL = 31, LSTR = 36;
  __shared__ uint32_t peq_sm[kEdWarps][kEdRuns * 33];
  __shared__ uint32_t text_raw[kEdWarps][32 * LSTR / 4];
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t* peq = peq_sm[w];
  for (uint32_t q = lane; q < (uint32_t)kEdRuns * 33; q += 32) peq[q] = (q * 2654435761u) >> 7;
  for (uint32_t q = lane; q < 32u * LSTR / 4; q += 32) text_raw[w][q] = ((q * 0x01010101u) & 0x0F0F0F0Fu) + 0x01020304u;
  __syncwarp();
  const uint32_t two = blockDim.x / (kEdWarps * 16), one = blockDim.x / (kEdWarps * 32);
  const uint32_t four = blockDim.x / (kEdWarps * 8);
  const uint32_t pq = (uint32_t)__cvta_generic_to_shared(peq);
  const uint32_t t0 = (uint32_t)__cvta_generic_to_shared(&text_raw[w][0]) + lane * LSTR;
  const uint32_t tbase = t0 - (uint32_t)(NCOL - Lmax);
  uint32_t acc = 0;
  for (int it = 0; it < iters; ++it) {
    uint32_t ones;
    asm volatile("ld.shared.u32 %0, [%1+1020];" : "=r"(ones) : "r"(pq) : "memory");
    uint32_t Pv = ones ^ (acc & 0xFFu), Mv = 0u;
    uint32_t resN, EqA, EqB;
    {
      uint32_t r0, ad;
      asm("ld.shared.u8 %0, [%1];" : "=r"(r0) : "r"(t0), "r"(ones));
      asm("ld.shared.u8 %0, [%1+1];" : "=r"(resN) : "r"(t0), "r"(ones));
      asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(ad) : "r"(r0), "r"(four), "r"(pq));
      asm volatile("ld.shared.u32 %0, [%1];" : "=r"(EqA) : "r"(ad), "r"(ones));
      asm volatile("ld.shared.u32 %0, [%1];" : "=r"(EqB) : "r"(ad), "r"(ones));
    }
    SQ_W1_CHAIN31(Lmax)
    acc = acc * 3u + (Pv ^ Mv);
  }
  if (acc == 0x12345u) sink[threadIdx.x] = acc;      // practically never true: keeps the chain live
}

template <int W>
int launch_edit(sq_ctx* c, const uint8_t* packedB, int64_t nB, const uint32_t* pairs, int64_t n_pairs,
                int max_d, uint16_t* dist_out) {
  const int threads = W <= 2 ? 256 : 128;
  const size_t smem = (size_t)c->alphabet * W * threads * sizeof(uint32_t);
  if (smem > 48 * 1024)
    SQ_CUDA(c, cudaFuncSetAttribute(edit_pairs_kernel<W>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)smem));
  const int64_t blocks = (n_pairs + threads - 1) / threads;
  SQ_TIMED(c, SQ_K_EDIT, edit_pairs_kernel<W><<<(unsigned)blocks, threads, smem, c->stream>>>(
      c->packed, c->stride, c->n, packedB, nB, reinterpret_cast<const uint2*>(pairs), n_pairs, max_d,
      c->alphabet, dist_out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

// ---- long sequences, banded, Peq shared per run of equal i --------------------------------------
// For pairs that passed a filter (most are within max_d) and come grouped by i: a warp takes 32
// consecutive pairs, builds the Peq table of every distinct pattern once (match.any per 32
// pattern positions, as in the single-word kernel) in shared memory [run][residue][word], and each
// lane runs the column step of sq_dp.cuh restricted to the diagonal band |x - y| <= max_d
// (Ukkonen's cut-off on the word grid) as a SLIDING WINDOW of NWIN words.  Text index y produces
// DP column y + 1, whose band rows y + 1 - max_d .. y + 1 + max_d lie in words (y - max_d) >> 5
// .. (y + max_d) >> 5; the window's first word is (y - max_d) >> 5 and 32 NWIN >= 2 max_d + 32
// makes it cover the band and, in the last column, row m (|m - n| <= max_d is checked first).
//  * when the window moves down, a fresh word (all vertical deltas +1) enters at the bottom: an
//    OVERESTIMATE of the column it joins, a true vertical delta being at most +1;
//  * the word that leaves at the top is dropped, and the window's first word takes the boundary
//    inputs of word 0 (horizontal delta +1, no carry): again an overestimate.
// The DP is monotone, so every computed value is >= the true one, and a cell whose true value is
// <= max_d is exact (its optimal path never leaves the band; a minimum over one exact and other
// overestimated candidates is exact).  Hence min(result, max_d + 1) is exact.  The tracked value
// is the cell at the bottom of the window; D[m][n] is read off it through the vertical deltas
// below row m.  No early exit (an overestimate proves nothing about columns to come).
constexpr int kLgWarps = 8;
constexpr int kLgRuns = 2;

template <int NWIN>
__global__ void __launch_bounds__(kLgWarps * 32)
edit_long_shared_kernel(const uint8_t* __restrict__ packedA, int64_t nA, const uint8_t* __restrict__ packedB,
                        int64_t nB, int stride, int alphabet, int W, const uint2* __restrict__ pairs,
                        int64_t n_pairs, int max_d, uint16_t* __restrict__ dist) {
  extern __shared__ uint32_t lg_smem[];                 // [kLgWarps][kLgRuns][alphabet * WP] + lengths
  const int WP = W | 1;                                 // odd word stride per residue
  const int tsz = alphabet * WP;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t* peq = lg_smem + (size_t)w * kLgRuns * tsz;
  uint32_t* mlen = lg_smem + (size_t)kLgWarps * kLgRuns * tsz + w * kLgRuns;
  const int64_t p = ((int64_t)blockIdx.x * kLgWarps + w) * 32 + lane;
  const bool valid = p < n_pairs;
  uint2 pr = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
  if (valid) pr = pairs[p];
  const bool inrange = valid && pr.x < (uint64_t)nA && pr.y < (uint64_t)nB;
  const uint32_t i = inrange ? pr.x : 0xFFFFFFFFu;
  const uint8_t* rowB = packedB + (int64_t)(inrange ? pr.y : 0u) * stride;
  const int n = inrange ? (int)rowB[stride - 1] : 0;
  const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, i, 1);
  const uint32_t hm = __ballot_sync(0xFFFFFFFFu, lane == 0 || i != prev);
  const int run = __popc(hm & (0xFFFFFFFFu >> (31 - lane))) - 1;
  const int nruns = __popc(hm);
  uint32_t rem = hm;
  int d = 0;
#pragma unroll 1
  for (int rbase = 0; rbase < nruns; rbase += kLgRuns) {
    const int nr = min(kLgRuns, nruns - rbase);
    __syncwarp();
#pragma unroll 1
    for (int r = 0; r < nr; ++r) {
      const int hl = __ffs(rem) - 1;
      rem &= rem - 1;
      const uint32_t ir = __shfl_sync(0xFFFFFFFFu, i, hl);
      uint32_t* t = peq + r * tsz;
      for (int q = lane; q < tsz; q += 32) t[q] = 0u;
      int m = 0;
      if (ir != 0xFFFFFFFFu) m = packedA[(int64_t)ir * stride + stride - 1];
      __syncwarp();
      for (int k = 0; 32 * k < m; ++k) {
        const int x = 32 * k + lane;
        const uint32_t ch = x < m ? packedA[(int64_t)ir * stride + x] : 0xFFu;
        const uint32_t mm = __match_any_sync(0xFFFFFFFFu, ch);
        if (x < m && lane == __ffs(mm) - 1) t[ch * WP + k] = mm;
      }
      if (lane == 0) mlen[r] = (uint32_t)m;
    }
    __syncwarp();
    if (!inrange || run < rbase || run >= rbase + nr) continue;
    const int m = (int)mlen[run - rbase];
    const uint32_t* t = peq + (run - rbase) * tsz;
    const int diff = m > n ? m - n : n - m;
    if (diff > max_d) { d = max_d + 1; continue; }
    if (m == 0) { d = n; continue; }
    if (n == 0) { d = m; continue; }
    const int last = (m - 1) >> 5, topbit = (m - 1) & 31;
    uint32_t Pw[NWIN], Mw[NWIN];
#pragma unroll
    for (int k = 0; k < NWIN; ++k) { Pw[k] = 0xFFFFFFFFu; Mw[k] = 0u; }
    int wlo = 0;
    int sb = 32 * NWIN;                                  // D at the bottom row of the window
    const uint32_t* b32 = reinterpret_cast<const uint32_t*>(rowB);
    for (int y0 = 0; y0 < n; y0 += 4) {
      const uint32_t word = b32[y0 >> 2];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int y = y0 + q;
        if (y >= n) break;
        if (y >= max_d && ((y - max_d) >> 5) > wlo) {    // the band has left the top word
#pragma unroll
          for (int k = 0; k + 1 < NWIN; ++k) { Pw[k] = Pw[k + 1]; Mw[k] = Mw[k + 1]; }
          Pw[NWIN - 1] = 0xFFFFFFFFu; Mw[NWIN - 1] = 0u;
          ++wlo;
          sb += 32;
        }
        const uint32_t* te = t + ((word >> (8 * q)) & 0xFFu) * WP + wlo;
        uint32_t carry = 0u, ph_in = 1u, mh_in = 0u;
#pragma unroll
        for (int k = 0; k < NWIN; ++k) {
          const uint32_t Eq = wlo + k < W ? te[k] : 0u;
          const uint32_t pv = Pw[k], mv = Mw[k];
          const uint32_t Xv = Eq | mv;
          const uint64_t s64 = (uint64_t)(Eq & pv) + (uint64_t)pv + (uint64_t)carry;
          carry = (uint32_t)(s64 >> 32);
          const uint32_t Xh = ((uint32_t)s64 ^ pv) | Eq;
          uint32_t Ph = mv | ~(Xh | pv);
          uint32_t Mh = pv & Xh;
          const uint32_t ph_out = Ph >> 31, mh_out = Mh >> 31;
          if (k == NWIN - 1) sb += (int)ph_out - (int)mh_out;
          Ph = (Ph << 1) | ph_in;
          Mh = (Mh << 1) | mh_in;
          ph_in = ph_out;
          mh_in = mh_out;
          Pw[k] = Mh | ~(Xv | Ph);
          Mw[k] = Ph & Xv;
        }
      }
    }
    // from the window's bottom row up to row m
    const int kl = last - wlo;                           // 0 <= kl < NWIN (see the header comment)
#pragma unroll
    for (int k = 0; k < NWIN; ++k) {
      if (k > kl) sb -= __popc(Pw[k]) - __popc(Mw[k]);
      else if (k == kl) {
        const uint32_t above = topbit == 31 ? 0u : (0xFFFFFFFFu << (topbit + 1));
        sb -= __popc(Pw[k] & above) - __popc(Mw[k] & above);
      }
    }
    d = sb;
  }
  if (!valid) return;
  if (!inrange) { dist[p] = 0xFFFFu; return; }
  if (d > max_d) d = max_d + 1;
  dist[p] = (uint16_t)d;
}

template <int NWIN>
int launch_edit_long(sq_ctx* c, const uint8_t* packedB, int64_t nB, int words, const uint32_t* pairs,
                     int64_t n_pairs, int max_d, uint16_t* dist_out) {
  const int WP = words | 1;
  const size_t smem = ((size_t)kLgWarps * kLgRuns * c->alphabet * WP + kLgWarps * kLgRuns) * sizeof(uint32_t);
  if (smem > 48 * 1024)
    SQ_CUDA(c, cudaFuncSetAttribute(edit_long_shared_kernel<NWIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t blocks = (n_pairs + kLgWarps * 32 - 1) / (kLgWarps * 32);
  SQ_TIMED(c, SQ_K_EDIT, edit_long_shared_kernel<NWIN><<<(unsigned)blocks, kLgWarps * 32, smem, c->stream>>>(
      c->packed, c->n, packedB, nB, c->stride, c->alphabet, words, reinterpret_cast<const uint2*>(pairs),
      n_pairs, max_d, dist_out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
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
  if (banded && words >= 3 && words <= 8 && max_d >= 0 && max_d <= 32 && c->alphabet <= 32) {
    // filtered pairs grouped by i: shared Peq tables, sliding band window
    if (max_d <= 16) return launch_edit_long<2>(c, packedB, nB, words, pairs, n_pairs, max_d, dist_out);
    return launch_edit_long<3>(c, packedB, nB, words, pairs, n_pairs, max_d, dist_out);
  }
  if (words <= 1) return launch_edit<1>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  if (words <= 2) return launch_edit<2>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  if (words <= 4) return launch_edit<4>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  if (words <= 5) return launch_edit<5>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  if (words <= 8) return launch_edit<8>(c, packedB, nB, pairs, n_pairs, max_d, dist_out);
  return SQ_ERR_UNSUPPORTED;
}

// Distances of the survivors of a coarse filter (sq_all_pairs, sq_join).  Long sequences: the
// survivors are grouped by i (radix sort on the i field, ping-pong between surv and surv2) and
// take the shared-Peq banded kernel.  *live_out = the list sdist refers to (surv or surv2).
int sq_survivor_distances(sq_ctx* c, const uint8_t* packedB, int64_t nB, int max_len_b, uint2* surv,
                          int64_t ns, int max_d, uint2* surv2, void* sort_tmp, uint16_t* sdist,
                          const uint2** live_out, int64_t* nlive_out) {
  *live_out = surv; *nlive_out = ns;
  if (ns <= 0) return SQ_OK;
  const int ml = c->max_len > max_len_b ? c->max_len : max_len_b;
  const int applied = (ml > 64 && max_d >= 0 && max_d <= 32 && c->alphabet <= 32) ? 1 : 0;
  uint2* live = surv;
  int64_t nlive = ns;
  int rc = SQ_OK;
  if (applied && nlive > 1) {
    // group by i: LSD passes over the low word (a uint2 (i, j) is the 64-bit key i | j << 32)
    int nb = 1;
    while (nb < 32 && (1ll << nb) < c->n) ++nb;
    int shifts[4], widths[4], q = 0;
    for (int b = 0; b < nb; b += 8) { shifts[q] = b; widths[q] = nb - b >= 8 ? 8 : nb - b; ++q; }
    int in_alt = 0;
    rc = sq_radix_sort(c, reinterpret_cast<uint64_t*>(surv), reinterpret_cast<uint64_t*>(surv2), nullptr,
                       nullptr, nlive, 1, shifts, widths, q, sort_tmp, &in_alt);
    if (rc != SQ_OK) return rc;
    if (in_alt) live = surv2;
  }
  *live_out = live; *nlive_out = nlive;
  if (nlive == 0) return SQ_OK;
  return sq_edit_distance_ab(c, packedB, nB, max_len_b, reinterpret_cast<const uint32_t*>(live), nlive, max_d,
                             sdist, applied != 0);
}

int sq_edit_distance_impl(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                          uint16_t* dist_out) {
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  return sq_edit_distance_ab(c, c->packed, c->n, c->max_len, pairs, n_pairs, max_d, dist_out, false);
}

extern "C" int sq_dp_chain_peak(sq_ctx* c, int text_len, int iters, double* lane_columns_per_s) {
  if (!c || !lane_columns_per_s || iters < 1 || text_len < 1 || text_len > 31) return SQ_ERR_INVALID_ARG;
  if (!c->ws) return SQ_ERR_WORKSPACE;
  SqDeviceGuard guard(c);
  const size_t top = c->scratch_top;
  uint32_t* sink = sq_scratch<uint32_t>(c, 256);     // handed back at once: practically never written
  c->scratch_top = top;
  if (!sink) return SQ_ERR_WORKSPACE;
  const int blocks = c->sm_count * (64 / kEdWarps);
  cudaEvent_t e0, e1;
  SQ_CUDA(c, cudaEventCreate(&e0));
  if (cudaEventCreate(&e1) != cudaSuccess) { c->last_err = cudaGetLastError(); cudaEventDestroy(e0); return SQ_ERR_CUDA; }
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, c->stream);
    edit_chain_probe_kernel<<<blocks, kEdWarps * 32, 0, c->stream>>>(iters, text_len, sink);
    c->launches++;
    cudaEventRecord(e1, c->stream);
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
      c->last_err = cudaGetLastError();
      cudaEventDestroy(e0); cudaEventDestroy(e1);
      return SQ_ERR_CUDA;
    }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *lane_columns_per_s = (double)blocks * kEdWarps * 32.0 * (double)iters * (double)text_len / (best * 1e-3);
  return SQ_OK;
}
