// sq_wedit.cu -- weighted edit distance on an explicit pair list: the
// recurrence of PAPER.md L754 Eq. (46) as printed,
//     D(x,y) = min(D(x-1,y) + indel, D(x,y-1) + indel, D(x-1,y-1) + substitution_cost(a_x, b_y)),
// with the substitution cost from a caller-supplied table ("typically based on biochemical
// similarity", L760) and D(x,0) = x*indel, D(0,y) = y*indel.  Bit-parallelism does not apply to
// general costs: this is the plain DP, organised for the machine.
//
// Short sequences (<= 31 residues, one 16/32-byte slot): a warp takes 32 pairs (family-ordered
// schedule of sq_lsh_candidates when available, like the unit-cost kernel).  The pairs arrive
// grouped by i, so per run of equal i the warp builds a QUERY PROFILE in shared memory --
// prof[c][x] = cost(a_x, c), one byte per pattern position, 32 bytes per residue c -- and a DP
// column step is: two 16-byte loads of the text residue's profile row, then per pattern row one
// byte extract and  new = min(up + indel, min(diag + cost, old + indel))  on a register-resident
// column (rows padded to a multiple of 4, picked per run).
// Longer sequences: one thread per pair, the DP column in shared memory [row][thread].
#include "sq_common.cuh"

namespace {

constexpr int kWeWarps = 2;
constexpr int kWeRuns = 4;               // query profiles resident per warp (1 KB each)

// one text column against MR pattern rows; D[x] = D(x+1, y) on entry for column y, updated in place
template <int MR>
__device__ __forceinline__ void we_column(int (&D)[32], const uint32_t* __restrict__ prow, int y,
                                          int indel) {
  uint32_t cw[MR / 4];
#pragma unroll
  for (int q = 0; q < MR / 16; ++q) {
    const uint4 v = *reinterpret_cast<const uint4*>(prow + 4 * q);
    cw[4 * q] = v.x; cw[4 * q + 1] = v.y; cw[4 * q + 2] = v.z; cw[4 * q + 3] = v.w;
  }
  if (MR % 16 >= 8) {                     // one more 8-byte piece
    const uint2 v = *reinterpret_cast<const uint2*>(prow + (MR / 16) * 4);
    cw[(MR / 16) * 4] = v.x; cw[(MR / 16) * 4 + 1] = v.y;
  }
  if (MR % 8 >= 4) cw[MR / 4 - 1] = prow[MR / 4 - 1];   // and / or a 4-byte one (MR is a multiple of 4)
  int diag = y * indel;                   // D(0, y)
  int up = diag + indel;                  // D(0, y+1)
#pragma unroll
  for (int x = 0; x < MR; ++x) {
    const int cost = (int)((cw[x >> 2] >> (8 * (x & 3))) & 0xFFu);
    const int old = D[x];
    const int nw = min(up + indel, min(diag + cost, old + indel));
    diag = old; up = nw; D[x] = nw;
  }
}

// the text is read byte by byte from shared memory (a runtime loop keeps the code and the register
// count small: the column step itself is MR fully unrolled cells)
template <int MR>
__device__ __forceinline__ int we_dp(const uint32_t* __restrict__ prof, int m,
                                     const uint8_t* __restrict__ text, int nlen, int indel) {
  int D[32];
#pragma unroll
  for (int x = 0; x < MR; ++x) D[x] = (x + 1) * indel;
#pragma unroll 1
  for (int y = 0; y < nlen; ++y) we_column<MR>(D, prof + (text[y] & 31u) * 8, y, indel);
  // D(m, n): picked with masks, not with an index, so that D stays in registers
  int res = 0;
#pragma unroll
  for (int x = 0; x < MR; ++x) res |= D[x] & -(int)(x == m - 1);
  return res;
}

template <int STRIDE, bool SCHED>
__global__ void __launch_bounds__(kWeWarps * 32)
wedit_short_kernel(const uint8_t* __restrict__ packed, int64_t n, const uint2* __restrict__ pairs,
                   int64_t n_pairs, const uint8_t* __restrict__ sub, int sigma, int indel, int max_d,
                   uint16_t* __restrict__ dist, const uint4* __restrict__ sched,
                   const uint32_t* __restrict__ rowstart, const uint32_t* __restrict__ delta) {
  constexpr int WORDS = STRIDE / 4;
  __shared__ __align__(16) uint32_t prof_sm[kWeWarps][kWeRuns * 32 * 8];
  __shared__ uint32_t mlen_sm[kWeWarps][kWeRuns];
  __shared__ uint32_t text_sm[kWeWarps][32 * 9];     // 36-byte stride per lane: conflict-free
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t wk = (int64_t)blockIdx.x * kWeWarps + w;
  int64_t p = wk * 32 + lane;
  bool valid = p < n_pairs;
  if (SCHED && valid) {
    const uint4 ch = sched[wk];
    const uint32_t q = (uint32_t)p;
    if (q < ch.z) p = (int64_t)(uint32_t)(ch.y + q);
    else {
      uint32_t r = ch.x + 1;
      while (q >= rowstart[r + 1]) ++r;
      p = (int64_t)(uint32_t)(delta[r] + q);
    }
  }
  uint2 pr = make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
  if (valid) pr = pairs[p];
  const bool inrange = valid && pr.x < (uint64_t)n && pr.y < (uint64_t)n;
  const uint32_t i = inrange ? pr.x : 0xFFFFFFFFu;
  uint32_t tw[WORDS];
  {
    const uint4* rowB = reinterpret_cast<const uint4*>(packed + (int64_t)(inrange ? pr.y : 0u) * STRIDE);
#pragma unroll
    for (int q = 0; q < WORDS / 4; ++q) {
      const uint4 v = inrange ? rowB[q] : make_uint4(0, 0, 0, 0);
      tw[4 * q] = v.x; tw[4 * q + 1] = v.y; tw[4 * q + 2] = v.z; tw[4 * q + 3] = v.w;
    }
  }
  const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, i, 1);
  const bool head = lane == 0 || i != prev;
  const uint32_t hm = __ballot_sync(0xFFFFFFFFu, head);
  const uint32_t run = __popc(hm & (0xFFFFFFFFu >> (31 - lane))) - 1;
  const int nruns = __popc(hm);
  uint32_t* prof = prof_sm[w];
  uint32_t rem = hm;
  const int nlen = (int)(tw[WORDS - 1] >> 24);
#pragma unroll
  for (int q = 0; q < WORDS; ++q) text_sm[w][lane * 9 + q] = tw[q];
  const uint8_t* text = reinterpret_cast<const uint8_t*>(&text_sm[w][lane * 9]);
  int d = 0;
#pragma unroll 1
  for (int rbase = 0; rbase < nruns; rbase += kWeRuns) {
    const int nr = min(kWeRuns, nruns - rbase);
    __syncwarp();
#pragma unroll 1
    for (int r = 0; r < nr; ++r) {        // the query profile of run r: prof[c][x] = cost(a_x, c)
      const int hl = __ffs(rem) - 1;
      rem &= rem - 1;
      const uint32_t ir = __shfl_sync(0xFFFFFFFFu, i, hl);
      uint32_t ax = 0xFFu;
      if (ir != 0xFFFFFFFFu && lane < (uint32_t)STRIDE) ax = packed[(int64_t)ir * STRIDE + lane];
      const uint32_t m = ir != 0xFFFFFFFFu ? __shfl_sync(0xFFFFFFFFu, ax, STRIDE - 1) : 0u;
      uint8_t* pb = reinterpret_cast<uint8_t*>(prof + r * 256);
      for (int c = 0; c < sigma; ++c)
        pb[c * 32 + lane] = (lane < m && ax != (uint32_t)c) ? sub[ax * sigma + c] : (uint8_t)0;   // Eq. 46: I(a != b) * cost
      if (lane == 0) mlen_sm[w][r] = m;
    }
    __syncwarp();
    if (!inrange || (int)run < rbase || (int)run >= rbase + nr) continue;
    const int m = (int)mlen_sm[w][run - rbase];
    const uint32_t* pq = prof + (run - rbase) * 256;
    const int diff = m > nlen ? m - nlen : nlen - m;
    if (max_d >= 0 && diff * indel > max_d) d = max_d + 1;
    else if (m == 0) d = nlen * indel;
    else if (nlen == 0) d = m * indel;
    // (the pattern rows of a run are padded to a multiple of 4: the column step is MR unrolled cells)
    else if (m <= 8) d = we_dp<8>(pq, m, text, nlen, indel);
    else if (m <= 12) d = we_dp<12>(pq, m, text, nlen, indel);
    else if (m <= 16) d = we_dp<16>(pq, m, text, nlen, indel);
    else if (m <= 20) d = we_dp<20>(pq, m, text, nlen, indel);
    else if (m <= 24) d = we_dp<24>(pq, m, text, nlen, indel);
    else if (m <= 28) d = we_dp<28>(pq, m, text, nlen, indel);
    else d = we_dp<32>(pq, m, text, nlen, indel);
  }
  if (!valid) return;
  if (!inrange) { dist[p] = 0xFFFFu; return; }
  if (d > 65535) d = 65535;
  if (max_d >= 0 && d > max_d) d = max_d + 1;
  dist[p] = (uint16_t)d;
}

// any length <= SQ_MAX_LEN: one thread per pair, DP column D(1..m, y) in shared memory
constexpr int kWlThreads = 64;

__global__ void __launch_bounds__(kWlThreads)
wedit_long_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n,
                  const uint2* __restrict__ pairs, int64_t n_pairs, const uint8_t* __restrict__ sub,
                  int sigma, int indel, int max_d, int max_len, uint16_t* __restrict__ dist) {
  extern __shared__ int col_sm[];           // [max_len][kWlThreads]
  __shared__ uint8_t sub_sm[32 * 32];
  // Eq. 46 multiplies the cost by I(a != b): the table's diagonal is never used
  for (int t = threadIdx.x; t < sigma * sigma; t += kWlThreads) sub_sm[t] = (t / sigma == t % sigma) ? (uint8_t)0 : sub[t];
  __syncthreads();
  const int64_t p = (int64_t)blockIdx.x * kWlThreads + threadIdx.x;
  if (p >= n_pairs) return;
  const uint2 pr = pairs[p];
  if (pr.x >= (uint64_t)n || pr.y >= (uint64_t)n) { dist[p] = 0xFFFFu; return; }
  const uint8_t* a = packed + (int64_t)pr.x * stride;
  const uint8_t* b = packed + (int64_t)pr.y * stride;
  const int m = a[stride - 1], nl = b[stride - 1];
  int* D = col_sm + threadIdx.x;
  for (int x = 0; x < m; ++x) D[x * kWlThreads] = (x + 1) * indel;
  for (int y = 0; y < nl; ++y) {
    const uint8_t* srow = sub_sm + b[y];     // cost(a_x, b_y) = sub[a_x * sigma + b_y]
    int diag = y * indel, up = diag + indel;
    for (int x = 0; x < m; ++x) {
      const int old = D[x * kWlThreads];
      const int nw = min(up + indel, min(diag + (int)srow[a[x] * sigma], old + indel));
      diag = old; up = nw; D[x * kWlThreads] = nw;
    }
  }
  int d = m == 0 ? nl * indel : D[(m - 1) * kWlThreads];
  if (m > 0 && nl == 0) d = m * indel;
  if (d > 65535) d = 65535;
  if (max_d >= 0 && d > max_d) d = max_d + 1;
  dist[p] = (uint16_t)d;
  (void)max_len;
}

template <int STRIDE>
int launch_short(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, const uint8_t* sub, int indel,
                 int max_d, uint16_t* dist_out) {
  const bool big = (size_t)c->n * (size_t)c->stride > (size_t)c->sched_min_bytes;
  if (big && c->sched && c->sched_pairs == pairs && c->sched_npairs == n_pairs && c->sched_chunks > 0) {
    const int64_t blocks = (c->sched_chunks + kWeWarps - 1) / kWeWarps;
    SQ_TIMED(c, SQ_K_EDIT, wedit_short_kernel<STRIDE, true><<<(unsigned)blocks, kWeWarps * 32, 0, c->stream>>>(
        c->packed, c->n, reinterpret_cast<const uint2*>(pairs), n_pairs, sub, c->alphabet, indel, max_d,
        dist_out, c->sched, c->sched_rowstart, c->sched_delta));
  } else {
    const int64_t per_block = kWeWarps * 32;
    const int64_t blocks = (n_pairs + per_block - 1) / per_block;
    SQ_TIMED(c, SQ_K_EDIT, wedit_short_kernel<STRIDE, false><<<(unsigned)blocks, kWeWarps * 32, 0, c->stream>>>(
        c->packed, c->n, reinterpret_cast<const uint2*>(pairs), n_pairs, sub, c->alphabet, indel, max_d,
        dist_out, nullptr, nullptr, nullptr));
  }
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

}  // namespace

extern "C" int sq_edit_distance_weighted(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs,
                                         const uint8_t* sub_cost, int indel, int max_d,
                                         uint16_t* dist_out) {
  if (!c) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (n_pairs < 0 || indel < 1 || indel > 255) return SQ_ERR_INVALID_ARG;
  if (n_pairs == 0) return SQ_OK;
  if (!pairs || !dist_out || !sub_cost) return SQ_ERR_INVALID_ARG;
  if (n_pairs >= (1ll << 31) * 64) return SQ_ERR_UNSUPPORTED;
  if (max_d > 65534) max_d = -1;
  if (c->stride == 16) return launch_short<16>(c, pairs, n_pairs, sub_cost, indel, max_d, dist_out);
  if (c->stride == 32) return launch_short<32>(c, pairs, n_pairs, sub_cost, indel, max_d, dist_out);
  const size_t smem = (size_t)(c->max_len > 0 ? c->max_len : 1) * kWlThreads * sizeof(int);
  if (smem > 200 * 1024) return SQ_ERR_UNSUPPORTED;
  if (smem > 48 * 1024)
    SQ_CUDA(c, cudaFuncSetAttribute(wedit_long_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t blocks = (n_pairs + kWlThreads - 1) / kWlThreads;
  SQ_TIMED(c, SQ_K_EDIT, wedit_long_kernel<<<(unsigned)blocks, kWlThreads, smem, c->stream>>>(
      c->packed, c->stride, c->n, reinterpret_cast<const uint2*>(pairs), n_pairs, sub_cost, c->alphabet,
      indel, max_d, c->max_len, dist_out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}
