// sq_graph.cu -- from verified candidates to the sparse similarity graph:
// PAPER.md L71-73 Eq. (1) G = (V, E, W); Alg. 1 step 12 "build similarity matrix A" (L185); the
// MinHash Jaccard estimate (L495-497 Eq. 30) thresholded at tau (tau = 0.7 in L269, L638).
//
//   edge (i, j), i < j, is kept iff  d(i, j) <= max_d  AND  #{c : sig[i][c] == sig[j][c]} >= min_matches
//   (the caller turns tau into the integer min_matches = ceil(tau * H), so no floating-point
//   comparison decides anything);  weight = 1 - d / max(len_i, len_j)  in fp32.
//
// Output: upper-triangular CSR -- row_ptr[n+1], col[] ascending inside a row, weight[] -- built
// from a pair list whose first index is non-decreasing (both orders of sq_lsh_candidates are).
//   keep_kernel    one warp per pair: the two signature rows are read coalesced (lane = column),
//                  equal columns counted with a ballot; kept pairs are flagged and counted per row.
//   scans          flags -> edge slots (stable), row counts -> row_ptr.
//   edge_kernel    kept pair p -> col / weight at its slot.
#include "sq_common.cuh"

namespace {

// A warp takes 32 pairs (positions [32k, 32k+32) of the family-ordered schedule left by sq_lsh_candidates
// when SCHED -- the signature rows of one family stay in L2 -- else pairs [32k, 32k+32)) and works on
// FOUR pairs at a time, eight lanes per pair: lane l8 of a group compares columns [l8 * H/8, +H/8) of the
// two signature rows, read by 16-byte loads (a row of H = 64 columns is two loads per lane, the eight
// lanes of a group cover 128 contiguous bytes per load); the equal columns are summed over the group
// with three shuffles.  Row i's share of the signature stays in registers while i does not change (the
// pairs arrive grouped by i).  Round 1 gave a whole warp to every pair (two 4-byte loads and a ballot
// per 32 columns: ~45 warp instructions per pair); this needs ~12.
// CPL4 = 16-byte pieces per lane = H / 32.
template <bool SCHED, int CPL4>
__global__ void __launch_bounds__(256)
graph_keep_kernel(const uint2* __restrict__ pairs, const uint16_t* __restrict__ dist, int64_t n_pairs,
                  int max_d, const uint32_t* __restrict__ sig, int H, int min_matches, int64_t n,
                  uint32_t* __restrict__ keep, uint32_t* __restrict__ row_cnt,
                  const uint4* __restrict__ sched, const uint32_t* __restrict__ rowstart,
                  const uint32_t* __restrict__ delta) {
  const int lane = threadIdx.x & 31;
  const int64_t wk = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t q0 = wk * 32;
  if (q0 >= n_pairs) return;
  int64_t p = q0 + lane;                              // lane t owns position q0 + t
  const bool valid = p < n_pairs;
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
  bool ok = false;
  if (valid) {
    pr = pairs[p];
    ok = pr.x < (uint64_t)n && pr.y < (uint64_t)n && (int)dist[p] <= max_d;
  }
  if (min_matches > 0) {
    const int sub = lane >> 3, l8 = lane & 7;
    uint4 ra[CPL4];
    uint32_t cur_i = 0xFFFFFFFFu;
    int mine = 0;                                     // equal columns of this lane's own pair
#pragma unroll 1
    for (int g = 0; g < 8; ++g) {
      const int t = 4 * g + sub;                      // the pair this group of eight lanes works on
      const uint32_t it = __shfl_sync(0xFFFFFFFFu, pr.x, t), jt = __shfl_sync(0xFFFFFFFFu, pr.y, t);
      const bool okt = __shfl_sync(0xFFFFFFFFu, ok ? 1 : 0, t) != 0;
      int m = 0;
      if (okt) {
        if (it != cur_i) {
          const uint4* a = reinterpret_cast<const uint4*>(sig + (int64_t)it * H) + l8 * CPL4;
#pragma unroll
          for (int q = 0; q < CPL4; ++q) ra[q] = a[q];
          cur_i = it;
        }
        const uint4* b = reinterpret_cast<const uint4*>(sig + (int64_t)jt * H) + l8 * CPL4;
#pragma unroll
        for (int q = 0; q < CPL4; ++q) {
          const uint4 v = b[q];
          m += (v.x == ra[q].x) + (v.y == ra[q].y) + (v.z == ra[q].z) + (v.w == ra[q].w);
        }
      }
      m += __shfl_xor_sync(0xFFFFFFFFu, m, 1);
      m += __shfl_xor_sync(0xFFFFFFFFu, m, 2);
      m += __shfl_xor_sync(0xFFFFFFFFu, m, 4);
      // pair t's count sits in group t & 3; its owner is lane t
      const int got = __shfl_sync(0xFFFFFFFFu, m, (lane & 3) * 8);
      if ((lane >> 2) == g) mine = got;
    }
    ok = ok && mine >= min_matches;
  }
  if (valid) keep[p] = ok ? 1u : 0u;
  // kept pairs per row: one atomic per run of equal i inside the warp
  const uint32_t key = ok ? pr.x : 0xFFFFFFFFu;
  const uint32_t peers = __match_any_sync(0xFFFFFFFFu, key);
  if (ok && lane == __ffs(peers) - 1) atomicAdd(&row_cnt[pr.x], (uint32_t)__popc(peers));
}

__global__ void __launch_bounds__(256)
graph_edge_kernel(const uint2* __restrict__ pairs, const uint16_t* __restrict__ dist, int64_t n_pairs,
                  const uint32_t* __restrict__ slot, const uint8_t* __restrict__ len8,
                  uint32_t* __restrict__ col, float* __restrict__ weight) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_pairs) return;
  const uint32_t s = slot[p];
  if (slot[p + 1] == s) return;                 // not kept (the scan covers n_pairs + 1 entries)
  const uint2 pr = pairs[p];
  const int la = len8[pr.x], lb = len8[pr.y];      // (one byte per sequence: the table stays in L2)
  const int L = la > lb ? la : lb;
  col[s] = pr.y;
  weight[s] = L > 0 ? 1.0f - (float)dist[p] / (float)L : 1.0f;
}

// the lengths of all sequences as one byte each (the slots' length bytes are a stride apart: 32 bytes of
// DRAM traffic per lookup, two lookups per edge)
__global__ void __launch_bounds__(256)
graph_len_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n, uint8_t* __restrict__ len8) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) len8[i] = packed[i * stride + stride - 1];
}

__global__ void __launch_bounds__(256)
graph_rowptr_kernel(const uint32_t* __restrict__ row_off, int64_t n, unsigned long long total,
                    int64_t* __restrict__ row_ptr) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) row_ptr[i] = (int64_t)row_off[i];
  if (i == n) row_ptr[n] = (int64_t)total;
}

}  // namespace

size_t sq_graph_scratch_bytes(int64_t n, int64_t n_pairs) {
  const size_t np = (size_t)(n_pairs > 0 ? n_pairs : 1), nn = (size_t)(n > 0 ? n : 1);
  return sq_align_up((np + 2) * 4 + 16) + sq_align_up((nn + 2) * 4 + 16) +
         sq_align_up((np / 2048 + nn / 2048 + 8) * 4 + 16) + 4096;
}

extern "C" int sq_affinity_graph(sq_ctx* c, const uint32_t* pairs, const uint16_t* dist, int64_t n_pairs,
                                 int max_d, const uint32_t* sig, int H, int min_matches,
                                 int64_t* row_ptr, uint32_t* col, float* weight, int64_t capacity,
                                 int64_t* n_edges) {
  if (!c || !n_edges || !row_ptr) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  *n_edges = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (n_pairs < 0 || capacity < 0 || max_d < 0 || min_matches < 0) return SQ_ERR_INVALID_ARG;
  if (min_matches > 0 && (!sig || H < 32 || (H % 32) != 0 || H > SQ_MAX_H || min_matches > H ||
                          (reinterpret_cast<uintptr_t>(sig) & 15) != 0))      // rows are read by 16-byte loads
    return SQ_ERR_INVALID_ARG;
  if (n_pairs >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;
  const int64_t n = c->n;
  cudaStream_t st = c->stream;
  // the schedule of sq_lsh_candidates lives in the scratch: keep it (and allocate above it) when
  // it describes these very pairs and the signatures do not fit the L2
  bool use_sched = c->sched && c->sched_pairs == pairs && c->sched_npairs == n_pairs &&
                   min_matches > 0 && (size_t)n * H * 4 > (size_t)c->sched_min_bytes;
  const uint4* sched = c->sched; const uint32_t* srow = c->sched_rowstart; const uint32_t* sdel = c->sched_delta;
  const size_t top_before = c->scratch_top;
  uint32_t* keep = nullptr; uint32_t* row_cnt = nullptr; uint32_t* tmp = nullptr;
  for (int attempt = 0; attempt < 2; ++attempt) {
    if (!use_sched) sq_scratch_reset(c);
    keep = sq_scratch<uint32_t>(c, (size_t)n_pairs + 2);
    row_cnt = sq_scratch<uint32_t>(c, (size_t)n + 2);
    tmp = sq_scratch<uint32_t>(c, (size_t)n_pairs / 2048 + (size_t)n / 2048 + 8);
    if (keep && row_cnt && tmp) break;
    if (!use_sched) return SQ_ERR_WORKSPACE;
    c->scratch_top = top_before;                     // no room above the schedule: do without it
    use_sched = false;
  }
  SQ_CUDA(c, cudaMemsetAsync(row_cnt, 0, ((size_t)n + 2) * 4, st));
  SQ_CUDA(c, cudaMemsetAsync(keep + n_pairs, 0, 8, st));
  SQ_CUDA(c, cudaMemsetAsync(c->dflags, 0, 64, st));
  if (n_pairs > 0) {
    if (!pairs || !dist) return SQ_ERR_INVALID_ARG;
    const int64_t blocks = ((n_pairs + 31) / 32 * 32 + 255) / 256;       // a warp per 32 pairs
    if (blocks >= (1ll << 31)) return SQ_ERR_UNSUPPORTED;
    const uint2* pp = reinterpret_cast<const uint2*>(pairs);
#define SQ_GRAPH_LAUNCH(SCHED_, C4_)                                                                       \
    SQ_TIMED(c, SQ_K_MISC, (graph_keep_kernel<SCHED_, C4_><<<(unsigned)blocks, 256, 0, st>>>(               \
        pp, dist, n_pairs, max_d, sig, H, min_matches, n, keep, row_cnt, use_sched ? sched : nullptr,        \
        use_sched ? srow : nullptr, use_sched ? sdel : nullptr)))
#define SQ_GRAPH_DISPATCH(SCHED_)                                                                          \
    switch (min_matches > 0 ? H / 32 : 1) {                                                                \
      case 1: SQ_GRAPH_LAUNCH(SCHED_, 1); break;                                                           \
      case 2: SQ_GRAPH_LAUNCH(SCHED_, 2); break;                                                           \
      case 3: SQ_GRAPH_LAUNCH(SCHED_, 3); break;                                                           \
      case 4: SQ_GRAPH_LAUNCH(SCHED_, 4); break;                                                           \
      case 5: SQ_GRAPH_LAUNCH(SCHED_, 5); break;                                                           \
      case 6: SQ_GRAPH_LAUNCH(SCHED_, 6); break;                                                           \
      case 7: SQ_GRAPH_LAUNCH(SCHED_, 7); break;                                                           \
      default: SQ_GRAPH_LAUNCH(SCHED_, 8); break;                                                          \
    }
    if (use_sched) { SQ_GRAPH_DISPATCH(true) } else { SQ_GRAPH_DISPATCH(false) }
#undef SQ_GRAPH_DISPATCH
#undef SQ_GRAPH_LAUNCH
    SQ_LAUNCH_CHECK(c);
    int rc = sq_exclusive_scan_u32(c, keep, keep, n_pairs + 1, tmp, c->dflags);
    if (rc != SQ_OK) return rc;
  }
  int rc = sq_exclusive_scan_u32(c, row_cnt, row_cnt, n, tmp, nullptr);
  if (rc != SQ_OK) return rc;
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, c->dflags, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  const int64_t edges = (int64_t)c->pinned[0];
  *n_edges = edges;
  SQ_TIMED(c, SQ_K_MISC, graph_rowptr_kernel<<<(unsigned)((n + 256) / 256), 256, 0, st>>>(
      row_cnt, n, (unsigned long long)edges, row_ptr));
  SQ_LAUNCH_CHECK(c);
  if (edges > capacity) { SQ_CUDA(c, cudaStreamSynchronize(st)); return SQ_ERR_CAPACITY; }
  if (edges > 0) {
    if (!col || !weight) return SQ_ERR_INVALID_ARG;
    // (row_cnt has been copied into row_ptr: its buffer takes the byte-per-sequence length table)
    uint8_t* len8 = reinterpret_cast<uint8_t*>(row_cnt);
    SQ_TIMED(c, SQ_K_MISC, graph_len_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(c->packed, c->stride, n, len8));
    SQ_LAUNCH_CHECK(c);
    SQ_TIMED(c, SQ_K_MISC, graph_edge_kernel<<<(unsigned)((n_pairs + 255) / 256), 256, 0, st>>>(
        reinterpret_cast<const uint2*>(pairs), dist, n_pairs, keep, len8, col, weight));
    SQ_LAUNCH_CHECK(c);
  }
  SQ_CUDA(c, cudaStreamSynchronize(st));
  if (use_sched) c->scratch_top = top_before;           // give the scratch above the schedule back
  return SQ_OK;
}
