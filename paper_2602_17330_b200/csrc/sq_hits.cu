// sq_hits.cu -- a6 with compacted hits: sq_edit_distance followed by an order-preserving
// compaction of the pairs with d <= max_d (north_star (d): "warp-ballot compaction of hits";
// SURVEY.md 8(a) a6 "(+ optional compacted hits)"; App. F.3).
//
//   hits_count_kernel    one block per tile of 2,048 pairs: number of hits of the tile
//   hits_scan_kernel     one block: exclusive scan of the tile counts (+ the total)
//   hits_scatter_kernel  one block per tile: warp ballots + popc rank every hit inside the tile;
//                        hit k of the list is the k-th hit in input order (deterministic)
//
// The only scratch is one word per tile.  Two entry points share the kernels:
//   sq_edit_distance_hits         scratch from the caller's workspace (any n_pairs)
//   sq_edit_distance_hits_static  scratch in a file-scope __device__ array: allocates nothing and needs
//                                 no free workspace, for callers that cannot allocate (code under CUDA
//                                 graph capture, tight serving loops); n_pairs <= SQ_HITS_STATIC_MAX_PAIRS
#include "sq_common.cuh"
#include <mutex>

namespace {

constexpr int kHtThreads = 256;
constexpr int kHtItems = 8;
constexpr int kHtTile = kHtThreads * kHtItems;                       // pairs per tile
constexpr int kStaticWords = (int)(SQ_HITS_STATIC_MAX_PAIRS / kHtTile) + 8;   // 65,544 words = 256 KB

// Scratch of sq_edit_distance_hits_static.  Every GPU that loads the library holds these 256 KB until
// the process exits.  All calls share it and it keeps the last call's contents: a call overwrites the
// words it reads (tile counts [0, ntiles) and the total at [ntiles]) before reading them, so nothing
// has to start at zero -- but two calls that overlap on the GPU (different streams) race on it.
static __device__ __align__(256) uint32_t g_hits_scratch[kStaticWords];

__device__ __forceinline__ bool is_hit(uint16_t d, int max_d) { return (int)d <= max_d; }

__global__ void __launch_bounds__(kHtThreads)
hits_count_kernel(const uint16_t* __restrict__ dist, int64_t n, int max_d, uint32_t* __restrict__ counts) {
  __shared__ uint32_t wsum[kHtThreads / 32];
  const int64_t base = (int64_t)blockIdx.x * kHtTile;
  uint32_t c = 0;
#pragma unroll
  for (int k = 0; k < kHtItems; ++k) {
    const int64_t p = base + (int64_t)k * kHtThreads + threadIdx.x;
    if (p < n && is_hit(dist[p], max_d)) ++c;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, d);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int w = 0; w < kHtThreads / 32; ++w) t += wsum[w];
    counts[blockIdx.x] = t;
  }
}

// counts[0 .. ntiles) -> exclusive offsets (64-bit running total kept in registers; an offset that
// does not fit 32 bits can only belong to a hit beyond any capacity < 2^32 and is clamped);
// counts[ntiles], counts[ntiles + 1] = the total (lo, hi)
__global__ void __launch_bounds__(1024)
hits_scan_kernel(uint32_t* __restrict__ counts, int64_t ntiles) {
  __shared__ unsigned long long wtot[32];
  __shared__ unsigned long long carry_sh;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_sh = 0ull;
  __syncthreads();
  for (int64_t t0 = 0; t0 < ntiles; t0 += 1024) {
    const int64_t t = t0 + threadIdx.x;
    const unsigned long long v = t < ntiles ? counts[t] : 0u;
    unsigned long long inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const unsigned long long o = __shfl_up_sync(0xFFFFFFFFu, inc, d);
      if (lane >= d) inc += o;
    }
    if (lane == 31) wtot[w] = inc;
    __syncthreads();
    unsigned long long before = carry_sh;
    for (int q = 0; q < w; ++q) before += wtot[q];
    const unsigned long long ex = before + inc - v;
    if (t < ntiles) counts[t] = ex > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)ex;
    __syncthreads();
    if (threadIdx.x == 1023) carry_sh = before + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    counts[ntiles] = (uint32_t)(carry_sh & 0xFFFFFFFFull);
    counts[ntiles + 1] = (uint32_t)(carry_sh >> 32);
  }
}

// hit k of the output = the k-th hit in input order.  Rank inside the tile: the tile is 8 rows of 256
// consecutive pairs; a warp's ballot ranks its 32 pairs, a 64-entry table ranks the (row, warp) pieces.
__global__ void __launch_bounds__(kHtThreads)
hits_scatter_kernel(const uint2* __restrict__ pairs, const uint16_t* __restrict__ dist, int64_t n, int max_d,
                    const uint32_t* __restrict__ offsets, uint2* __restrict__ hit_pairs,
                    uint16_t* __restrict__ hit_dist, unsigned long long capacity) {
  __shared__ uint32_t piece[kHtItems * (kHtThreads / 32) + 1];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t base = (int64_t)blockIdx.x * kHtTile;
  uint32_t masks[kHtItems];
  uint16_t dv[kHtItems];
#pragma unroll
  for (int k = 0; k < kHtItems; ++k) {
    const int64_t p = base + (int64_t)k * kHtThreads + threadIdx.x;
    dv[k] = p < n ? dist[p] : (uint16_t)0xFFFFu;
    const bool h = p < n && is_hit(dv[k], max_d);
    masks[k] = __ballot_sync(0xFFFFFFFFu, h);
    if (lane == 0) piece[k * (kHtThreads / 32) + w] = (uint32_t)__popc(masks[k]);
  }
  __syncthreads();
  if (threadIdx.x == 0) {                       // exclusive scan of the 64 pieces (input order: row, then warp)
    uint32_t run = 0;
    for (int q = 0; q < kHtItems * (kHtThreads / 32); ++q) { const uint32_t v = piece[q]; piece[q] = run; run += v; }
  }
  __syncthreads();
  const unsigned long long tile_off = offsets[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kHtItems; ++k) {
    if ((masks[k] >> lane) & 1u) {
      const int64_t p = base + (int64_t)k * kHtThreads + threadIdx.x;
      const unsigned long long at = tile_off + piece[k * (kHtThreads / 32) + w] +
                                    (uint32_t)__popc(masks[k] & ((1u << lane) - 1u));
      if (at < capacity) { hit_pairs[at] = pairs[p]; hit_dist[at] = dv[k]; }
    }
  }
}

// distances -> compacted hits, `counts` = ntiles + 2 words of scratch (device pointer)
int hits_core(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d, uint16_t* dist_out,
              uint32_t* hit_pairs, uint16_t* hit_dist, int64_t capacity, uint32_t* counts, int64_t* n_hits) {
  int rc = sq_edit_distance_impl(c, pairs, n_pairs, max_d, dist_out);
  if (rc != SQ_OK) return rc;
  const int64_t ntiles = (n_pairs + kHtTile - 1) / kHtTile;
  cudaStream_t st = c->stream;
  SQ_TIMED(c, SQ_K_MISC, hits_count_kernel<<<(unsigned)ntiles, kHtThreads, 0, st>>>(dist_out, n_pairs, max_d, counts));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_MISC, hits_scan_kernel<<<1, 1024, 0, st>>>(counts, ntiles));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_MISC, hits_scatter_kernel<<<(unsigned)ntiles, kHtThreads, 0, st>>>(
      reinterpret_cast<const uint2*>(pairs), dist_out, n_pairs, max_d, counts, reinterpret_cast<uint2*>(hit_pairs),
      hit_dist, (unsigned long long)capacity));
  SQ_LAUNCH_CHECK(c);
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, counts + ntiles, 8, cudaMemcpyDeviceToHost, st));
  SQ_CUDA(c, cudaStreamSynchronize(st));
  *n_hits = (int64_t)c->pinned[0];
  return *n_hits > capacity ? SQ_ERR_CAPACITY : SQ_OK;
}

int hits_check(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d, uint16_t* dist_out,
               uint32_t* hit_pairs, uint16_t* hit_dist, int64_t capacity, int64_t* n_hits) {
  if (!c || !n_hits) return SQ_ERR_INVALID_ARG;
  *n_hits = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (n_pairs < 0 || capacity < 0 || max_d < 0 || max_d > 65534) return SQ_ERR_INVALID_ARG;
  if (n_pairs > 0 && (!pairs || !dist_out)) return SQ_ERR_INVALID_ARG;
  if (capacity > 0 && (!hit_pairs || !hit_dist)) return SQ_ERR_INVALID_ARG;
  if (n_pairs >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;        // 32-bit tile offsets
  return SQ_OK;
}

// device address of g_hits_scratch, looked up once per device with that device current (in host code
// the array's name is a host-side stand-in, not a device address)
constexpr int kMaxDevices = 64;
std::mutex g_sym_mutex;
uint32_t* g_sym_addr[kMaxDevices] = {nullptr};

int static_scratch(sq_ctx* c, uint32_t** out) {
  if (c->device < 0 || c->device >= kMaxDevices) return SQ_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_sym_mutex);
  if (!g_sym_addr[c->device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_hits_scratch);   // the context's device is current (guard)
    if (e != cudaSuccess || !p) { c->last_err = e; return SQ_ERR_CUDA; }
    g_sym_addr[c->device] = static_cast<uint32_t*>(p);
  }
  *out = g_sym_addr[c->device];
  return SQ_OK;
}

}  // namespace

extern "C" int sq_edit_distance_hits(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                                     uint16_t* dist_out, uint32_t* hit_pairs_out, uint16_t* hit_dist_out,
                                     int64_t capacity, int64_t* n_hits) {
  int rc = hits_check(c, pairs, n_pairs, max_d, dist_out, hit_pairs_out, hit_dist_out, capacity, n_hits);
  if (rc != SQ_OK || n_pairs == 0) return rc;
  SqDeviceGuard guard(c);
  // one word per tile above whatever the scratch holds (the schedule of sq_lsh_candidates stays valid)
  const size_t top = c->scratch_top;
  uint32_t* counts = sq_scratch<uint32_t>(c, (size_t)((n_pairs + kHtTile - 1) / kHtTile) + 2);
  c->scratch_top = top;
  if (!counts) return SQ_ERR_WORKSPACE;
  return hits_core(c, pairs, n_pairs, max_d, dist_out, hit_pairs_out, hit_dist_out, capacity, counts, n_hits);
}

extern "C" int sq_edit_distance_hits_static(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                                            uint16_t* dist_out, uint32_t* hit_pairs_out,
                                            uint16_t* hit_dist_out, int64_t capacity, int64_t* n_hits) {
  int rc = hits_check(c, pairs, n_pairs, max_d, dist_out, hit_pairs_out, hit_dist_out, capacity, n_hits);
  if (rc != SQ_OK || n_pairs == 0) return rc;
  if (n_pairs > SQ_HITS_STATIC_MAX_PAIRS) return SQ_ERR_UNSUPPORTED;   // beyond the static scratch
  SqDeviceGuard guard(c);
  uint32_t* counts = nullptr;
  if ((rc = static_scratch(c, &counts)) != SQ_OK) return rc;
  return hits_core(c, pairs, n_pairs, max_d, dist_out, hit_pairs_out, hit_dist_out, capacity, counts, n_hits);
}
