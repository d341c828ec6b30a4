// sq_sort.cu -- hand-written device-wide primitives used by the bucketing stage (step a4) and
// by the final ordering of pair lists: an exclusive prefix sum and a stable LSD radix sort of
// (uint64 key [, uint32 value]) records, batched over independent arrays (one per LSH band).
//
// Radix pass = 3 launches: per-tile digit histogram -> exclusive scan of the [batch][digit][tile]
// table -> stable scatter.  Stability inside a tile comes from a warp-striped arrangement
// (warp w owns a contiguous run of the tile) ranked with match.any + per-warp digit counters.
// HBM-bound: each pass reads the keys twice and the values once, and writes both once.
#include "sq_common.cuh"

namespace {

constexpr int kSortThreads = 256;
constexpr int kSortItems = 8;                       // keys per thread
constexpr int kSortTile = kSortThreads * kSortItems;  // 2048 keys per block
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanChunk = kScanThreads * kScanItems;  // 2048

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t t = __shfl_up_sync(0xFFFFFFFFu, v, d);
    if (lane >= d) v += t;
  }
  return v;
}

// block-wide exclusive scan of one value per thread (256 threads); returns exclusive prefix,
// *total gets the block sum.  `sh` needs 9 words.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* sh, uint32_t* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t inc = warp_incl_scan(v, lane);
  if (lane == 31) sh[w] = inc;
  __syncthreads();
  if (w == 0) {
    uint32_t s = lane < (kScanThreads / 32) ? sh[lane] : 0;
    uint32_t si = warp_incl_scan(s, lane);
    if (lane < (kScanThreads / 32)) sh[lane] = si - s;
    if (lane == (kScanThreads / 32) - 1) sh[8] = si;
  }
  __syncthreads();
  uint32_t res = inc - v + sh[w];
  *total = sh[8];
  __syncthreads();
  return res;
}

__global__ void __launch_bounds__(kScanThreads)
scan_reduce_kernel(const uint32_t* __restrict__ in, int64_t n, uint32_t* __restrict__ block_sums) {
  __shared__ uint32_t sh[9];
  const int64_t base = (int64_t)blockIdx.x * kScanChunk;
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    int64_t idx = base + k * kScanThreads + threadIdx.x;
    if (idx < n) s += in[idx];
  }
  uint32_t tot;
  block_excl_scan(s, sh, &tot);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = tot;
}

// single block: exclusive scan of block_sums in place; writes the grand total
__global__ void __launch_bounds__(kScanThreads)
scan_spine_kernel(uint32_t* __restrict__ block_sums, int64_t nblk,
                  unsigned long long* __restrict__ total_out) {
  __shared__ uint32_t sh[9];
  unsigned long long carry = 0;    // the grand total is kept in 64 bits so a wrap is detectable
  for (int64_t base = 0; base < nblk; base += kScanThreads) {
    int64_t idx = base + threadIdx.x;
    uint32_t v = idx < nblk ? block_sums[idx] : 0;
    uint32_t tot;
    uint32_t ex = block_excl_scan(v, sh, &tot);
    if (idx < nblk) block_sums[idx] = ex + (uint32_t)carry;
    carry += tot;
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(kScanThreads)
scan_apply_kernel(const uint32_t* in, uint32_t* out, int64_t n,
                  const uint32_t* __restrict__ block_offs) {
  __shared__ uint32_t sh[9];
  const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
  uint32_t v[kScanItems];
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    v[k] = (base + k < n) ? in[base + k] : 0;
    s += v[k];
  }
  uint32_t tot;
  uint32_t ex = block_excl_scan(s, sh, &tot) + block_offs[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < n) out[base + k] = ex;
    ex += v[k];
  }
}

// ------------------------------ radix sort ------------------------------------------------

__global__ void __launch_bounds__(kSortThreads)
radix_hist_kernel(const uint64_t* __restrict__ keys, int64_t n, int shift, uint32_t mask,
                  uint32_t* __restrict__ tile_hist, int ntiles) {
  __shared__ uint32_t hist[256];
  const int batch = blockIdx.y;
  hist[threadIdx.x] = 0;
  __syncthreads();
  const uint64_t* k = keys + (int64_t)batch * n;
  const int64_t base = (int64_t)blockIdx.x * kSortTile;
#pragma unroll
  for (int it = 0; it < kSortItems; ++it) {
    int64_t idx = base + it * kSortThreads + threadIdx.x;
    if (idx < n) atomicAdd(&hist[(uint32_t)(k[idx] >> shift) & mask], 1u);
  }
  __syncthreads();
  tile_hist[((int64_t)batch * 256 + threadIdx.x) * ntiles + blockIdx.x] = hist[threadIdx.x];
}

template <bool HAS_VALS>
__global__ void __launch_bounds__(kSortThreads)
radix_scatter_kernel(const uint64_t* __restrict__ keys_in, uint64_t* __restrict__ keys_out,
                     const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ vals_out,
                     int64_t n, int shift, uint32_t mask, const uint32_t* __restrict__ tile_offs,
                     int ntiles) {
  __shared__ uint32_t cnt[kSortThreads / 32][256];
  const int batch = blockIdx.y;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
  for (int q = 0; q < kSortThreads / 32; ++q) cnt[q][threadIdx.x] = 0;
  __syncthreads();
  const int64_t boff = (int64_t)batch * n;
  const int64_t base = (int64_t)blockIdx.x * kSortTile + w * (32 * kSortItems);
  uint64_t key[kSortItems];
  uint32_t val[kSortItems];
  uint32_t rank[kSortItems];
#pragma unroll
  for (int it = 0; it < kSortItems; ++it) {
    int64_t idx = base + it * 32 + lane;
    bool valid = idx < n;
    key[it] = valid ? keys_in[boff + idx] : 0;
    if (HAS_VALS) val[it] = valid ? vals_in[boff + idx] : 0;
  }
#pragma unroll
  for (int it = 0; it < kSortItems; ++it) {
    int64_t idx = base + it * 32 + lane;
    bool valid = idx < n;
    uint32_t d = valid ? ((uint32_t)(key[it] >> shift) & mask) : 256u;
    uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
    uint32_t prev = valid ? cnt[w][d] : 0;
    __syncwarp();
    if (valid && (peers & lt) == 0) cnt[w][d] = prev + __popc(peers);
    __syncwarp();
    rank[it] = prev + __popc(peers & lt);
  }
  __syncthreads();
  {  // per digit (= thread): exclusive scan over the warps, seeded with the global tile offset
    const int d = threadIdx.x;
    // tile_offs is the scan over the whole [batch][digit][tile] table: subtract the batch base
    uint32_t run = tile_offs[((int64_t)batch * 256 + d) * ntiles + blockIdx.x] -
                   tile_offs[((int64_t)batch * 256) * ntiles];
#pragma unroll
    for (int q = 0; q < kSortThreads / 32; ++q) {
      uint32_t t = cnt[q][d];
      cnt[q][d] = run;
      run += t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int it = 0; it < kSortItems; ++it) {
    int64_t idx = base + it * 32 + lane;
    if (idx < n) {
      uint32_t d = (uint32_t)(key[it] >> shift) & mask;
      int64_t dst = boff + cnt[w][d] + rank[it];
      keys_out[dst] = key[it];
      if (HAS_VALS) vals_out[dst] = val[it];
    }
  }
}

}  // namespace

size_t sq_sort_scratch_bytes(int64_t n, int nbatch) {
  int64_t ntiles = (n + kSortTile - 1) / kSortTile;
  if (ntiles < 1) ntiles = 1;
  size_t table = (size_t)ntiles * 256 * (size_t)nbatch;
  size_t nblk = (table + kScanChunk - 1) / kScanChunk + 2;
  return sq_align_up(table * 4 + 16) + sq_align_up(nblk * 4 + 16);
}

int sq_exclusive_scan_u32(sq_ctx* c, const uint32_t* in, uint32_t* out, int64_t n, uint32_t* tmp,
                          unsigned long long* total_out_dev) {
  if (n <= 0) {
    if (total_out_dev) SQ_CUDA(c, cudaMemsetAsync(total_out_dev, 0, 8, c->stream));
    return SQ_OK;
  }
  int64_t nblk = (n + kScanChunk - 1) / kScanChunk;
  SQ_TIMED(c, SQ_K_SCAN, scan_reduce_kernel<<<(unsigned)nblk, kScanThreads, 0, c->stream>>>(in, n, tmp));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SCAN, scan_spine_kernel<<<1, kScanThreads, 0, c->stream>>>(tmp, nblk, total_out_dev));
  SQ_LAUNCH_CHECK(c);
  SQ_TIMED(c, SQ_K_SCAN, scan_apply_kernel<<<(unsigned)nblk, kScanThreads, 0, c->stream>>>(in, out, n, tmp));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int sq_radix_sort(sq_ctx* c, uint64_t* keys_in, uint64_t* keys_alt, uint32_t* vals_in,
                  uint32_t* vals_alt, int64_t n, int nbatch, const int* shifts, const int* widths,
                  int npasses, void* tmp, int* result_in_alt) {
  *result_in_alt = 0;
  if (n <= 0 || nbatch <= 0 || npasses <= 0) return SQ_OK;
  if (n >= (1ll << 32) - 1 || nbatch > 65535) return SQ_ERR_UNSUPPORTED;
  const int64_t ntiles = (n + kSortTile - 1) / kSortTile;
  const size_t table = (size_t)ntiles * 256 * (size_t)nbatch;
  uint32_t* tile_hist = static_cast<uint32_t*>(tmp);
  uint32_t* scan_tmp = reinterpret_cast<uint32_t*>(static_cast<uint8_t*>(tmp) +
                                                  sq_align_up(table * 4 + 16));
  uint64_t* kin = keys_in; uint64_t* kout = keys_alt;
  uint32_t* vin = vals_in; uint32_t* vout = vals_alt;
  dim3 grid((unsigned)ntiles, (unsigned)nbatch);
  for (int p = 0; p < npasses; ++p) {
    const uint32_t mask = (1u << widths[p]) - 1u;
    SQ_TIMED(c, SQ_K_SORT_HIST, radix_hist_kernel<<<grid, kSortThreads, 0, c->stream>>>(
        kin, n, shifts[p], mask, tile_hist, (int)ntiles));
    SQ_LAUNCH_CHECK(c);
    int rc = sq_exclusive_scan_u32(c, tile_hist, tile_hist, (int64_t)table, scan_tmp, nullptr);
    if (rc != SQ_OK) return rc;
    if (vals_in)
      SQ_TIMED(c, SQ_K_SORT_SCATTER, radix_scatter_kernel<true><<<grid, kSortThreads, 0, c->stream>>>(
          kin, kout, vin, vout, n, shifts[p], mask, tile_hist, (int)ntiles));
    else
      SQ_TIMED(c, SQ_K_SORT_SCATTER, radix_scatter_kernel<false><<<grid, kSortThreads, 0, c->stream>>>(
          kin, kout, nullptr, nullptr, n, shifts[p], mask, tile_hist, (int)ntiles));
    SQ_LAUNCH_CHECK(c);
    uint64_t* tk = kin; kin = kout; kout = tk;
    uint32_t* tv = vin; vin = vout; vout = tv;
    *result_in_alt ^= 1;
  }
  return SQ_OK;
}
