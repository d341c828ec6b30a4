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

size_t sq_onesweep_scratch_bytes(int64_t n, int nbatch);

size_t sq_sort_scratch_bytes(int64_t n, int nbatch) {
  int64_t ntiles = (n + kSortTile - 1) / kSortTile;
  if (ntiles < 1) ntiles = 1;
  size_t table = (size_t)ntiles * 256 * (size_t)nbatch;
  size_t nblk = (table + kScanChunk - 1) / kScanChunk + 2;
  const size_t three_kernel = sq_align_up(table * 4 + 16) + sq_align_up(nblk * 4 + 16);
  const size_t single_sweep = sq_onesweep_scratch_bytes(n, nbatch);
  return three_kernel > single_sweep ? three_kernel : single_sweep;
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

// ------------------------------ single-sweep radix passes ---------------------------------
// The LSD passes above cost three launches and read the keys twice per pass.  The digit
// histograms of ALL passes do not depend on the order of the keys, so they are taken once, up
// front; a pass is then ONE kernel: a tile ranks its 4,096 records (stable: warp-striped
// match.any ranking), publishes its per-digit counts, obtains the counts of the tiles before it
// by decoupled look-back (one thread per digit walks the predecessors' descriptors: count +
// 2 flag bits in one word), reorders the tile in shared memory and writes every digit's run
// coalesced.  Tiles take their index from a counter in the order they start running, so a tile
// only ever waits for tiles that already run.
namespace {

constexpr int kOsThreads = 512;
constexpr int kOsItems = 8;
constexpr int kOsTile = kOsThreads * kOsItems;        // 4096 records
constexpr uint32_t kOsAgg = 1u << 30, kOsPrefix = 2u << 30, kOsValue = (1u << 30) - 1u;

// hist[batch][pass][256]: one pass over the keys, all digits at once
__global__ void __launch_bounds__(256)
os_hist_kernel(const uint64_t* __restrict__ keys, int64_t n, int first_pass, int npasses,
               uint32_t* __restrict__ hist) {
  __shared__ uint32_t sh[8 * 256];
  const int batch = blockIdx.y;
  for (int t = threadIdx.x; t < npasses * 256; t += 256) sh[t] = 0u;
  __syncthreads();
  const uint64_t* __restrict__ k = keys + (int64_t)batch * n;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
    const uint64_t key = k[i];
    for (int p = 0; p < npasses; ++p)
      atomicAdd(&sh[p * 256 + (uint32_t)((key >> (8 * (first_pass + p))) & 255u)], 1u);
  }
  __syncthreads();
  for (int t = threadIdx.x; t < npasses * 256; t += 256)
    if (sh[t]) atomicAdd(&hist[((int64_t)batch * 8 + t / 256) * 256 + (t & 255)], sh[t]);
}

// in place: every 256-bin histogram -> exclusive prefix (one warp each)
__global__ void __launch_bounds__(32)
os_hist_scan_kernel(uint32_t* __restrict__ hist) {
  uint32_t* h = hist + (int64_t)blockIdx.x * 256;
  const int lane = threadIdx.x;
  uint32_t v[8], s = 0;
#pragma unroll
  for (int q = 0; q < 8; ++q) { v[q] = h[lane * 8 + q]; s += v[q]; }
  uint32_t inc = s;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, inc, d);
    if (lane >= d) inc += o;
  }
  uint32_t run = inc - s;
#pragma unroll
  for (int q = 0; q < 8; ++q) { h[lane * 8 + q] = run; run += v[q]; }
}

template <bool HAS_VALS>
__global__ void __launch_bounds__(kOsThreads, 2)
os_pass_kernel(const uint64_t* __restrict__ keys_in, uint64_t* __restrict__ keys_out,
               const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ vals_out, int64_t n,
               int pass, int shift, const uint32_t* __restrict__ hist, uint32_t* desc, uint32_t* tile_ctr,
               int ntiles) {
  extern __shared__ __align__(16) uint8_t os_smem[];
  uint64_t* skey = reinterpret_cast<uint64_t*>(os_smem);                       // [kOsTile]
  uint32_t* sval = reinterpret_cast<uint32_t*>(os_smem + (size_t)kOsTile * 8); // [kOsTile]
  uint32_t* cnt = sval + kOsTile;                                              // [8][256]
  uint32_t* dstart = cnt + (kOsThreads / 32) * 256;                            // [256] tile-local
  uint32_t* gbase = dstart + 256;                                              // [256] global
  __shared__ uint32_t sh_tile;
  __shared__ uint32_t sh_scan[kOsThreads / 32 + 1];
  const int batch = blockIdx.y;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  if (threadIdx.x == 0) sh_tile = atomicAdd(&tile_ctr[batch], 1u);
#pragma unroll
  for (int q = threadIdx.x; q < (kOsThreads / 32) * 256; q += kOsThreads) cnt[q] = 0u;
  __syncthreads();
  const uint32_t tile = sh_tile;
  const int64_t boff = (int64_t)batch * n;
  const int64_t base = (int64_t)tile * kOsTile + (int64_t)w * (32 * kOsItems);
  uint64_t key[kOsItems];
  uint32_t val[kOsItems];
  uint32_t rank[kOsItems];
#pragma unroll
  for (int it = 0; it < kOsItems; ++it) {
    const int64_t idx = base + it * 32 + lane;
    const bool ok = idx < n;
    key[it] = ok ? keys_in[boff + idx] : 0ull;
    if (HAS_VALS) val[it] = ok ? vals_in[boff + idx] : 0u;
  }
#pragma unroll
  for (int it = 0; it < kOsItems; ++it) {
    const bool ok = base + it * 32 + lane < n;
    const uint32_t d = ok ? (uint32_t)((key[it] >> shift) & 255u) : 256u;
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
    const uint32_t prev = ok ? cnt[w * 256 + d] : 0u;
    __syncwarp();
    if (ok && (peers & lt) == 0u) cnt[w * 256 + d] = prev + __popc(peers);
    __syncwarp();
    rank[it] = prev + __popc(peers & lt);
  }
  __syncthreads();
  // per digit (= thread): scan over the warps -> offset of (warp, digit) inside the digit's run
  const int d = threadIdx.x & 255;               // threads 0..255 each own one digit
  const bool owner = threadIdx.x < 256;
  uint32_t total = 0, excl = 0, inc = 0;
  if (owner) {
#pragma unroll
  for (int q = 0; q < kOsThreads / 32; ++q) { const uint32_t t = cnt[q * 256 + d]; cnt[q * 256 + d] = total; total += t; }
  // publish, then look back
  uint32_t* my = desc + ((int64_t)batch * ntiles + tile) * 256 + d;
  if (tile == 0) {
    atomicExch(my, total | kOsPrefix);
  } else {
    atomicExch(my, total | kOsAgg);
    // eight predecessors' descriptors are fetched at a time (independent loads), then read in order
    const volatile uint32_t* p = my - 256;
    uint32_t left = tile;                      // predecessors not yet looked at
    for (bool done = false; !done;) {
      uint32_t v[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) v[q] = (uint32_t)q < left ? p[-256 * q] : kOsPrefix;
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        if (!done) {
          uint32_t x = v[q];
          while ((x >> 30) == 0u) x = p[-256 * q];
          excl += x & kOsValue;
          done = (x & kOsPrefix) != 0u;
        }
      }
      p -= 256 * 8;
      left = left > 8u ? left - 8u : 0u;
    }
    atomicExch(my, (excl + total) | kOsPrefix);
  }
  gbase[d] = hist[((int64_t)batch * 8 + pass) * 256 + d] + excl;
  // tile-local start of every digit: exclusive scan of `total` over the 256 threads
  inc = total;
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, inc, s);
    if (lane >= s) inc += o;
  }
  }
  if (owner && lane == 31) sh_scan[w] = inc;
  __syncthreads();
  if (owner) {
    uint32_t woff = 0;
    for (int q = 0; q < w; ++q) woff += sh_scan[q];
    dstart[d] = woff + inc - total;
  }
  __syncthreads();
  // reorder the tile in shared memory
#pragma unroll
  for (int it = 0; it < kOsItems; ++it) {
    if (base + it * 32 + lane < n) {
      const uint32_t dg = (uint32_t)((key[it] >> shift) & 255u);
      const uint32_t pos = dstart[dg] + cnt[w * 256 + dg] + rank[it];
      skey[pos] = key[it];
      if (HAS_VALS) sval[pos] = val[it];
    }
  }
  __syncthreads();
  const int64_t tile_n = min((int64_t)kOsTile, n - (int64_t)tile * kOsTile);
#pragma unroll 4
  for (int pos = threadIdx.x; pos < tile_n; pos += kOsThreads) {
    const uint64_t kk = skey[pos];
    const uint32_t dg = (uint32_t)((kk >> shift) & 255u);
    const int64_t dst = boff + gbase[dg] + (uint32_t)(pos - dstart[dg]);
    keys_out[dst] = kk;
    if (HAS_VALS) vals_out[dst] = sval[pos];
  }
}

constexpr size_t kOsSmem = (size_t)kOsTile * 12 + (kOsThreads / 32) * 256 * 4 + 2 * 256 * 4;

}  // namespace

size_t sq_onesweep_scratch_bytes(int64_t n, int nbatch) {
  int64_t ntiles = (n + kOsTile - 1) / kOsTile;
  if (ntiles < 1) ntiles = 1;
  return sq_align_up((size_t)nbatch * 8 * 256 * 4 + 16) +             // histograms
         sq_align_up((size_t)nbatch * ntiles * 256 * 4 + 16) +        // tile descriptors
         sq_align_up((size_t)nbatch * 8 * 4 + 16);                    // tile counters, per pass
}

// Byte-wise LSD sort on the key bytes [first_pass, first_pass + npasses); same contract as
// sq_radix_sort.
int sq_onesweep_sort(sq_ctx* c, uint64_t* keys_in, uint64_t* keys_alt, uint32_t* vals_in,
                     uint32_t* vals_alt, int64_t n, int nbatch, int first_pass, int npasses, void* tmp,
                     int* result_in_alt) {
  *result_in_alt = 0;
  if (n <= 0 || nbatch <= 0 || npasses <= 0) return SQ_OK;
  if (n >= (1ll << 30) || nbatch > 65535 || first_pass < 0 || first_pass + npasses > 8) return SQ_ERR_UNSUPPORTED;
  const int64_t ntiles = (n + kOsTile - 1) / kOsTile;
  uint8_t* p = static_cast<uint8_t*>(tmp);
  uint32_t* hist = reinterpret_cast<uint32_t*>(p);      p += sq_align_up((size_t)nbatch * 8 * 256 * 4 + 16);
  uint32_t* desc = reinterpret_cast<uint32_t*>(p);      p += sq_align_up((size_t)nbatch * ntiles * 256 * 4 + 16);
  uint32_t* ctr = reinterpret_cast<uint32_t*>(p);
  cudaStream_t st = c->stream;
  SQ_CUDA(c, cudaMemsetAsync(hist, 0, (size_t)nbatch * 8 * 256 * 4, st));
  SQ_CUDA(c, cudaMemsetAsync(ctr, 0, (size_t)nbatch * 8 * 4, st));
  {
    int64_t gx = (n + 256 * 16 - 1) / (256 * 16);
    const int64_t cap = (int64_t)c->sm_count * 8 / nbatch + 1;
    if (gx > cap) gx = cap;
    dim3 grid((unsigned)gx, (unsigned)nbatch);
    SQ_TIMED(c, SQ_K_SORT_HIST, os_hist_kernel<<<grid, 256, 0, st>>>(keys_in, n, first_pass, npasses, hist));
    SQ_LAUNCH_CHECK(c);
    SQ_TIMED(c, SQ_K_SORT_HIST, os_hist_scan_kernel<<<(unsigned)(nbatch * 8), 32, 0, st>>>(hist));
    SQ_LAUNCH_CHECK(c);
  }
  // (per device and cheap: set on every call, not once per process)
  SQ_CUDA(c, cudaFuncSetAttribute(os_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kOsSmem));
  SQ_CUDA(c, cudaFuncSetAttribute(os_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kOsSmem));
  uint64_t* kin = keys_in; uint64_t* kout = keys_alt;
  uint32_t* vin = vals_in; uint32_t* vout = vals_alt;
  dim3 grid((unsigned)ntiles, (unsigned)nbatch);
  for (int pass = 0; pass < npasses; ++pass) {
    SQ_CUDA(c, cudaMemsetAsync(desc, 0, (size_t)nbatch * ntiles * 256 * 4, st));
    if (vals_in)
      SQ_TIMED(c, SQ_K_SORT_SCATTER, os_pass_kernel<true><<<grid, kOsThreads, kOsSmem, st>>>(
          kin, kout, vin, vout, n, pass, 8 * (first_pass + pass), hist, desc, ctr + (size_t)pass * nbatch,
          (int)ntiles));
    else
      SQ_TIMED(c, SQ_K_SORT_SCATTER, os_pass_kernel<false><<<grid, kOsThreads, kOsSmem, st>>>(
          kin, kout, nullptr, nullptr, n, pass, 8 * (first_pass + pass), hist, desc,
          ctr + (size_t)pass * nbatch, (int)ntiles));
    SQ_LAUNCH_CHECK(c);
    uint64_t* tk = kin; kin = kout; kout = tk;
    uint32_t* tv = vin; vin = vout; vout = tv;
    *result_in_alt ^= 1;
  }
  return SQ_OK;
}
