// sq_minhash.cu -- step a2: k-mer MinHash sketch (Alg. 1 step 1 "compute MinHash
// sketches"; sketch sizes {64,128,256} L269; hash family = spec C2, see include/subquad.h).
//
// One thread per (sequence, chunk of HT hashes).  The thread rolls the k-mer value over its
// sequence (5 bits per residue), mixes it once with g(), and keeps HT running minima in
// registers: one IMAD (fma pipe) + one unsigned min (alu pipe) per (k-mer, hash).  The per-hash
// multipliers/offsets sit in the kernel parameter block, i.e. the constant bank, and are read
// as instruction operands.  Sequences are visited longest-first (order[] from sq_pack) so the 32
// lanes of a warp run (nearly) the same trip count.  The HT minima of 32 sequences are
// transposed through shared memory so that every store instruction of a warp writes one full,
// contiguous 128-byte line of a signature row.
//
// Roofline: bytes/sequence = stride (slot read) + 4 (order) + 4*H (signature write);
// instructions/sequence ~ (len-k+1) * (2*H + ~10).  At H=64 the two are within ~1.3x of each
// other on B200, so the kernel is reported against both.
#include "sq_common.cuh"

namespace {

struct HashParams {
  uint32_t a[SQ_MAX_H];
  uint32_t b[SQ_MAX_H];
};

__host__ __device__ __forceinline__ uint32_t sq_mix32(uint32_t x) {
  x ^= x >> 16;
  x *= 0x6A09E667u;
  x ^= x >> 15;
  x *= 0xBB67AE85u;
  x ^= x >> 16;
  return x;
}

constexpr int kMhThreads = 128;

template <int HT>
__global__ void __launch_bounds__(kMhThreads)
minhash_kernel(const uint8_t* __restrict__ packed, int stride, const uint32_t* __restrict__ order,
               int64_t n, int k, int H, const __grid_constant__ HashParams hp,
               uint32_t* __restrict__ sig) {
  __shared__ uint32_t stage[kMhThreads / 32][32][HT + 1];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t t = (int64_t)blockIdx.x * kMhThreads + threadIdx.x;
  const int hbase = blockIdx.y * HT;
  uint32_t m[HT];
#pragma unroll
  for (int j = 0; j < HT; ++j) m[j] = SQ_EMPTY_SIG;
  uint32_t id = 0;
  if (t < n) {
    id = order[t];
    const uint8_t* row = packed + (int64_t)id * stride;
    const int len = row[stride - 1];
    const uint32_t kmask = (k * 5 >= 32) ? 0xFFFFFFFFu : ((1u << (5 * k)) - 1u);
    const uint32_t* row32 = reinterpret_cast<const uint32_t*>(row);
    uint32_t x = 0;
    for (int wi = 0; wi * 4 < len; ++wi) {
      const uint32_t word = row32[wi];
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int pos = wi * 4 + b;
        if (pos >= len) break;
        x = ((x << 5) | ((word >> (8 * b)) & 31u)) & kmask;
        if (pos >= k - 1) {
          const uint32_t y = sq_mix32(x);
#pragma unroll
          for (int j = 0; j < HT; ++j) m[j] = min(m[j], hp.a[hbase + j] * y + hp.b[hbase + j]);
        }
      }
    }
  }
  // transpose through shared memory: lane l then writes column l of each of the warp's rows
#pragma unroll
  for (int j = 0; j < HT; ++j) stage[w][lane][j] = m[j];
  __syncwarp();
  const int64_t tw = (int64_t)blockIdx.x * kMhThreads + w * 32;   // first rank of this warp
  for (int r = 0; r < 32; ++r) {
    if (tw + r >= n) break;
    const uint32_t rid = __shfl_sync(0xFFFFFFFFu, id, r);
    uint32_t* dst = sig + (int64_t)rid * H + hbase;
#pragma unroll
    for (int j = lane; j < HT; j += 32) dst[j] = stage[w][r][j];
  }
}

}  // namespace

int sq_minhash_impl(sq_ctx* c, int k, int H, uint64_t seed, uint32_t* sig_out) {
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (k < 1 || 5 * k > 32 || H < 32 || (H % 32) != 0) return SQ_ERR_INVALID_ARG;
  if (H > SQ_MAX_H) return SQ_ERR_UNSUPPORTED;
  if (c->n == 0) return SQ_OK;
  if (!sig_out) return SQ_ERR_INVALID_ARG;
  HashParams hp;
  const uint32_t lo = (uint32_t)(seed & 0xFFFFFFFFull), hi = (uint32_t)(seed >> 32);
  for (int j = 0; j < SQ_MAX_H; ++j) {
    hp.a[j] = sq_mix32(lo ^ sq_mix32((uint32_t)(2 * j + 1))) | 1u;
    hp.b[j] = sq_mix32(hi ^ sq_mix32((uint32_t)(2 * j + 2)));
  }
  const unsigned gx = (unsigned)((c->n + kMhThreads - 1) / kMhThreads);
  if (H % 64 == 0) {
    dim3 grid(gx, H / 64);
    SQ_TIMED(c, SQ_K_MINHASH, minhash_kernel<64><<<grid, kMhThreads, 0, c->stream>>>(
        c->packed, c->stride, c->order, c->n, k, H, hp, sig_out));
  } else {
    dim3 grid(gx, H / 32);
    SQ_TIMED(c, SQ_K_MINHASH, minhash_kernel<32><<<grid, kMhThreads, 0, c->stream>>>(
        c->packed, c->stride, c->order, c->n, k, H, hp, sig_out));
  }
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}
