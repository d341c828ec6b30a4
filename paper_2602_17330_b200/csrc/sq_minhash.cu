// sq_minhash.cu -- step a2: k-mer MinHash sketch (Alg. 1 step 1 "compute MinHash
// sketches"; sketch sizes {64,128,256} L269; hash family = spec C2, see include/subquad.h).
//
// One thread per (sequence, chunk of HT hashes), kMhIters sequences per thread one after the
// other.  The thread rolls the k-mer value over its sequence (5 bits per residue), mixes it once
// with g(), and keeps HT running minima in registers: one IMAD (fma pipe) + one unsigned min (alu
// pipe) per (k-mer, hash) and nothing else -- the chunk's HT multipliers a_j are copied into
// registers once per thread and its offsets b_j sit at compile-time addresses of the kernel
// parameter block (which holds exactly the chunk's parameters; one launch per chunk), so an
// update needs no load or address of its own (2.4 issued instructions per update; 3.9 when the
// parameters were indexed by blockIdx.y).  Sequences are visited longest-first (order[] from
// sq_pack) so the 32 lanes of a warp run (nearly) the same trip count.  Loads are software
// pipelined: the next 4 residues of the slot, and the slot of the thread's NEXT sequence, are in
// flight behind the current word's 4 x HT updates.  The HT minima leave as HT/8 32-byte stores
// (STG.256, one whole sector each) straight into the thread's signature row: no shared-memory
// transpose (16-byte stores -- half sectors -- were slower than the transpose, 32-byte ones are
// faster).  Config 4: 1.42 -> 1.08 ms.
//
// Roofline: bytes/sequence = stride (slot read) + 4 (order) + 4*H (signature write);
// instructions/sequence ~ (len-k+1) * (2*H + ~20).  At H=64 the two are within ~1.3x of each
// other on B200, so the kernel is reported against both.
#include "sq_common.cuh"

namespace {

template <int HT>
struct HashChunk {            // parameters of hashes [hbase, hbase + HT)
  uint32_t a[HT];
  uint32_t b[HT];
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
constexpr int kMhIters = 4;      // sequences per thread (the next one's loads fly behind the current one's updates)

template <int HT, int MINB>
__global__ void __launch_bounds__(kMhThreads, MINB)
minhash_kernel(const uint8_t* __restrict__ packed, int stride, const uint32_t* __restrict__ order,
               int64_t n, int k, int H, int hbase, const __grid_constant__ HashChunk<HT> hp,
               uint32_t* __restrict__ sig, int iters) {
  uint32_t a[HT];
#pragma unroll
  for (int j = 0; j < HT; ++j)
    asm volatile("mov.u32 %0, %1;" : "=r"(a[j]) : "r"(hp.a[j]));     // pinned to a register
  const uint32_t kmask = (k * 5 >= 32) ? 0xFFFFFFFFu : ((1u << (5 * k)) - 1u);
  const int lastw = stride / 4 - 1;                                  // word holding the length byte
  int64_t t = (int64_t)blockIdx.x * (kMhThreads * iters) + threadIdx.x;
  if (t >= n) return;
  uint32_t id = order[t];
  const uint32_t* row32 = reinterpret_cast<const uint32_t*>(packed + (int64_t)id * stride);
  uint32_t next = row32[0], lenw = row32[lastw];
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
    const int64_t t2 = t + kMhThreads;
    const bool more = it + 1 < iters && t2 < n;
    const uint32_t id2 = more ? order[t2] : 0u;                      // needed one word of updates later
    const uint32_t* row2 = row32;
    uint32_t next2 = 0u, lenw2 = 0u;
    const int len = (int)(lenw >> 24);
    uint32_t m[HT];
#pragma unroll
    for (int j = 0; j < HT; ++j) m[j] = SQ_EMPTY_SIG;
    uint32_t x = 0;
    for (int wi = 0; wi * 4 < len || wi < 2; ++wi) {
      if (wi == 1 && more) {                                         // the next sequence's slot
        row2 = reinterpret_cast<const uint32_t*>(packed + (int64_t)id2 * stride);
        next2 = row2[0];
        lenw2 = row2[lastw];
      }
      const uint32_t word = next;
      if (wi < lastw) next = row32[wi + 1];                          // in flight behind this word's updates
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int pos = wi * 4 + b;
        if (pos >= len) break;
        x = ((x << 5) | ((word >> (8 * b)) & 31u)) & kmask;
        if (pos >= k - 1) {
          const uint32_t y = sq_mix32(x);
#pragma unroll
          for (int j = 0; j < HT; ++j) m[j] = min(m[j], a[j] * y + hp.b[j]);
        }
      }
    }
    // the thread's HT minima are HT/8 32-byte stores (STG.256) into its own signature row: every
    // store writes one whole sector, nothing is staged or transposed
    uint32_t* dst = sig + (int64_t)id * H + hbase;
#pragma unroll
    for (int j = 0; j < HT; j += 8)
      asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(dst + j), "r"(m[j]),
                   "r"(m[j + 1]), "r"(m[j + 2]), "r"(m[j + 3]), "r"(m[j + 4]), "r"(m[j + 5]), "r"(m[j + 6]),
                   "r"(m[j + 7]) : "memory");
    if (!more) break;
    t = t2; id = id2; row32 = row2; next = next2; lenw = lenw2;
  }
}

}  // namespace

int sq_minhash_impl(sq_ctx* c, int k, int H, uint64_t seed, uint32_t* sig_out) {
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (k < 1 || 5 * k > 32 || H < 32 || (H % 32) != 0) return SQ_ERR_INVALID_ARG;
  if (H > SQ_MAX_H) return SQ_ERR_UNSUPPORTED;
  if (c->n == 0) return SQ_OK;
  if (!sig_out || ((uintptr_t)sig_out & 31u)) return SQ_ERR_INVALID_ARG;
  const uint32_t lo = (uint32_t)(seed & 0xFFFFFFFFull), hi = (uint32_t)(seed >> 32);
  const int iters = kMhIters;
  const int64_t per_block = (int64_t)kMhThreads * iters;
  const unsigned gx = (unsigned)((c->n + per_block - 1) / per_block);
  if (H % 64 == 0) {
    for (int hbase = 0; hbase < H; hbase += 64) {
      HashChunk<64> hp;
      for (int j = 0; j < 64; ++j) {
        hp.a[j] = sq_mix32(lo ^ sq_mix32((uint32_t)(2 * (hbase + j) + 1))) | 1u;
        hp.b[j] = sq_mix32(hi ^ sq_mix32((uint32_t)(2 * (hbase + j) + 2)));
      }
      SQ_TIMED(c, SQ_K_MINHASH, minhash_kernel<64, 3><<<gx, kMhThreads, 0, c->stream>>>(
          c->packed, c->stride, c->order, c->n, k, H, hbase, hp, sig_out, iters));
      SQ_LAUNCH_CHECK(c);
    }
    return SQ_OK;
  }
  for (int hbase = 0; hbase < H; hbase += 32) {
    HashChunk<32> hp;
    for (int j = 0; j < 32; ++j) {
      hp.a[j] = sq_mix32(lo ^ sq_mix32((uint32_t)(2 * (hbase + j) + 1))) | 1u;
      hp.b[j] = sq_mix32(hi ^ sq_mix32((uint32_t)(2 * (hbase + j) + 2)));
    }
    SQ_TIMED(c, SQ_K_MINHASH, minhash_kernel<32, 6><<<gx, kMhThreads, 0, c->stream>>>(
        c->packed, c->stride, c->order, c->n, k, H, hbase, hp, sig_out, iters));
    SQ_LAUNCH_CHECK(c);
  }
  return SQ_OK;
}
