// sq_pack.cu -- step a1: validate residue codes and copy the sequences into the fixed-stride,
// 16-byte aligned slot layout every later kernel reads (App. F.2: "contiguous
// memory blocks with proper alignment to enable coalesced global memory access"; L157
// "trim/pad").  Also builds the longest-first processing order used by the sketch kernel.
//
// Slot layout (stride = round_up(max_len+1, 16) bytes):
//   [0, len)  residue codes   [len, stride-1)  0xFF   [stride-1]  len
// HBM-bound: reads total_len + 8(n+1) bytes, writes n*stride bytes.
#include "sq_common.cuh"

size_t sq_pack_scratch_bytes(int64_t n) {
  size_t nn = (size_t)(n > 0 ? n : 1);
  return 2 * sq_align_up(nn * 8 + 16) + 2 * sq_align_up(nn * 4 + 16) + sq_sort_scratch_bytes(n, 1);
}

size_t sq_persist_bytes(int64_t n, int max_len) {
  size_t nn = (size_t)(n > 0 ? n : 1);
  // packed slots + order; the pack's own scratch is accounted here too so that every op's
  // workspace (persist + op scratch) is always large enough to run sq_pack first
  return sq_align_up(nn * sq_stride_for(max_len) + 16) + sq_align_up(nn * 4 + 16) +
         sq_pack_scratch_bytes(n);
}

// One thread per (sequence, 16-byte chunk): coalesced 16-byte stores; source bytes are read
// with byte loads (the source is unaligned) that hit L1 after the first touch of a sector.
__global__ void __launch_bounds__(256)
pack_kernel(const uint8_t* __restrict__ seqs, const int64_t* __restrict__ off, int64_t n,
            int alphabet, int max_len, int stride, uint8_t* __restrict__ packed,
            uint64_t* __restrict__ sort_key, uint32_t* __restrict__ sort_val,
            unsigned long long* __restrict__ flags) {
  const int chunks = stride >> 4;
  const int64_t total = n * chunks;
  unsigned bad = 0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t i = t / chunks;
    const int c = (int)(t - i * chunks);
    const int64_t beg = off[i];
    int64_t len64 = off[i + 1] - beg;
    // offsets must start at >= 0, never decrease and stay inside [0, offsets[n]] (the caller's
    // statement of the size of `seqs`): anything else would read outside the buffer
    if (beg < 0 || len64 < 0 || off[i + 1] > off[n]) { bad |= 4u; len64 = 0; }
    else if (len64 > max_len) { bad |= 2u; len64 = 0; }
    const int len = (int)len64;
    uint32_t w[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      uint32_t word = 0;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        const int pos = c * 16 + q * 4 + b;
        uint32_t v = SQ_PAD_BYTE;
        if (pos < len) {
          v = seqs[beg + pos];
          if (v >= (uint32_t)alphabet) { bad |= 1u; v = 0; }
        }
        word |= v << (8 * b);
      }
      w[q] = word;
    }
    if (c == chunks - 1) {
      w[3] = (w[3] & 0x00FFFFFFu) | ((uint32_t)len << 24);
      sort_key[i] = (uint64_t)(255 - len);   // longest first
      sort_val[i] = (uint32_t)i;
    }
    *reinterpret_cast<uint4*>(packed + i * stride + c * 16) = make_uint4(w[0], w[1], w[2], w[3]);
  }
  if (bad) atomicOr(flags, (unsigned long long)bad);
}

extern "C" int sq_pack(sq_ctx* c, const uint8_t* seqs, const int64_t* offsets, int64_t n,
                       int alphabet, int max_len) {
  if (!c || !offsets || n < 0 || alphabet < 1 || alphabet > 32 || max_len < 0)
    return SQ_ERR_INVALID_ARG;
  if (n > 0 && !seqs) return SQ_ERR_INVALID_ARG;
  if (n >= (1ll << 31)) return SQ_ERR_UNSUPPORTED;
  if (max_len > SQ_MAX_LEN) return SQ_ERR_UNSUPPORTED;
  if (!c->ws) return SQ_ERR_WORKSPACE;
  SqDeviceGuard guard(c);
  c->n = -1;
  c->sched = nullptr;
  const int stride = sq_stride_for(max_len);
  const size_t nn = (size_t)(n > 0 ? n : 1);
  // persistent region
  size_t top = 256;
  uint8_t* packed = c->ws + top;                 top += sq_align_up(nn * stride + 16);
  uint32_t* order = (uint32_t*)(c->ws + top);    top += sq_align_up(nn * 4 + 16);
  if (top + sq_pack_scratch_bytes(n) > c->ws_bytes) return SQ_ERR_WORKSPACE;
  c->persist = top;
  sq_scratch_reset(c);
  uint64_t* k0 = sq_scratch<uint64_t>(c, nn);
  uint64_t* k1 = sq_scratch<uint64_t>(c, nn);
  uint32_t* v0 = sq_scratch<uint32_t>(c, nn);
  uint32_t* v1 = sq_scratch<uint32_t>(c, nn);
  void* tmp = sq_scratch<uint8_t>(c, sq_sort_scratch_bytes(n, 1));
  if (!k0 || !k1 || !v0 || !v1 || !tmp) return SQ_ERR_WORKSPACE;

  SQ_CUDA(c, cudaMemsetAsync(c->dflags, 0, 64, c->stream));
  if (n > 0) {
    const int64_t total = n * (stride >> 4);
    int64_t blocks = (total + 255) / 256;
    const int64_t cap = (int64_t)c->sm_count * 16;
    if (blocks > cap) blocks = cap;
    SQ_TIMED(c, SQ_K_PACK, pack_kernel<<<(unsigned)blocks, 256, 0, c->stream>>>(
        seqs, offsets, n, alphabet, max_len, stride, packed, k0, v0, c->dflags));
    SQ_LAUNCH_CHECK(c);
    const int shifts[1] = {0}, widths[1] = {8};
    int in_alt = 0;
    int rc = sq_radix_sort(c, k0, k1, v0, v1, n, 1, shifts, widths, 1, tmp, &in_alt);
    if (rc != SQ_OK) return rc;
    SQ_CUDA(c, cudaMemcpyAsync(order, in_alt ? v1 : v0, (size_t)n * 4, cudaMemcpyDeviceToDevice,
                               c->stream));
  }
  SQ_CUDA(c, cudaMemcpyAsync(c->pinned, c->dflags, 8, cudaMemcpyDeviceToHost, c->stream));
  SQ_CUDA(c, cudaStreamSynchronize(c->stream));
  if (c->pinned[0] & 4ull) return SQ_ERR_INVALID_ARG;       // malformed offsets
  if (c->pinned[0] & 2ull) return SQ_ERR_UNSUPPORTED;       // a sequence longer than max_len
  if (c->pinned[0] & 1ull) return SQ_ERR_BAD_RESIDUE;
  c->n = n;
  c->stride = stride;
  c->max_len = max_len;
  c->alphabet = alphabet;
  c->packed = packed;
  c->order = order;
  sq_scratch_reset(c);
  return SQ_OK;
}
