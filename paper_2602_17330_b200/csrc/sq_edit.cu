// sq_edit.cu -- step a6: batched exact Levenshtein distance on an explicit pair list
// (App. F.3: "for each sequence pair processed by an individual thread",
// recurrence Eq. 46).  One thread per pair, Myers/Hyyro bit-parallel DP (sq_dp.cuh) instead of
// the paper's cell-by-cell DP; 32-bit words, W = ceil(max_len/32) words per column.
#include "sq_common.cuh"
#include "sq_dp.cuh"

namespace {

template <int W>
__global__ void edit_pairs_kernel(const uint8_t* __restrict__ packed, int stride, int64_t n,
                                  const uint2* __restrict__ pairs, int64_t n_pairs, int max_d,
                                  int alphabet, uint16_t* __restrict__ dist) {
  extern __shared__ uint32_t peq_smem[];
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_pairs) return;
  const uint2 pr = pairs[p];
  if (pr.x >= (uint64_t)n || pr.y >= (uint64_t)n) { dist[p] = 0xFFFFu; return; }
  const int d = sq_pair_distance<W>(packed + (int64_t)pr.x * stride, packed + (int64_t)pr.y * stride,
                                    stride, alphabet, max_d, peq_smem + threadIdx.x, blockDim.x);
  dist[p] = (uint16_t)d;
}

template <int W>
int launch_edit(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d, uint16_t* dist_out) {
  const int threads = W <= 2 ? 256 : 128;
  const size_t smem = (size_t)c->alphabet * W * threads * sizeof(uint32_t);
  if (smem > 48 * 1024)
    SQ_CUDA(c, cudaFuncSetAttribute(edit_pairs_kernel<W>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)smem));
  const int64_t blocks = (n_pairs + threads - 1) / threads;
  SQ_TIMED(c, SQ_K_EDIT, edit_pairs_kernel<W><<<(unsigned)blocks, threads, smem, c->stream>>>(
      c->packed, c->stride, c->n, reinterpret_cast<const uint2*>(pairs), n_pairs, max_d, c->alphabet,
      dist_out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

}  // namespace

int sq_edit_distance_impl(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                          uint16_t* dist_out) {
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (n_pairs < 0) return SQ_ERR_INVALID_ARG;
  if (n_pairs == 0) return SQ_OK;
  if (!pairs || !dist_out) return SQ_ERR_INVALID_ARG;
  if (n_pairs >= (1ll << 31) * 128) return SQ_ERR_UNSUPPORTED;
  if (max_d > 65534) max_d = -1;
  const int words = (c->max_len + 31) / 32;
  if (words <= 1) return launch_edit<1>(c, pairs, n_pairs, max_d, dist_out);
  if (words <= 2) return launch_edit<2>(c, pairs, n_pairs, max_d, dist_out);
  if (words <= 4) return launch_edit<4>(c, pairs, n_pairs, max_d, dist_out);
  if (words <= 5) return launch_edit<5>(c, pairs, n_pairs, max_d, dist_out);
  if (words <= 8) return launch_edit<8>(c, pairs, n_pairs, max_d, dist_out);
  return SQ_ERR_UNSUPPORTED;
}
