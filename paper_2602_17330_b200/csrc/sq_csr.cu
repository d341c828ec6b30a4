// sq_csr.cu -- the verified candidates as a compressed sparse row structure for the trip to the host.
//
// sq_pipeline_host ships (i, j) pairs and 16-bit distances: 10 bytes per candidate, and at
// config 4 the 16 GB crossing PCIe is three quarters of the end-to-end time.  The pair list is
// ascending in (i, j), so i is redundant given row offsets, and a thresholded distance
// min(d, max_d + 1) fits one byte: row_ptr (8 bytes per SEQUENCE) + col 4 + dist 1 = 5 bytes per
// candidate -- the same content (Eq. 1: the graph's edges and weights; L158 CAND).
//   csr_split_kernel   one pass over a chunk of the pair list: col[p] = j, and at every change
//                      of i the row offsets of the rows in between (rows without partners get
//                      the offset of the next row that has some).
//   csr_narrow_kernel  uint16 distances -> uint8.
#include "sq_common.cuh"

namespace {

__global__ void __launch_bounds__(256)
csr_split_kernel(const uint2* __restrict__ pairs, int64_t p0, int64_t p1, int64_t n_pairs, int64_t n,
                 uint32_t* __restrict__ col, int64_t* __restrict__ row_ptr) {
  const int64_t p = p0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= p1) return;
  const uint2 pr = pairs[p];
  col[p] = pr.y;
  // rows (prev.x, pr.x] start at p; the very first pair also covers rows [0, pr.x]
  int64_t lo = p == 0 ? 0 : (int64_t)pairs[p - 1].x + 1;
  const int64_t hi = (int64_t)pr.x < n ? (int64_t)pr.x : n - 1;
  for (int64_t r = lo; r <= hi; ++r) row_ptr[r] = p;
  if (p == n_pairs - 1)
    for (int64_t r = (int64_t)pr.x + 1; r <= n; ++r) row_ptr[r] = n_pairs;
}

__global__ void __launch_bounds__(256)
csr_fill_kernel(int64_t* __restrict__ row_ptr, int64_t n, int64_t v) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r <= n) row_ptr[r] = v;
}

__global__ void __launch_bounds__(256)
csr_narrow_kernel(const uint16_t* __restrict__ in, int64_t n, uint8_t* __restrict__ out) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;       // four distances per thread
  const int64_t p = q * 4;
  if (p + 3 < n) {
    const uint2 v = reinterpret_cast<const uint2*>(in)[q];
    const uint32_t b = (v.x & 0xFFu) | ((v.x >> 8) & 0xFF00u) | ((v.y & 0xFFu) << 16) | ((v.y >> 16) << 24);
    reinterpret_cast<uint32_t*>(out)[q] = b;
  } else {
    for (int64_t t = p; t < n; ++t) out[t] = (uint8_t)in[t];
  }
}

}  // namespace

// col / row offsets of pairs [p0, p1) of an (i, j)-ascending list, on `st`
int sq_csr_split(sq_ctx* c, cudaStream_t st, const uint32_t* pairs, int64_t p0, int64_t p1,
                 int64_t n_pairs, uint32_t* col, int64_t* row_ptr) {
  if (p1 <= p0) return SQ_OK;
  csr_split_kernel<<<(unsigned)((p1 - p0 + 255) / 256), 256, 0, st>>>(
      reinterpret_cast<const uint2*>(pairs), p0, p1, n_pairs, c->n, col, row_ptr);
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int sq_csr_fill(sq_ctx* c, cudaStream_t st, int64_t* row_ptr, int64_t v) {
  csr_fill_kernel<<<(unsigned)((c->n + 256) / 256), 256, 0, st>>>(row_ptr, c->n, v);
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}

int sq_csr_narrow(sq_ctx* c, const uint16_t* dist, int64_t n_pairs, uint8_t* out) {
  if (n_pairs <= 0) return SQ_OK;
  SQ_TIMED(c, SQ_K_MISC, csr_narrow_kernel<<<(unsigned)(((n_pairs + 3) / 4 + 255) / 256), 256, 0, c->stream>>>(
      dist, n_pairs, out));
  SQ_LAUNCH_CHECK(c);
  return SQ_OK;
}
