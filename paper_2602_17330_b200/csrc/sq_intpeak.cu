// sq_intpeak.cu -- integer-pipe micro-benchmark: the roofline denominator of the DP stage.
// MEASURED_PEAKS.json carries no INT32/logic peak, so the library
// measures it: 8 independent dependency chains per thread, 64 instructions per loop trip,
// every SM filled with 2048 resident threads.  Result = lane-operations per second.
#include "sq_common.cuh"

namespace {

template <int KIND>
__global__ void __launch_bounds__(256)
int_peak_kernel(int iters, uint32_t seed, uint32_t* __restrict__ sink) {
  uint32_t r[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) r[q] = seed * (threadIdx.x + 1u) + q * 0x9E3779B9u;
  const uint32_t k1 = seed | 1u, k2 = seed ^ 0x5bd1e995u;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        if (KIND == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[q]) : "r"(k1), "r"(k2));
        if (KIND == 1) asm volatile("add.u32 %0, %0, %1;" : "+r"(r[q]) : "r"(k1));
        if (KIND == 2) asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(r[q]) : "r"(k2));
        if (KIND == 3) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[q]) : "r"(k1), "r"(k2));
        if (KIND == 4) asm volatile("min.u32 %0, %0, %1;" : "+r"(r[q]) : "r"(k2 + u * 8 + q));
        if (KIND == 5) {
          if (q & 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[q]) : "r"(k1), "r"(k2));
          else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[q]) : "r"(k1), "r"(k2));
        }
        if (KIND == 6) asm volatile("popc.b32 %0, %0;" : "+r"(r[q]));
        if (KIND == 7) asm volatile("vabsdiff4.u32.u32.u32.add %0, %0, %1, %2;" : "+r"(r[q]) : "r"(k1), "r"(k2));
        // 8, 9: what the register file feeds TWO pipes at once when every operand is a fresh register
        // (the streams above reuse two loop-invariant operands, which the operand reuse cache serves)
        if (KIND == 8) {          // LOP3 / IMAD alternating, three fresh operands each
          if (q & 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[q]) : "r"(r[(q + 3) & 7]), "r"(r[(q + 5) & 7]));
          else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[q]) : "r"(r[(q + 3) & 7]), "r"(r[(q + 5) & 7]));
        }
        if (KIND == 9) {          // the mix of the DP column: 7 LOP3 (three fresh operands) : 4 multiply-adds (two fresh)
          if ((u * 8 + q) % 11 < 7) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[q]) : "r"(r[(q + 3) & 7]), "r"(r[(q + 5) & 7]));
          else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[q]) : "r"(r[(q + 3) & 7]), "r"(k2));
        }
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int q = 0; q < 8; ++q) acc ^= r[q];
  if (acc == 0x12345u) sink[threadIdx.x] = acc;     // practically never true: keeps the chains live
}

}  // namespace

extern "C" int sq_int_peak(sq_ctx* c, int kind, int iters, double* ops_per_s) {
  if (!c || !ops_per_s || iters < 1 || kind < 0 || kind > 9) return SQ_ERR_INVALID_ARG;
  if (!c->ws) return SQ_ERR_WORKSPACE;
  SqDeviceGuard guard(c);
  // 256 words of the free scratch (handed back at once: the kernels practically never write them)
  const size_t top = c->scratch_top;
  uint32_t* sink = sq_scratch<uint32_t>(c, 256);
  c->scratch_top = top;
  if (!sink) return SQ_ERR_WORKSPACE;
  const int blocks = c->sm_count * 8;
  cudaEvent_t e0, e1;
  SQ_CUDA(c, cudaEventCreate(&e0));
  if (cudaEventCreate(&e1) != cudaSuccess) { c->last_err = cudaGetLastError(); cudaEventDestroy(e0); return SQ_ERR_CUDA; }
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, c->stream);
    switch (kind) {
      case 0: int_peak_kernel<0><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 1: int_peak_kernel<1><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 2: int_peak_kernel<2><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 3: int_peak_kernel<3><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 4: int_peak_kernel<4><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 5: int_peak_kernel<5><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 6: int_peak_kernel<6><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 7: int_peak_kernel<7><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      case 8: int_peak_kernel<8><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
      default: int_peak_kernel<9><<<blocks, 256, 0, c->stream>>>(iters, 12345u + rep, sink); break;
    }
    c->launches++;
    cudaEventRecord(e1, c->stream);
    if (cudaEventSynchronize(e1) != cudaSuccess) {
      c->last_err = cudaGetLastError();
      cudaEventDestroy(e0); cudaEventDestroy(e1);
      return SQ_ERR_CUDA;
    }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  const double ops = (double)blocks * 256.0 * (double)iters * 64.0;
  *ops_per_s = ops / (best * 1e-3);
  return SQ_OK;
}
