// sq_api.cu -- context life cycle, workspace accounting, error strings and the host-buffer
// pipeline entry point of libsubquad.so (C ABI: include/subquad.h).
#include "sq_common.cuh"
#include <new>

extern "C" {

int sq_create(sq_ctx** out, int device, void* cuda_stream) {
  if (!out) return SQ_ERR_INVALID_ARG;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return SQ_ERR_CUDA;
  if (cudaSetDevice(device) != cudaSuccess) return SQ_ERR_CUDA;
  sq_ctx* c = new (std::nothrow) sq_ctx();
  if (!c) return SQ_ERR_INVALID_ARG;
  c->device = device;
  c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
  if (cudaHostAlloc(reinterpret_cast<void**>(&c->pinned), 16 * sizeof(unsigned long long),
                    cudaHostAllocDefault) != cudaSuccess) {
    delete c;
    return SQ_ERR_CUDA;
  }
  // second stream of the *_host entry points (device->host copies beside the compute stream)
  if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaFreeHost(c->pinned);
    delete c;
    return SQ_ERR_CUDA;
  }
  *out = c;
  return SQ_OK;
}

void sq_destroy(sq_ctx* c) {
  if (!c) return;
  SqDeviceGuard guard(c);
  if (c->prof_ev) {
    for (int i = 0; i < 2 * kSqProfSlots; ++i) cudaEventDestroy(c->prof_ev[i]);
    delete[] c->prof_ev;
  }
  if (c->pinned) cudaFreeHost(c->pinned);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  delete c;
}

int sq_set_workspace(sq_ctx* c, void* dev_ptr, size_t bytes) {
  if (!c || !dev_ptr || (reinterpret_cast<uintptr_t>(dev_ptr) & 255)) return SQ_ERR_INVALID_ARG;
  if (bytes < 4096) return SQ_ERR_WORKSPACE;
  c->ws = static_cast<uint8_t*>(dev_ptr);
  c->ws_bytes = bytes;
  c->dflags = reinterpret_cast<unsigned long long*>(c->ws);   // first 256 bytes: flag words
  c->persist = 256;
  c->scratch_top = c->persist;
  c->n = -1;
  c->packed = nullptr;
  c->order = nullptr;
  c->sched = nullptr;
  return SQ_OK;
}

int sq_profile_enable(sq_ctx* c, int on) {
  if (!c) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  if (on && !c->prof_ev) {
    c->prof_ev = new (std::nothrow) cudaEvent_t[2 * kSqProfSlots];
    if (!c->prof_ev) return SQ_ERR_INVALID_ARG;
    for (int i = 0; i < 2 * kSqProfSlots; ++i) SQ_CUDA(c, cudaEventCreate(&c->prof_ev[i]));
  }
  if (!on && c->prof_on) sq_prof_drain(c);
  c->prof_on = on != 0;
  return SQ_OK;
}

int sq_profile_reset(sq_ctx* c) {
  if (!c) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  sq_prof_drain(c);
  for (int k = 0; k < SQ_K_COUNT; ++k) { c->prof_ms[k] = 0.0; c->prof_launches[k] = 0; }
  return SQ_OK;
}

int sq_profile_read(sq_ctx* c, int cls, double* ms, int64_t* launches) {
  if (!c || cls < 0 || cls >= SQ_K_COUNT || !ms || !launches) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  sq_prof_drain(c);
  *ms = c->prof_ms[cls];
  *launches = c->prof_launches[cls];
  return SQ_OK;
}

const char* sq_profile_name(int cls) {
  static const char* names[SQ_K_COUNT] = {"pack", "minhash", "band_key", "sort_hist", "scan",
                                          "sort_scatter", "bucket_scan", "emit", "edit_distance",
                                          "all_pairs", "misc", "row_sort"};
  return (cls >= 0 && cls < SQ_K_COUNT) ? names[cls] : nullptr;
}

int64_t sq_packed_n(const sq_ctx* c) { return c ? c->n : -1; }
int sq_packed_stride(const sq_ctx* c) { return c ? c->stride : 0; }
int64_t sq_last_raw_pairs(const sq_ctx* c) { return c ? c->last_raw_pairs : 0; }
int64_t sq_kernel_launches(const sq_ctx* c) { return c ? c->launches : 0; }
const char* sq_last_cuda_error(const sq_ctx* c) {
  return c ? cudaGetErrorString(c->last_err) : "no context";
}

const char* sq_strerror(int code) {
  switch (code) {
    case SQ_OK: return "ok";
    case SQ_ERR_INVALID_ARG: return "invalid argument";
    case SQ_ERR_BAD_RESIDUE: return "residue code >= alphabet";
    case SQ_ERR_NOT_PACKED: return "sq_pack has not been called on this workspace";
    case SQ_ERR_CAPACITY: return "output capacity too small (required count returned)";
    case SQ_ERR_WORKSPACE: return "workspace missing or too small";
    case SQ_ERR_UNSUPPORTED: return "unsupported size (sequence longer than max_len, or length, H or bands over the compiled maximum)";
    case SQ_ERR_CUDA: return "CUDA runtime error";
    default: return "unknown error";
  }
}

size_t sq_workspace_bytes(const sq_ctx*, int op, const sq_sizes* s) {
  if (!s || s->n < 0) return 0;
  size_t persist = 256 + sq_persist_bytes(s->n, s->max_len);
  size_t slack = 1 << 16;
  switch (op) {
    case SQ_OP_PACK:
    case SQ_OP_MINHASH:
    case SQ_OP_EDIT_DISTANCE:
      return persist + slack;
    case SQ_OP_LSH:
      return persist + sq_lsh_scratch_bytes(s->n, s->bands, s->pair_capacity) + slack;
    case SQ_OP_ALL_PAIRS:
      return persist + sq_allpairs_scratch_bytes(s->n, s->pair_capacity) + slack;
    case SQ_OP_GRAPH:
      return persist + sq_graph_scratch_bytes(s->n, s->pair_capacity) + slack;
    case SQ_OP_JOIN:
      return persist + sq_join_scratch_bytes(s->n, s->n_other, s->pair_capacity) + slack;
    case SQ_OP_PIPELINE_HOST: {
      size_t io = sq_align_up((size_t)s->total_len + 16) + sq_align_up((size_t)(s->n + 1) * 8 + 16) +
                  sq_align_up((size_t)s->n * s->H * 4 + 16) +
                  sq_align_up((size_t)s->pair_capacity * 8 + 16) +
                  sq_align_up((size_t)s->pair_capacity * 2 + 16) +
                  sq_align_up((size_t)s->pair_capacity * 4 + 16) +      // sq_pipeline_host_csr: col,
                  sq_align_up((size_t)s->pair_capacity + 16) +          // byte distances,
                  sq_align_up((size_t)(s->n + 1) * 8 + 16);             // row offsets
      return persist + io + sq_lsh_scratch_bytes(s->n, s->bands, s->pair_capacity) + slack;
    }
    default: return 0;
  }
}

int sq_set_option(sq_ctx* c, int option, int64_t value) {
  if (!c) return SQ_ERR_INVALID_ARG;
  if (option == SQ_OPT_SORT_KEY_BYTES && value >= 1 && value <= 8) { c->sort_key_bytes = (int)value; return SQ_OK; }
  if (option == SQ_OPT_SCHED_MIN_BYTES && value >= 0) { c->sched_min_bytes = value; return SQ_OK; }
  if (option == SQ_OPT_SCHED_BY_LABEL && (value == 0 || value == 1)) { c->sched_by_label = (int)value; return SQ_OK; }
  return SQ_ERR_INVALID_ARG;
}

int sq_minhash(sq_ctx* c, int k, int H, uint64_t seed, uint32_t* sig_out) {
  if (!c) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  return sq_minhash_impl(c, k, H, seed, sig_out);
}

int sq_edit_distance(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                     uint16_t* dist_out) {
  if (!c) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  return sq_edit_distance_impl(c, pairs, n_pairs, max_d, dist_out);
}

// shared body of sq_pipeline_host / sq_pipeline_host_csr
static int pipeline_host_impl(sq_ctx* c, const uint8_t* seqs_host, const int64_t* offsets_host, int64_t n,
                              int alphabet, int max_len, int k, int H, uint64_t seed, int bands, int rows,
                              int bucket_cap, int max_d, uint32_t* pairs_out_host, uint16_t* dist_out_host,
                              int64_t* row_ptr_host, uint32_t* col_host, uint8_t* dist8_host,
                              int64_t capacity, int64_t* n_pairs) {
  const bool csr = row_ptr_host != nullptr;
  if (!c || !offsets_host || !n_pairs || n < 0 || capacity < 0) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  *n_pairs = 0;
  // everything the carving of the I/O region depends on is checked before it is used
  if (H < 1 || k < 1 || bands < 1 || rows < 1 || bucket_cap < 1 || alphabet < 1 || alphabet > 32)
    return SQ_ERR_INVALID_ARG;
  if (H > SQ_MAX_H || bands > SQ_MAX_BANDS) return SQ_ERR_UNSUPPORTED;
  if (!c->ws) return SQ_ERR_WORKSPACE;
  if (max_len < 0 || max_len > SQ_MAX_LEN) return SQ_ERR_UNSUPPORTED;
  if (csr && (max_d < 0 || max_d > 254)) return SQ_ERR_UNSUPPORTED;      // min(d, max_d+1) in a byte
  const int64_t total = offsets_host[n];
  if (total < 0 || offsets_host[0] != 0 || (total > 0 && !seqs_host)) return SQ_ERR_INVALID_ARG;
  if (capacity > 0 && !csr && (!pairs_out_host || !dist_out_host)) return SQ_ERR_INVALID_ARG;
  // Device I/O buffers sit at the END of the workspace so that sq_pack's persistent region
  // and the per-op scratch (both allocated from the front) cannot overlap them.
  size_t io = sq_align_up((size_t)total + 16) + sq_align_up((size_t)(n + 1) * 8 + 16) +
              sq_align_up((size_t)n * H * 4 + 16) + sq_align_up((size_t)capacity * 8 + 16) +
              sq_align_up((size_t)capacity * 2 + 16);
  if (csr) io += sq_align_up((size_t)capacity * 4 + 16) + sq_align_up((size_t)capacity + 16) +
                 sq_align_up((size_t)(n + 1) * 8 + 16);
  if (io + 4096 > c->ws_bytes) return SQ_ERR_WORKSPACE;
  size_t full = c->ws_bytes;
  uint8_t* p = c->ws + (full - io) / 256 * 256;
  uint8_t* d_seqs = p;            p += sq_align_up((size_t)total + 16);
  int64_t* d_off = (int64_t*)p;   p += sq_align_up((size_t)(n + 1) * 8 + 16);
  uint32_t* d_sig = (uint32_t*)p; p += sq_align_up((size_t)n * H * 4 + 16);
  uint32_t* d_pairs = (uint32_t*)p; p += sq_align_up((size_t)capacity * 8 + 16);
  uint16_t* d_dist = (uint16_t*)p;  p += sq_align_up((size_t)capacity * 2 + 16);
  uint32_t* d_col = nullptr; uint8_t* d_dist8 = nullptr; int64_t* d_rowptr = nullptr;
  if (csr) {
    d_col = (uint32_t*)p;   p += sq_align_up((size_t)capacity * 4 + 16);
    d_dist8 = p;            p += sq_align_up((size_t)capacity + 16);
    d_rowptr = (int64_t*)p;
  }
  // shrink the arena seen by the ops to the part in front of the I/O buffers
  size_t saved = c->ws_bytes;
  c->ws_bytes = (size_t)((c->ws + (full - io) / 256 * 256) - c->ws);
  int rc = SQ_OK;
  do {
    if (total > 0 && cudaMemcpyAsync(d_seqs, seqs_host, (size_t)total, cudaMemcpyHostToDevice,
                                     c->stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    if (cudaMemcpyAsync(d_off, offsets_host, (size_t)(n + 1) * 8, cudaMemcpyHostToDevice,
                        c->stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    if ((rc = sq_pack(c, d_seqs, d_off, n, alphabet, max_len)) != SQ_OK) break;
    if ((rc = sq_minhash(c, k, H, seed, d_sig)) != SQ_OK) break;
    if ((rc = sq_lsh_candidates(c, d_sig, H, bands, rows, bucket_cap, SQ_LSH_SORTED, d_pairs,
                                capacity, n_pairs)) != SQ_OK) break;
    // sq_lsh_candidates has synchronised: the pairs are final.  Their copy to the host (the bulk
    // of the output) runs on the context's second stream while the DP kernel works on the first.
    const int64_t np = *n_pairs;
    if (!csr) {
      if (np > 0 &&
          cudaMemcpyAsync(pairs_out_host, d_pairs, (size_t)np * 8, cudaMemcpyDeviceToHost,
                          c->copy_stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    } else if (np == 0) {
      if ((rc = sq_csr_fill(c, c->copy_stream, d_rowptr, 0)) != SQ_OK) break;
    } else {
      // col + row offsets: the first chunk is split and sent at once on the copy stream; the rest
      // is split on the main stream AHEAD of the DP kernel (behind it the split would wait for
      // SMs and starve the copy engine -- PCIe is the critical path, the DP has slack)
      const int64_t first = np < (1ll << 24) ? np : (1ll << 24);
      rc = sq_csr_split(c, c->copy_stream, d_pairs, 0, first, np, d_col, d_rowptr);
      if (rc == SQ_OK && cudaMemcpyAsync(col_host, d_col, (size_t)first * 4, cudaMemcpyDeviceToHost,
                                         c->copy_stream) != cudaSuccess) rc = SQ_ERR_CUDA;
      if (rc == SQ_OK && first < np) {
        rc = sq_csr_split(c, c->stream, d_pairs, first, np, np, d_col, d_rowptr);
        cudaEvent_t ev;
        if (rc == SQ_OK && cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) rc = SQ_ERR_CUDA;
        if (rc == SQ_OK) {
          if (cudaEventRecord(ev, c->stream) != cudaSuccess ||
              cudaStreamWaitEvent(c->copy_stream, ev, 0) != cudaSuccess ||
              cudaMemcpyAsync(col_host + first, d_col + first, (size_t)(np - first) * 4,
                              cudaMemcpyDeviceToHost, c->copy_stream) != cudaSuccess) rc = SQ_ERR_CUDA;
          cudaEventDestroy(ev);
        }
      }
      if (rc != SQ_OK) break;
    }
    if (csr && cudaMemcpyAsync(row_ptr_host, d_rowptr, (size_t)(n + 1) * 8, cudaMemcpyDeviceToHost,
                               c->copy_stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    if ((rc = sq_edit_distance(c, d_pairs, np, max_d, d_dist)) != SQ_OK) break;
    if (!csr) {
      if (np > 0 &&
          cudaMemcpyAsync(dist_out_host, d_dist, (size_t)np * 2, cudaMemcpyDeviceToHost,
                          c->stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    } else if (np > 0) {
      if ((rc = sq_csr_narrow(c, d_dist, np, d_dist8)) != SQ_OK) break;
      if (cudaMemcpyAsync(dist8_host, d_dist8, (size_t)np, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) {
        rc = SQ_ERR_CUDA; break;
      }
    }
    if (cudaStreamSynchronize(c->copy_stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
  } while (0);
  if (rc == SQ_ERR_CUDA) c->last_err = cudaGetLastError();
  if (rc != SQ_OK) {
    // nothing may still be writing the caller's host buffers once an error is returned
    cudaStreamSynchronize(c->copy_stream);
    cudaStreamSynchronize(c->stream);
  }
  c->ws_bytes = saved;
  return rc;
}

int sq_pipeline_host(sq_ctx* c, const uint8_t* seqs_host, const int64_t* offsets_host, int64_t n,
                     int alphabet, int max_len, int k, int H, uint64_t seed, int bands, int rows,
                     int bucket_cap, int max_d, uint32_t* pairs_out_host, uint16_t* dist_out_host,
                     int64_t capacity, int64_t* n_pairs) {
  return pipeline_host_impl(c, seqs_host, offsets_host, n, alphabet, max_len, k, H, seed, bands, rows,
                            bucket_cap, max_d, pairs_out_host, dist_out_host, nullptr, nullptr, nullptr,
                            capacity, n_pairs);
}

int sq_pipeline_host_csr(sq_ctx* c, const uint8_t* seqs_host, const int64_t* offsets_host, int64_t n,
                         int alphabet, int max_len, int k, int H, uint64_t seed, int bands, int rows,
                         int bucket_cap, int max_d, int64_t* row_ptr_host, uint32_t* col_host,
                         uint8_t* dist_host, int64_t capacity, int64_t* n_pairs) {
  if (!row_ptr_host || (capacity > 0 && (!col_host || !dist_host))) return SQ_ERR_INVALID_ARG;
  return pipeline_host_impl(c, seqs_host, offsets_host, n, alphabet, max_len, k, H, seed, bands, rows,
                            bucket_cap, max_d, nullptr, nullptr, row_ptr_host, col_host, dist_host,
                            capacity, n_pairs);
}

// Out-of-core / sharded form of a3-a6: the candidate list is produced and verified batch by batch of
// rows (external ids), every batch copied to the host on the copy stream while the next one is
// emitted.  See subquad.h.
int sq_candidates_stream_host(sq_ctx* c, const uint32_t* sig, int H, int bands, int rows, int bucket_cap,
                              int max_d, int64_t batch_rows, int64_t block_capacity, int part, int n_parts,
                              uint32_t* pairs_host, uint16_t* dist_host, int64_t capacity, int64_t* n_pairs,
                              int64_t* n_raw) {
  if (!c || !n_pairs) return SQ_ERR_INVALID_ARG;
  SqDeviceGuard guard(c);
  *n_pairs = 0;
  if (n_raw) *n_raw = 0;
  if (c->n < 0) return SQ_ERR_NOT_PACKED;
  if (capacity < 0 || block_capacity < 1 || n_parts < 1 || part < 0 || part >= n_parts) return SQ_ERR_INVALID_ARG;
  if (capacity > 0 && (!pairs_host || !dist_host)) return SQ_ERR_INVALID_ARG;
  if (block_capacity >= (1ll << 32) - 1) return SQ_ERR_UNSUPPORTED;
  if (!c->ws) return SQ_ERR_WORKSPACE;
  const int64_t n = c->n;
  // two device blocks (pairs + distances) at the END of the workspace, out of the scratch's way
  const size_t blk = sq_align_up((size_t)block_capacity * 8 + 16) + sq_align_up((size_t)block_capacity * 2 + 16);
  if (2 * blk + c->persist + 4096 > c->ws_bytes) return SQ_ERR_WORKSPACE;
  const size_t saved = c->ws_bytes;
  uint8_t* io = c->ws + (saved - 2 * blk) / 256 * 256;
  c->ws_bytes = (size_t)(io - c->ws);
  uint32_t* dp[2]; uint16_t* dd[2];
  for (int s = 0; s < 2; ++s) {
    dp[s] = reinterpret_cast<uint32_t*>(io + s * blk);
    dd[s] = reinterpret_cast<uint16_t*>(io + s * blk + sq_align_up((size_t)block_capacity * 8 + 16));
  }
  cudaEvent_t done[2] = {nullptr, nullptr}, ready = nullptr;
  int rc = SQ_OK;
  int64_t total = 0;
  do {
    if ((rc = sq_lsh_prepare(c, sig, H, bands, rows, bucket_cap, n_raw)) != SQ_OK) break;
    if (cudaEventCreateWithFlags(&done[0], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&done[1], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ready, cudaEventDisableTiming) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
    if (batch_rows <= 0) {
      // PAPER.md Eq. 12 with M_avail = the bytes of one device block, c = 10 bytes per candidate
      // (pair + distance) and l_max = 1: B rows whose B x B tile of cells would fill the block
      batch_rows = sq_batch_size(n, (uint64_t)block_capacity * 10ull, 10u, 1u);
    }
    if (batch_rows < 1) batch_rows = 1;
    bool used[2] = {false, false};
    int slot = 0;
    const int64_t nbatch = n > 0 ? (n + batch_rows - 1) / batch_rows : 0;
    for (int64_t b = part; b < nbatch && rc == SQ_OK; b += n_parts) {
      // a batch that does not fit one block is halved (a small stack of row ranges, in order)
      int64_t stack_lo[64], stack_hi[64];
      int sp = 0;
      stack_lo[0] = b * batch_rows;
      stack_hi[0] = stack_lo[0] + batch_rows < n ? stack_lo[0] + batch_rows : n;
      sp = 1;
      while (sp > 0 && rc == SQ_OK) {
        const int64_t lo = stack_lo[sp - 1], hi = stack_hi[sp - 1];
        --sp;
        if (used[slot]) {
          if (cudaEventSynchronize(done[slot]) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }   // its last copy has left
          used[slot] = false;
        }
        int64_t cnt = 0;
        int r2 = sq_lsh_emit_range(c, lo, hi, SQ_LSH_SORTED, dp[slot], block_capacity, &cnt);
        if (r2 == SQ_ERR_CAPACITY || r2 == SQ_ERR_WORKSPACE || r2 == SQ_ERR_UNSUPPORTED) {
          if (hi - lo <= 1 || sp + 2 > 64) { rc = r2; if (r2 == SQ_ERR_CAPACITY) total += cnt; break; }
          const int64_t mid = lo + (hi - lo) / 2;
          stack_lo[sp] = mid; stack_hi[sp] = hi; ++sp;          // second half is done after the first
          stack_lo[sp] = lo; stack_hi[sp] = mid; ++sp;
          continue;
        }
        if (r2 != SQ_OK) { rc = r2; break; }
        if (cnt == 0) continue;
        if (total + cnt <= capacity) {
          if ((rc = sq_edit_distance_impl(c, dp[slot], cnt, max_d, dd[slot])) != SQ_OK) break;
          if (cudaEventRecord(ready, c->stream) != cudaSuccess ||
              cudaStreamWaitEvent(c->copy_stream, ready, 0) != cudaSuccess ||
              cudaMemcpyAsync(pairs_host + 2 * total, dp[slot], (size_t)cnt * 8, cudaMemcpyDeviceToHost,
                              c->copy_stream) != cudaSuccess ||
              cudaMemcpyAsync(dist_host + total, dd[slot], (size_t)cnt * 2, cudaMemcpyDeviceToHost,
                              c->copy_stream) != cudaSuccess ||
              cudaEventRecord(done[slot], c->copy_stream) != cudaSuccess) { rc = SQ_ERR_CUDA; break; }
          used[slot] = true;
          slot ^= 1;
        }
        total += cnt;                                            // keeps counting past `capacity`
      }
    }
  } while (0);
  cudaStreamSynchronize(c->copy_stream);
  cudaStreamSynchronize(c->stream);
  if (rc == SQ_ERR_CUDA) c->last_err = cudaGetLastError();
  for (int s = 0; s < 2; ++s) if (done[s]) cudaEventDestroy(done[s]);
  if (ready) cudaEventDestroy(ready);
  c->ws_bytes = saved;
  sq_scratch_reset(c);
  if (rc != SQ_OK) return rc;
  *n_pairs = total;
  return total > capacity ? SQ_ERR_CAPACITY : SQ_OK;
}

}  // extern "C"

void sq_prof_drain(sq_ctx* c) {
  if (!c->prof_ev || c->prof_n == 0) return;
  cudaEventSynchronize(c->prof_ev[2 * (c->prof_n - 1) + 1]);
  for (int i = 0; i < c->prof_n; ++i) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]) == cudaSuccess) {
      c->prof_ms[c->prof_cls[i]] += ms;
      c->prof_launches[c->prof_cls[i]] += 1;
    }
  }
  c->prof_n = 0;
}
