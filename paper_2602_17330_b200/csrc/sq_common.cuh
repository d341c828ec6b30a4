// sq_common.cuh -- context, workspace arena and small helpers shared by the kernels of
// libsubquad.so (C ABI in include/subquad.h).  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/subquad.h"

#define SQ_EMPTY_SIG 0xFFFFFFFFu
#define SQ_PAD_BYTE  0xFFu

// kernel classes of the built-in per-kernel timer (sq_profile_*)
enum {
  SQ_K_PACK = 0, SQ_K_MINHASH, SQ_K_BANDKEY, SQ_K_SORT_HIST, SQ_K_SCAN, SQ_K_SORT_SCATTER,
  SQ_K_SEGMENT, SQ_K_EMIT, SQ_K_EDIT, SQ_K_ALLPAIRS, SQ_K_MISC, SQ_K_ROWSORT, SQ_K_COUNT
};
constexpr int kSqProfSlots = 1024;

struct sq_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t copy_stream = nullptr;   // sq_pipeline_host: device->host copy of the pairs, beside the DP
  int sm_count = 148;
  // workspace arena: [0, persist) holds the packed copy, [persist, ws_bytes) is per-call scratch
  uint8_t* ws = nullptr;
  size_t ws_bytes = 0;
  size_t persist = 0;
  size_t scratch_top = 0;
  // state of the current pack
  int64_t n = -1;
  int stride = 0;
  int max_len = 0;
  int alphabet = 0;
  uint8_t* packed = nullptr;    // [n][stride]
  uint32_t* order = nullptr;    // [n] sequence ids, longest first (processing order of the sketch)
  // Family-ordered schedule of the last sq_lsh_candidates output, a performance hint for
  // sq_edit_distance: chunk k = the pairs at positions [32k, 32k+32) of the INTERNAL row order
  // (band 0's sorted order, family by family); sched[k] = (first row r0, delta[r0],
  // rowstart[r0+1], -), position q of row r is pair delta[r] + q of the caller's buffer.
  // It lives in the scratch part of the workspace and dies with the next scratch reset.
  const uint4* sched = nullptr;
  const uint32_t* sched_rowstart = nullptr;   // [n2 + 1]
  const uint32_t* sched_delta = nullptr;      // [n2]
  int64_t sched_chunks = 0;
  const void* sched_pairs = nullptr;          // the pair buffer it describes
  int64_t sched_npairs = 0;
  // State left by sq_lsh_prepare for sq_lsh_emit_range: the sorted records, the bucket-id table and
  // the unit lists live in the scratch below `mark`; every emit call allocates above it.  Dies with
  // the next scratch reset.
  struct LshState {
    bool valid = false;
    int64_t n = 0, n2 = 0, raw = 0;
    int bands = 0, bw = 0;
    uint32_t *vin = nullptr, *vint = nullptr, *S = nullptr, *cnt = nullptr, *ubase = nullptr;
    uint32_t *rowidx = nullptr, *ext_off = nullptr, *rowstart = nullptr, *active = nullptr;
    uint2 *loc = nullptr, *units = nullptr, *units0 = nullptr, *units_s = nullptr;
    uint8_t* tmp = nullptr;
    uint32_t nunits = 0, nunits0 = 0, nsmall = 0;
    unsigned long long ntiles = 0;
    size_t mark = 0;
  } lsh;
  // tuning (sq_set_option)
  int sort_key_bytes = 4;       // top bytes of the band key the bucket sort orders by (1..8)
  int64_t sched_min_bytes = (int64_t)96 << 20;   // packed bytes above which the DP follows the schedule
  int sched_by_label = 1;       // schedule rows in family-label order (0: internal row order)
  // bookkeeping
  int64_t launches = 0;
  int64_t last_raw_pairs = 0;
  cudaError_t last_err = cudaSuccess;
  unsigned long long* pinned = nullptr;   // 16 pinned host words for count / flag read-back
  unsigned long long* dflags = nullptr;   // 16 device words (lives at the start of the workspace)
  // per-kernel-class CUDA-event timer (off by default)
  bool prof_on = false;
  cudaEvent_t* prof_ev = nullptr;         // 2 * kSqProfSlots events, created on first enable
  int prof_cls[kSqProfSlots];
  int prof_n = 0;
  double prof_ms[SQ_K_COUNT] = {0};
  int64_t prof_launches[SQ_K_COUNT] = {0};
};

void sq_prof_drain(sq_ctx* c);           // synchronises the pending events into prof_ms

// RAII: every extern "C" entry point runs with the context's device current and puts the caller's
// device back on return, so contexts of several devices can live in one process
struct SqDeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit SqDeviceGuard(const sq_ctx* c) {
    if (!c) return;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
  }
  ~SqDeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// RAII: times everything enqueued on the context's stream during its lifetime as one launch
struct SqProfScope {
  sq_ctx* c; int slot;
  SqProfScope(sq_ctx* ctx, int cls) : c(ctx), slot(-1) {
    if (!c->prof_on) return;
    if (c->prof_n == kSqProfSlots) sq_prof_drain(c);
    slot = c->prof_n++;
    c->prof_cls[slot] = cls;
    cudaEventRecord(c->prof_ev[2 * slot], c->stream);
  }
  ~SqProfScope() { if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], c->stream); }
};

static inline size_t sq_align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// bump allocation out of the scratch part of the workspace; nullptr when it does not fit
template <typename T>
static inline T* sq_scratch(sq_ctx* c, size_t count) {
  size_t bytes = sq_align_up(count * sizeof(T) + 16);
  if (c->scratch_top + bytes > c->ws_bytes) return nullptr;
  T* p = reinterpret_cast<T*>(c->ws + c->scratch_top);
  c->scratch_top += bytes;
  return p;
}
static inline void sq_scratch_reset(sq_ctx* c) { c->scratch_top = c->persist; c->sched = nullptr; c->lsh.valid = false; }

#define SQ_CUDA(ctx, call)                                   \
  do {                                                       \
    cudaError_t e__ = (call);                                \
    if (e__ != cudaSuccess) { (ctx)->last_err = e__; return SQ_ERR_CUDA; } \
  } while (0)

// SQ_TIMED(ctx, class, launch-statement): the launch, bracketed by the optional event timer
#define SQ_TIMED(ctx, cls, ...) do { SqProfScope ps__((ctx), (cls)); __VA_ARGS__; } while (0)

#define SQ_LAUNCH_CHECK(ctx)                                 \
  do {                                                       \
    (ctx)->launches++;                                       \
    cudaError_t e__ = cudaGetLastError();                    \
    if (e__ != cudaSuccess) { (ctx)->last_err = e__; return SQ_ERR_CUDA; } \
  } while (0)

static inline int sq_stride_for(int max_len) { return ((max_len + 1) + 15) / 16 * 16; }

// ---- sizes of the per-op scratch (shared by sq_workspace_bytes and the ops themselves) ----
size_t sq_persist_bytes(int64_t n, int max_len);
size_t sq_lsh_scratch_bytes(int64_t n, int bands, int64_t pair_capacity);
size_t sq_allpairs_scratch_bytes(int64_t n, int64_t pair_capacity);
size_t sq_graph_scratch_bytes(int64_t n, int64_t n_pairs);
size_t sq_join_scratch_bytes(int64_t rows, int64_t n_b, int64_t pair_capacity);
size_t sq_sort_scratch_bytes(int64_t n_per_batch, int nbatch);

// ---- radix sort (sq_sort.cu) ----
// Stable LSD radix sort of `nbatch` independent arrays of `n` records each (batch b occupies
// [b*n, (b+1)*n)).  Keys are uint64; vals (uint32) may be nullptr for a keys-only sort.
// `shifts[p]`/`widths[p]` give the digit of pass p (width <= 8).  Ping-pongs between the in
// and alt buffers; returns (through *result_in_alt) where the result ended up.
// `tmp` must hold sq_sort_scratch_bytes(n, nbatch) bytes.
int sq_radix_sort(sq_ctx* c, uint64_t* keys_in, uint64_t* keys_alt, uint32_t* vals_in,
                  uint32_t* vals_alt, int64_t n, int nbatch, const int* shifts, const int* widths,
                  int npasses, void* tmp, int* result_in_alt);

// The same sort on the key bytes first_pass .. first_pass+npasses-1 (width 8 each) in ONE kernel
// per pass (all histograms up front, decoupled look-back between tiles).  n < 2^30 per batch.
int sq_onesweep_sort(sq_ctx* c, uint64_t* keys_in, uint64_t* keys_alt, uint32_t* vals_in,
                     uint32_t* vals_alt, int64_t n, int nbatch, int first_pass, int npasses, void* tmp,
                     int* result_in_alt);

// exclusive prefix sum of uint32 (offsets wrap mod 2^32; the grand total is returned in 64 bits
// so callers can detect the wrap).  In-place capable (out may equal in).
// `tmp` needs (n/2048 + 2) * 4 bytes.
int sq_exclusive_scan_u32(sq_ctx* c, const uint32_t* in, uint32_t* out, int64_t n, uint32_t* tmp,
                          unsigned long long* total_out_dev /* may be nullptr */);

// ---- ops implemented in their own translation units ----
int sq_minhash_impl(sq_ctx* c, int k, int H, uint64_t seed, uint32_t* sig_out);
int sq_edit_distance_impl(sq_ctx* c, const uint32_t* pairs, int64_t n_pairs, int max_d,
                          uint16_t* dist_out);
// pairs (i, j) with i in the context's own pack and j in `packedB` (same stride and alphabet)
// banded: the pairs passed a filter (most are within max_d) and come grouped by i -- sequences
// longer than 64 then take the banded shared-Peq kernel (no early exit)
int sq_edit_distance_ab(sq_ctx* c, const uint8_t* packedB, int64_t nB, int max_len_b,
                        const uint32_t* pairs, int64_t n_pairs, int max_d, uint16_t* dist_out,
                        bool banded);
// survivors of a coarse filter -> distances (grouping by i, banded shared-Peq kernel; sq_edit.cu)
int sq_survivor_distances(sq_ctx* c, const uint8_t* packedB, int64_t nB, int max_len_b, uint2* surv,
                          int64_t ns, int max_d, uint2* surv2, void* sort_tmp, uint16_t* sdist,
                          const uint2** live_out, int64_t* nlive_out);
// pieces of the thresholded all-pairs path (sq_allpairs.cu) shared with the join (sq_join.cu)
int sq_residue_hist(sq_ctx* c, const uint8_t* packed, int stride, int64_t n, uint32_t* rh, uint32_t* lens);
int sq_hit_compact(sq_ctx* c, const uint2* surv, const uint16_t* sdist, int64_t ns, int max_d,
                   uint64_t* hit_pairs, uint32_t* hit_dist, int64_t capacity, unsigned long long* counter);
int sq_narrow_dist(sq_ctx* c, const uint32_t* in, int64_t n, uint16_t* out);
// CSR form of an (i, j)-ascending pair list (sq_csr.cu)
int sq_csr_split(sq_ctx* c, cudaStream_t st, const uint32_t* pairs, int64_t p0, int64_t p1,
                 int64_t n_pairs, uint32_t* col, int64_t* row_ptr);
int sq_csr_fill(sq_ctx* c, cudaStream_t st, int64_t* row_ptr, int64_t v);
int sq_csr_narrow(sq_ctx* c, const uint16_t* dist, int64_t n_pairs, uint8_t* out);
// the bag-distance filter over a block of rows x all columns (sq_join.cu)
int sq_bag_filter(sq_ctx* c, const uint32_t* rhA, const uint32_t* lensA, int64_t row0, int64_t rows,
                  int64_t a_base, const uint32_t* rhB, const uint32_t* lensB, int64_t nB, int max_d,
                  int upper, uint2* surv, size_t scap, unsigned long long* counter);
