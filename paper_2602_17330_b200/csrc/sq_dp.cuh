// sq_dp.cuh -- Myers / Hyyro bit-parallel Levenshtein distance, the device routine behind
// sq_edit_distance (a6) and sq_all_pairs (a7).
//
// What it computes is the plain recurrence of PAPER.md L754 Eq. (46) with unit costs and the
// boundary D[x][0]=x, D[0][y]=y.  How: the column of vertical differences D[x][y]-D[x-1][y] is
// held as two bit-vectors Pv (+1) / Mv (-1) over the pattern positions; one text character
// advances the whole column with ~12 logic/add instructions per 32-bit word, and the bottom
// cell is tracked through the horizontal difference at bit m-1.  W 32-bit words are treated as
// one W*32-bit integer (carry of the addition and of the two shifts run across the words), so
// the multi-word case is the single-word algorithm on a wider word.
//
// Peq (for every residue c, the bit mask of pattern positions holding c) is private to the
// thread and lives in shared memory, laid out [c][word][thread] so that the 32 lanes of a warp
// always hit 32 different banks.
#pragma once
#include <stdint.h>

// Build the thread's Peq table for pattern `a` (m residues, read from the packed slot).
template <int W>
__device__ __forceinline__ void sq_peq_build(const uint8_t* __restrict__ a, int m, int alphabet,
                                             uint32_t* peq, int tstride) {
  for (int c = 0; c < alphabet; ++c)
#pragma unroll
    for (int w = 0; w < W; ++w) peq[(c * W + w) * tstride] = 0u;
  const uint32_t* a32 = reinterpret_cast<const uint32_t*>(a);
  for (int x0 = 0; x0 < m; x0 += 4) {
    const uint32_t word = a32[x0 >> 2];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int x = x0 + b;
      if (x < m) {
        const uint32_t ch = (word >> (8 * b)) & 0xFFu;
        uint32_t* p = peq + (ch * W + (W == 1 ? 0 : (x >> 5))) * tstride;
        *p |= 1u << (x & 31);
      }
    }
  }
}

// Distance between the pattern whose Peq is in `peq` (length m >= 1) and text `b` (length n).
// If max_d >= 0 the loop stops as soon as the bottom-row score can no longer come back to
// max_d (each remaining column lowers it by at most 1); the result is then > max_d.
// Peq word w of residue ch is peq[(ch * cstride + w) * tstride]: the private layout uses
// cstride = W, tstride = blockDim.x; a table shared by the whole block uses tstride = 1 and an
// odd cstride so that different residues fall into different banks.
template <int W>
__device__ __forceinline__ int sq_myers(const uint32_t* peq, int cstride, int tstride, int m,
                                        const uint8_t* __restrict__ b, int n, int max_d) {
  uint32_t Pv[W], Mv[W];
#pragma unroll
  for (int w = 0; w < W; ++w) { Pv[w] = 0xFFFFFFFFu; Mv[w] = 0u; }
  const int last = (m - 1) >> 5;            // word holding bit m-1
  const int topbit = (m - 1) & 31;
  int score = m;
  const uint32_t* b32 = reinterpret_cast<const uint32_t*>(b);
  for (int y0 = 0; y0 < n; y0 += 4) {
    const uint32_t word = b32[y0 >> 2];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int y = y0 + q;
      if (y >= n) break;
      const uint32_t ch = (word >> (8 * q)) & 0xFFu;
      uint32_t carry = 0u, ph_in = 1u, mh_in = 0u;
#pragma unroll
      for (int w = 0; w < W; ++w) {
        if (W > 1 && w > last) break;
        const uint32_t Eq = peq[(ch * cstride + w) * tstride];
        const uint32_t pv = Pv[w], mv = Mv[w];
        const uint32_t Xv = Eq | mv;
        const uint32_t t = Eq & pv;
        uint32_t sum;
        if (W == 1) {
          sum = t + pv;
        } else {
          const uint64_t s64 = (uint64_t)t + (uint64_t)pv + (uint64_t)carry;
          sum = (uint32_t)s64;
          carry = (uint32_t)(s64 >> 32);
        }
        const uint32_t Xh = (sum ^ pv) | Eq;
        uint32_t Ph = mv | ~(Xh | pv);
        uint32_t Mh = pv & Xh;
        if (w == last) score += (int)((Ph >> topbit) & 1u) - (int)((Mh >> topbit) & 1u);
        const uint32_t ph_out = Ph >> 31, mh_out = Mh >> 31;
        Ph = (Ph << 1) | ph_in;
        Mh = (Mh << 1) | mh_in;
        ph_in = ph_out;
        mh_in = mh_out;
        Pv[w] = Mh | ~(Xv | Ph);
        Mv[w] = Ph & Xv;
      }
      if (max_d >= 0 && score - (n - 1 - y) > max_d) return max_d + 1;
    }
  }
  return score;
}

// Whole distance for one pair of packed slots, with the trivial cases and the length filter.
template <int W>
__device__ __forceinline__ int sq_pair_distance(const uint8_t* __restrict__ rowA,
                                                const uint8_t* __restrict__ rowB, int stride,
                                                int alphabet, int max_d, uint32_t* peq,
                                                int tstride) {
  const int m = rowA[stride - 1], n = rowB[stride - 1];
  int d;
  const int diff = m > n ? m - n : n - m;
  if (max_d >= 0 && diff > max_d) d = max_d + 1;
  else if (m == 0) d = n;
  else if (n == 0) d = m;
  else {
    sq_peq_build<W>(rowA, m, alphabet, peq, tstride);
    d = sq_myers<W>(peq, W, tstride, m, rowB, n, max_d);
  }
  if (max_d >= 0 && d > max_d) d = max_d + 1;
  return d;
}
