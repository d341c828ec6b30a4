/*
 * sq_oracle.c -- plain, slow, obviously-correct CPU oracle for the SubQuad
 * candidate-pair affinity path (arxiv/paper_2602_17330).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check in
 * __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may load
 * it.  It shares no code, header, table or constant generator with the CUDA path
 * under paper_2602_17330_b200/csrc/; both follow the same WRITTEN spec
 * (restated in DESIGN.md "Readings").
 *
 * What the paper fixes and where:
 *   - edit distance recurrence: Eq. (46) (App. F.3); unit indel
 *     cost L760; boundary D[x][0]=x, D[0][y]=y (reading 12); unit substitution
 *     cost (reading 11, north_star "exact Levenshtein").
 *   - MinHash sketches of size M in {64,128,256}: PAPER.md L157 (Alg. 1 step 1),
 *     L269 (section 4.1); estimator error <= 1/sqrt(M): L495-497 Eq. (30).
 *     The hash family is NOT in the paper: spec C2.
 *   - MinHash LSH index -> candidate list CAND: PAPER.md L158 (Alg. 1 step 2),
 *     L273 (section 4.2).  Banding, keys and cap are NOT in the paper: spec C3.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): textbook distances, BFS over
 * edit operations, metric invariants, closed forms of the sketch, Jaccard
 * convergence within Eq. (30), brute force vs sorted bucketing, S-curve, closed
 * form candidate counts.  Unpinned by any external source: the numeric values of
 * the hash constants (they are the spec's own choice; the tests pin them to
 * frac(sqrt 2), frac(sqrt 3) and 2^64/phi computed with integer square roots).
 *
 * Plain C11, integer only.  OpenMP `parallel for` over independent sequences /
 * pairs is the only parallelism; no blocking, fusion, SIMD or reordering.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int t) {
#ifdef _OPENMP
  if (t > 0) omp_set_num_threads(t);
#else
  (void)t;
#endif
}

/* ------------------------------------------------------------------------ */
/* C1. Levenshtein distance: Wagner-Fischer, the definition written out.     */
/* d[x][y] = min(d[x-1][y]+1, d[x][y-1]+1, d[x-1][y-1] + [a_x != b_y])        */
/* (Eq. 46), d[x][0] = x, d[0][y] = y.                          */
/* ------------------------------------------------------------------------ */
int orc_wagner_fischer(const uint8_t* a, int la, const uint8_t* b, int lb) {
  int* prev = (int*)malloc(sizeof(int) * (size_t)(lb + 1));
  int* cur = (int*)malloc(sizeof(int) * (size_t)(lb + 1));
  for (int y = 0; y <= lb; ++y) prev[y] = y;               /* d[0][y] = y */
  for (int x = 1; x <= la; ++x) {
    cur[0] = x;                                            /* d[x][0] = x */
    for (int y = 1; y <= lb; ++y) {
      int del = prev[y] + 1;                               /* d[x-1][y] + deletion_cost  */
      int ins = cur[y - 1] + 1;                            /* d[x][y-1] + insertion_cost */
      int sub = prev[y - 1] + (a[x - 1] != b[y - 1]);      /* d[x-1][y-1] + I(a_x != b_y) */
      int m = del < ins ? del : ins;
      cur[y] = m < sub ? m : sub;
    }
    int* t = prev; prev = cur; cur = t;
  }
  int d = prev[lb];
  free(prev); free(cur);
  return d;
}

static inline uint16_t saturate(int d, int max_d) {
  /* output convention (spec C1 / reading 13): min(d, max_d+1); exact if max_d < 0 */
  if (max_d >= 0 && d > max_d) d = max_d + 1;
  return (uint16_t)d;
}

/* distances for an explicit pair list, in input order */
void orc_edit_distance_pairs(const uint8_t* seqs, const int64_t* off, const uint32_t* pairs,
                             int64_t n_pairs, int max_d, uint16_t* dist_out) {
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t p = 0; p < n_pairs; ++p) {
    uint32_t i = pairs[2 * p], j = pairs[2 * p + 1];
    int d = orc_wagner_fischer(seqs + off[i], (int)(off[i + 1] - off[i]),
                               seqs + off[j], (int)(off[j + 1] - off[j]));
    dist_out[p] = saturate(d, max_d);
  }
}

/* exhaustive all pairs, unthresholded: condensed row-major upper triangle
 * (0,1),(0,2)...(n-2,n-1)  (Eq. 45 read as a self-join, reading 15) */
void orc_all_pairs_full(const uint8_t* seqs, const int64_t* off, int64_t n, uint16_t* dist_out) {
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t i = 0; i < n; ++i) {
    int64_t base = i * (2 * n - i - 1) / 2;    /* number of pairs with first index < i */
    for (int64_t j = i + 1; j < n; ++j) {
      int d = orc_wagner_fischer(seqs + off[i], (int)(off[i + 1] - off[i]),
                                 seqs + off[j], (int)(off[j + 1] - off[j]));
      dist_out[base + (j - i - 1)] = (uint16_t)d;
    }
  }
}

/* Tier B distance with Ukkonen cut-off: exact d if d <= max_d, else any value > max_d.
 * Cells with |x-y| > max_d cannot lie on a path of cost <= max_d, so they are treated as
 * infinity; validated against orc_wagner_fischer in tests/test_oracle_edit.py. */
int orc_wagner_fischer_cutoff(const uint8_t* a, int la, const uint8_t* b, int lb, int max_d) {
  const int INF = 1 << 28;
  int diff = la > lb ? la - lb : lb - la;
  if (diff > max_d) return max_d + 1;
  int* prev = (int*)malloc(sizeof(int) * (size_t)(lb + 1));
  int* cur = (int*)malloc(sizeof(int) * (size_t)(lb + 1));
  for (int y = 0; y <= lb; ++y) prev[y] = (y <= max_d) ? y : INF;
  for (int x = 1; x <= la; ++x) {
    int ylo = x - max_d < 1 ? 1 : x - max_d;
    int yhi = x + max_d > lb ? lb : x + max_d;
    for (int y = 0; y <= lb; ++y) cur[y] = INF;
    if (x <= max_d) cur[0] = x;
    int best = cur[0];
    for (int y = ylo; y <= yhi; ++y) {
      int del = prev[y] + 1, ins = cur[y - 1] + 1, sub = prev[y - 1] + (a[x - 1] != b[y - 1]);
      int m = del < ins ? del : ins;
      m = m < sub ? m : sub;
      if (m > INF) m = INF;
      cur[y] = m;
      if (m < best) best = m;
    }
    int* t = prev; prev = cur; cur = t;
    if (best > max_d) { free(prev); free(cur); return max_d + 1; }
  }
  int d = prev[lb];
  free(prev); free(cur);
  return d > max_d ? max_d + 1 : d;
}

/* ------------------------------------------------------------------------ */
/* C1w. Weighted edit distance (reading 22). */
/* PAPER.md L754 Eq. (46) as printed: D(i,j) = min(D(i-1,j) + deletion_cost,  */
/* D(i,j-1) + insertion_cost, D(i-1,j-1) + substitution_cost(a_i, b_j)), with */
/* the substitution cost taken from a table ("typically based on biochemical  */
/* similarity", L760) and one common insertion/deletion cost `indel`.         */
/* Boundary D[x][0] = x*indel, D[0][y] = y*indel.  sub is [sigma][sigma],     */
/* row = residue of a, column = residue of b.  Wagner-Fischer, written out.   */
/* ------------------------------------------------------------------------ */
int orc_wagner_fischer_weighted(const uint8_t* a, int la, const uint8_t* b, int lb,
                                const uint8_t* sub, int sigma, int indel) {
  int* prev = (int*)malloc(sizeof(int) * (size_t)(lb + 1));
  int* cur = (int*)malloc(sizeof(int) * (size_t)(lb + 1));
  for (int y = 0; y <= lb; ++y) prev[y] = y * indel;
  for (int x = 1; x <= la; ++x) {
    cur[0] = x * indel;
    for (int y = 1; y <= lb; ++y) {
      int del = prev[y] + indel;
      int ins = cur[y - 1] + indel;
      /* Eq. 46: I(s_i[x] != s_j[y]) * substitution_cost -- equal residues cost 0, whatever the
       * table's diagonal holds (reading 22b) */
      int sb = prev[y - 1] + (a[x - 1] != b[y - 1] ? (int)sub[(int)a[x - 1] * sigma + (int)b[y - 1]] : 0);
      int m = del < ins ? del : ins;
      cur[y] = m < sb ? m : sb;
    }
    int* t = prev; prev = cur; cur = t;
  }
  int d = prev[lb];
  free(prev); free(cur);
  return d;
}

void orc_edit_distance_weighted_pairs(const uint8_t* seqs, const int64_t* off, const uint32_t* pairs,
                                      int64_t n_pairs, const uint8_t* sub, int sigma, int indel,
                                      int max_d, uint16_t* dist_out) {
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t p = 0; p < n_pairs; ++p) {
    uint32_t i = pairs[2 * p], j = pairs[2 * p + 1];
    int d = orc_wagner_fischer_weighted(seqs + off[i], (int)(off[i + 1] - off[i]),
                                        seqs + off[j], (int)(off[j + 1] - off[j]), sub, sigma, indel);
    dist_out[p] = saturate(d, max_d);
  }
}

/* exhaustive all pairs with threshold: hits (i<j, d <= max_d) in ascending (i,j) order.
 * use_cutoff = 0: Tier A (full Wagner-Fischer); 1: Tier B (cut-off DP).
 * Returns the number of hits; writes at most `capacity` of them. */
int64_t orc_all_pairs_threshold(const uint8_t* seqs, const int64_t* off, int64_t n, int max_d,
                                int use_cutoff, uint32_t* pairs_out, uint16_t* dist_out,
                                int64_t capacity) {
  int64_t* row_cnt = (int64_t*)calloc((size_t)n + 1, sizeof(int64_t));
  /* pass 1: count hits per row; pass 2: fill at the row's offset -> deterministic order */
  for (int pass = 0; pass < 2; ++pass) {
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t i = 0; i < n; ++i) {
      int64_t w = row_cnt[i], c = 0;
      int la = (int)(off[i + 1] - off[i]);
      for (int64_t j = i + 1; j < n; ++j) {
        int lb = (int)(off[j + 1] - off[j]);
        int d = use_cutoff ? orc_wagner_fischer_cutoff(seqs + off[i], la, seqs + off[j], lb, max_d)
                           : orc_wagner_fischer(seqs + off[i], la, seqs + off[j], lb);
        if (d <= max_d) {
          if (pass == 1 && w + c < capacity) {
            pairs_out[2 * (w + c)] = (uint32_t)i;
            pairs_out[2 * (w + c) + 1] = (uint32_t)j;
            dist_out[w + c] = (uint16_t)d;
          }
          ++c;
        }
      }
      if (pass == 0) row_cnt[i] = c;
    }
    if (pass == 0) {           /* exclusive prefix sum of the row counts */
      int64_t acc = 0;
      for (int64_t i = 0; i <= n; ++i) { int64_t c = row_cnt[i]; row_cnt[i] = acc; acc += c; }
    }
  }
  int64_t total = row_cnt[n];
  free(row_cnt);
  return total;
}

/* ------------------------------------------------------------------------ */
/* C2. MinHash.  All arithmetic mod 2^32.                                    */
/* ------------------------------------------------------------------------ */
/* base mixer g: uint32 -> uint32 (bijective) */
uint32_t orc_mix32(uint32_t x) {
  x ^= x >> 16;
  x *= 0x6A09E667u;     /* frac(sqrt 2) * 2^32, odd */
  x ^= x >> 15;
  x *= 0xBB67AE85u;     /* frac(sqrt 3) * 2^32, odd */
  x ^= x >> 16;
  return x;
}

/* per-hash parameters from the 64-bit seed: a_j = g(lo ^ g(2j+1)) | 1, b_j = g(hi ^ g(2j+2)) */
void orc_hash_params(uint64_t seed, int H, uint32_t* a, uint32_t* b) {
  uint32_t lo = (uint32_t)(seed & 0xFFFFFFFFu), hi = (uint32_t)(seed >> 32);
  for (int j = 0; j < H; ++j) {
    a[j] = orc_mix32(lo ^ orc_mix32((uint32_t)(2 * j + 1))) | 1u;
    b[j] = orc_mix32(hi ^ orc_mix32((uint32_t)(2 * j + 2)));
  }
}

static int cmp_u32(const void* p, const void* q) {
  uint32_t a = *(const uint32_t*)p, b = *(const uint32_t*)q;
  return a < b ? -1 : a > b;
}

/* signature of ONE sequence: explicit k-mer SET, then per-hash minimum over the set.
 * x_p = sum_t code[p+t] * 32^(k-1-t);  h_j(x) = a_j * g(x) + b_j;  sig[j] = min_x h_j(x).
 * L < k  ->  all 0xFFFFFFFF ("empty", reading 4). */
void orc_minhash_one(const uint8_t* s, int L, int k, int H, const uint32_t* a, const uint32_t* b,
                     uint32_t* sig) {
  for (int j = 0; j < H; ++j) sig[j] = 0xFFFFFFFFu;
  int nk = L - k + 1;
  if (nk <= 0) return;
  uint32_t* set = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)nk);
  for (int p = 0; p < nk; ++p) {
    uint32_t x = 0;
    for (int t = 0; t < k; ++t) x = x * 32u + s[p + t];
    set[p] = x;
  }
  qsort(set, (size_t)nk, sizeof(uint32_t), cmp_u32);       /* set semantics: dedupe */
  int m = 0;
  for (int p = 0; p < nk; ++p)
    if (p == 0 || set[p] != set[p - 1]) set[m++] = set[p];
  for (int j = 0; j < H; ++j) {
    uint32_t best = 0xFFFFFFFFu;
    for (int e = 0; e < m; ++e) {
      uint32_t h = a[j] * orc_mix32(set[e]) + b[j];
      if (h < best) best = h;
    }
    sig[j] = best;
  }
  free(set);
}

void orc_minhash(const uint8_t* seqs, const int64_t* off, int64_t n, int k, int H, uint64_t seed,
                 uint32_t* sig_out /* [n][H] row-major */) {
  uint32_t* a = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)H);
  uint32_t* b = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)H);
  orc_hash_params(seed, H, a, b);
#pragma omp parallel for schedule(dynamic, 256)
  for (int64_t i = 0; i < n; ++i)
    orc_minhash_one(seqs + off[i], (int)(off[i + 1] - off[i]), k, H, a, b, sig_out + i * H);
  free(a); free(b);
}

/* exact Jaccard of the k-mer SETS of two sequences, as a fraction num/den (pin for Eq. 30) */
void orc_kmer_jaccard(const uint8_t* s, int Ls, const uint8_t* t, int Lt, int k,
                      int* num, int* den) {
  int ns = Ls - k + 1, nt = Lt - k + 1;
  if (ns < 0) ns = 0;
  if (nt < 0) nt = 0;
  uint32_t* A = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(ns + 1));
  uint32_t* B = (uint32_t*)malloc(sizeof(uint32_t) * (size_t)(nt + 1));
  for (int p = 0; p < ns; ++p) { uint32_t x = 0; for (int q = 0; q < k; ++q) x = x * 32u + s[p + q]; A[p] = x; }
  for (int p = 0; p < nt; ++p) { uint32_t x = 0; for (int q = 0; q < k; ++q) x = x * 32u + t[p + q]; B[p] = x; }
  qsort(A, (size_t)ns, sizeof(uint32_t), cmp_u32);
  qsort(B, (size_t)nt, sizeof(uint32_t), cmp_u32);
  int ma = 0, mb = 0;
  for (int p = 0; p < ns; ++p) if (p == 0 || A[p] != A[p - 1]) A[ma++] = A[p];
  for (int p = 0; p < nt; ++p) if (p == 0 || B[p] != B[p - 1]) B[mb++] = B[p];
  int x = 0, y = 0, inter = 0;
  while (x < ma && y < mb) {
    if (A[x] == B[y]) { ++inter; ++x; ++y; }
    else if (A[x] < B[y]) ++x; else ++y;
  }
  *num = inter;
  *den = ma + mb - inter;
  free(A); free(B);
}

/* ------------------------------------------------------------------------ */
/* C3. LSH banding -> candidate pairs.                                       */
/* ------------------------------------------------------------------------ */
/* band key: acc = 0x6A09E667F3BCC908; for v in tuple: acc = (acc ^ v) * 0x9E3779B97F4A7C15;
 * acc ^= acc >> 29  (both statements inside the loop) */
uint64_t orc_band_key(const uint32_t* tuple, int rows) {
  uint64_t acc = 0x6A09E667F3BCC908ull;
  for (int r = 0; r < rows; ++r) {
    acc = (acc ^ (uint64_t)tuple[r]) * 0x9E3779B97F4A7C15ull;
    acc ^= acc >> 29;
  }
  return acc;
}

static int sig_is_empty(const uint32_t* sig, int H) {
  /* L < k  <=>  every entry is the sentinel.  (A non-empty k-mer set can reach the sentinel in
   * one hash, so the whole row is tested.) */
  for (int j = 0; j < H; ++j) if (sig[j] != 0xFFFFFFFFu) return 0;
  return 1;
}

static int cmp_pair(const void* p, const void* q) {
  const uint32_t* a = (const uint32_t*)p; const uint32_t* b = (const uint32_t*)q;
  if (a[0] != b[0]) return a[0] < b[0] ? -1 : 1;
  if (a[1] != b[1]) return a[1] < b[1] ? -1 : 1;
  return 0;
}

/* Tier A: brute force over all pairs and all bands by TUPLE equality.
 * kept[b][i] = 1 iff fewer than `cap` sequences with a smaller index share i's band-b tuple
 * ("keep the cap smallest indices", reading 8).  A pair is a candidate iff in some band both
 * are kept and their tuples are equal.  Output ascending (i,j), duplicate free by construction.
 * Returns the number of candidates; writes at most `capacity`.
 * *key_tuple_mismatch is set to the number of (pair, band) events where 64-bit key equality and
 * tuple equality disagree (spec C3 requires 0). */
int64_t orc_lsh_bruteforce(const uint32_t* sig, int64_t n, int H, int bands, int rows, int cap,
                           uint32_t* pairs_out, int64_t capacity, int64_t* key_tuple_mismatch) {
  uint8_t* kept = (uint8_t*)calloc((size_t)(n * bands) + 1, 1);
  uint8_t* empty = (uint8_t*)calloc((size_t)n + 1, 1);
  uint64_t* keys = (uint64_t*)malloc(sizeof(uint64_t) * (size_t)(n * bands + 1));
  for (int64_t i = 0; i < n; ++i) {
    empty[i] = (uint8_t)sig_is_empty(sig + i * H, H);
    for (int b = 0; b < bands; ++b) keys[i * bands + b] = orc_band_key(sig + i * H + b * rows, rows);
  }
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n; ++i) {
    if (empty[i]) continue;
    for (int b = 0; b < bands; ++b) {
      int rank = 0;
      const uint32_t* ti = sig + i * H + b * rows;
      for (int64_t j = 0; j < i && rank < cap; ++j)
        if (!empty[j] && memcmp(ti, sig + j * H + b * rows, sizeof(uint32_t) * (size_t)rows) == 0) ++rank;
      kept[i * bands + b] = (uint8_t)(rank < cap);
    }
  }
  int64_t* row_cnt = (int64_t*)calloc((size_t)n + 1, sizeof(int64_t));
  int64_t mism = 0;
  for (int pass = 0; pass < 2; ++pass) {
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : mism)
    for (int64_t i = 0; i < n; ++i) {
      int64_t w = row_cnt[i], c = 0;
      if (empty[i]) { if (pass == 0) row_cnt[i] = 0; continue; }
      for (int64_t j = i + 1; j < n; ++j) {
        if (empty[j]) continue;
        int cand = 0;
        for (int b = 0; b < bands; ++b) {
          int teq = memcmp(sig + i * H + b * rows, sig + j * H + b * rows,
                           sizeof(uint32_t) * (size_t)rows) == 0;
          int keq = keys[i * bands + b] == keys[j * bands + b];
          if (pass == 0 && teq != keq) ++mism;
          if (teq && kept[i * bands + b] && kept[j * bands + b]) cand = 1;
        }
        if (cand) {
          if (pass == 1 && w + c < capacity) {
            pairs_out[2 * (w + c)] = (uint32_t)i;
            pairs_out[2 * (w + c) + 1] = (uint32_t)j;
          }
          ++c;
        }
      }
      if (pass == 0) row_cnt[i] = c;
    }
    if (pass == 0) {
      int64_t acc = 0;
      for (int64_t i = 0; i <= n; ++i) { int64_t c = row_cnt[i]; row_cnt[i] = acc; acc += c; }
    }
  }
  int64_t total = row_cnt[n];
  if (key_tuple_mismatch) *key_tuple_mismatch = mism;
  free(kept); free(empty); free(keys); free(row_cnt);
  return total;
}

/* Tier B: sort (band, key, id) records with the C library sort, walk the buckets, keep the
 * `cap` smallest ids of each, emit all i<j among the kept, then sort + unique the pair list.
 * Buckets are formed by 64-bit KEY equality (authoritative, spec C3); every bucket is checked
 * for tuple equality and disagreements are counted in *key_tuple_mismatch.
 * Also returns the number of pairs before cross-band de-duplication in *n_raw.
 * Validated against orc_lsh_bruteforce in tests/test_oracle_lsh.py. */
typedef struct { uint64_t key; uint32_t band; uint32_t id; } rec_t;
static int cmp_rec(const void* p, const void* q) {
  const rec_t* a = (const rec_t*)p; const rec_t* b = (const rec_t*)q;
  if (a->band != b->band) return a->band < b->band ? -1 : 1;
  if (a->key != b->key) return a->key < b->key ? -1 : 1;
  if (a->id != b->id) return a->id < b->id ? -1 : 1;
  return 0;
}

int64_t orc_lsh_sorted(const uint32_t* sig, int64_t n, int H, int bands, int rows, int cap,
                       uint32_t* pairs_out, int64_t capacity, int64_t* n_raw,
                       int64_t* key_tuple_mismatch) {
  int64_t nrec = 0;
  rec_t* rec = (rec_t*)malloc(sizeof(rec_t) * (size_t)(n * bands + 1));
  for (int64_t i = 0; i < n; ++i) {
    if (sig_is_empty(sig + i * H, H)) continue;
    for (int b = 0; b < bands; ++b) {
      rec[nrec].band = (uint32_t)b;
      rec[nrec].key = orc_band_key(sig + i * H + b * rows, rows);
      rec[nrec].id = (uint32_t)i;
      ++nrec;
    }
  }
  qsort(rec, (size_t)nrec, sizeof(rec_t), cmp_rec);
  /* pass 1: count raw pairs; pass 2: fill */
  int64_t raw = 0, mism = 0;
  for (int64_t s = 0; s < nrec;) {
    int64_t e = s + 1;
    while (e < nrec && rec[e].band == rec[s].band && rec[e].key == rec[s].key) ++e;
    for (int64_t q = s + 1; q < e; ++q)
      if (memcmp(sig + (int64_t)rec[q].id * H + rec[q].band * rows,
                 sig + (int64_t)rec[s].id * H + rec[s].band * rows,
                 sizeof(uint32_t) * (size_t)rows) != 0) ++mism;
    int64_t m = e - s;
    if (m > cap) m = cap;
    raw += m * (m - 1) / 2;
    s = e;
  }
  uint32_t* tmp = (uint32_t*)malloc(sizeof(uint32_t) * 2 * (size_t)(raw + 1));
  int64_t w = 0;
  for (int64_t s = 0; s < nrec;) {
    int64_t e = s + 1;
    while (e < nrec && rec[e].band == rec[s].band && rec[e].key == rec[s].key) ++e;
    int64_t m = e - s;
    if (m > cap) m = cap;                 /* ids ascend inside the bucket: first `cap` kept */
    for (int64_t u = s; u < s + m; ++u)
      for (int64_t v = u + 1; v < s + m; ++v) {
        tmp[2 * w] = rec[u].id; tmp[2 * w + 1] = rec[v].id; ++w;
      }
    s = e;
  }
  qsort(tmp, (size_t)raw, 2 * sizeof(uint32_t), cmp_pair);
  int64_t uniq = 0;
  for (int64_t p = 0; p < raw; ++p) {
    if (p > 0 && tmp[2 * p] == tmp[2 * p - 2] && tmp[2 * p + 1] == tmp[2 * p - 1]) continue;
    if (uniq < capacity) { pairs_out[2 * uniq] = tmp[2 * p]; pairs_out[2 * uniq + 1] = tmp[2 * p + 1]; }
    ++uniq;
  }
  if (n_raw) *n_raw = raw;
  if (key_tuple_mismatch) *key_tuple_mismatch = mism;
  free(tmp); free(rec);
  return uniq;
}

/* One row of CAND by definition, for spot checks at sizes where the whole set is too large:
 * all partners j != i of sequence i (ascending, duplicate free).  For every band the whole
 * bucket of i is collected by one scan over all sequences (tuple equality), so the ranks that
 * decide "kept" are explicit.  Returns the partner count; writes at most `capacity`. */
int64_t orc_lsh_row(const uint32_t* sig, int64_t n, int H, int bands, int rows, int cap,
                    int64_t i, uint32_t* partners_out, int64_t capacity) {
  if (sig_is_empty(sig + i * H, H)) return 0;
  uint8_t* mark = (uint8_t*)calloc((size_t)n + 1, 1);
  for (int b = 0; b < bands; ++b) {
    const uint32_t* ti = sig + i * H + b * rows;
    int64_t rank = 0; int i_kept = 0;
    /* first scan: is i among the first `cap` members of its bucket? */
    for (int64_t j = 0; j < n && rank < cap; ++j) {
      if (sig_is_empty(sig + j * H, H)) continue;
      if (memcmp(ti, sig + j * H + b * rows, sizeof(uint32_t) * (size_t)rows) == 0) {
        if (j == i) i_kept = 1;
        ++rank;
      }
    }
    if (!i_kept) continue;
    rank = 0;
    for (int64_t j = 0; j < n && rank < cap; ++j) {
      if (sig_is_empty(sig + j * H, H)) continue;
      if (memcmp(ti, sig + j * H + b * rows, sizeof(uint32_t) * (size_t)rows) == 0) {
        if (j != i) mark[j] = 1;
        ++rank;
      }
    }
  }
  int64_t c = 0;
  for (int64_t j = 0; j < n; ++j)
    if (mark[j]) { if (c < capacity) partners_out[c] = (uint32_t)j; ++c; }
  free(mark);
  return c;
}
