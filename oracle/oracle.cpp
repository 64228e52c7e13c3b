// oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU restatement of what the hot path of
// arXiv 1702.08734 ("Billion-scale similarity search with GPUs") computes.
// Written from the paper (PAPER.md, cited as P:L<line>), before any kernel.
// It shares no code, header, table or helper with the CUDA path
// (paper_1702_08734_b200/csrc) and neither includes the other.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load this library.
//
// What each entry point follows:
//   orc_kselect        P:L48      k lowest values with their indices: the plain
//                                 definition, by a full sort of (value, index).
//   orc_kselect_largest P:L48     "other comparators": the k highest values, by a full
//                                 sort with the value order reversed (ties still to the
//                                 lower index, NaN still last).
//   orc_flat_l2_knn    P:L41-57   Eq. (1) with D squared, distances in
//                                 the DIRECT form sum_c (x_c - y_c)^2 in double
//                                 (deliberately not Eq. (2), which the GPU uses).
//   orc_pair_l2        P:L52      the same distance for given (query, id) pairs.
//   orc_ivfpq_encode   P:L61-63, L86-90   Eq. (3): q1 = nearest coarse centroid,
//                                 q2 = product quantizer on the residual, one byte
//                                 per sub-quantizer, byte m = sub-quantizer m.
//   orc_ivfpq_search   P:L72-78, L276, L327-353   Alg. 4 with Eq. (5)-(7):
//                                 tau-argmin over C1, then ||x - q(y)||^2 by
//                                 EXPLICIT RECONSTRUCTION (no lookup tables),
//                                 then k-select.
//   orc_adc_lut_sum    P:L288-290 Eq. (10): the same distance as a sum of b table
//                                 look-ups; exists so that a test can pin
//                                 "reconstruction distance == LUT sum".
//   orc_adc_eq11       P:L302     Eq. (11): term1 + term2 - 2*term3.
//   orc_kmeans_step    P:L392-398 one Lloyd iteration: nearest-centroid assignment
//                                 (double, direct form), cluster means; the library's
//                                 stated empty-cluster rule restated (fs.h, fs_kmeans).
//
// Readings of the paper where it is silent:
//   ties -> lower index / lower id / lower centroid number; -0 == +0; NaN sorts
//   after +inf; distances are squared; k > candidates pads with (+inf, -1).
//
// Pins: tests/test_oracle_*.py (hand-worked examples, closed forms, brute force
// by independent routines, invariants, limits that reduce to textbook cases).
// Parity-unpinned: nothing in this file; recall on the paper's datasets is out
// of scope (datasets absent).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Order used by every selection here: value ascending under IEEE comparison
// (so -0.0 == +0.0), NaN after everything, then index ascending.
template <typename V, typename I>
struct Pair {
  V v;
  I i;
};

template <typename V, typename I>
inline bool pair_less(const Pair<V, I>& a, const Pair<V, I>& b) {
  const bool an = std::isnan(a.v), bn = std::isnan(b.v);
  if (an != bn) return bn;           // the non-NaN one is smaller
  if (!an) {
    if (a.v < b.v) return true;
    if (b.v < a.v) return false;
  }
  return a.i < b.i;
}

// the reversed value order of the k-largest variant: higher value first, NaN last, then index ascending
template <typename V, typename I>
inline bool pair_greater(const Pair<V, I>& a, const Pair<V, I>& b) {
  const bool an = std::isnan(a.v), bn = std::isnan(b.v);
  if (an != bn) return bn;
  if (!an) {
    if (a.v > b.v) return true;
    if (b.v > a.v) return false;
  }
  return a.i < b.i;
}

}  // namespace

extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---------------------------------------------------------------------------
// k-selection.  rows: [n_rows][ld] fp32, the first n of each row are
// the array [a_i].  out_val/out_idx: [n_rows][k].  Full sort of all n pairs.
// ---------------------------------------------------------------------------
void orc_kselect(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int64_t k,
                 float* out_val, int32_t* out_idx) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t r = 0; r < n_rows; ++r) {
    const float* a = rows + r * ld;
    std::vector<Pair<float, int64_t>> p((size_t)n);
    for (int64_t i = 0; i < n; ++i) p[(size_t)i] = {a[i], i};
    std::sort(p.begin(), p.end(), pair_less<float, int64_t>);
    for (int64_t j = 0; j < k; ++j) {
      if (j < n) {
        out_val[r * k + j] = a[p[(size_t)j].i];  // original bits
        out_idx[r * k + j] = (int32_t)p[(size_t)j].i;
      } else {
        out_val[r * k + j] = std::numeric_limits<float>::infinity();
        out_idx[r * k + j] = -1;
      }
    }
  }
}

// P:L48 "other comparators are sometimes desired": the k HIGHEST values, descending.
void orc_kselect_largest(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int64_t k,
                         float* out_val, int32_t* out_idx) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t r = 0; r < n_rows; ++r) {
    const float* a = rows + r * ld;
    std::vector<Pair<float, int64_t>> p((size_t)n);
    for (int64_t i = 0; i < n; ++i) p[(size_t)i] = {a[i], i};
    std::sort(p.begin(), p.end(), pair_greater<float, int64_t>);
    for (int64_t j = 0; j < k; ++j) {
      if (j < n) {
        out_val[r * k + j] = a[p[(size_t)j].i];
        out_idx[r * k + j] = (int32_t)p[(size_t)j].i;
      } else {
        out_val[r * k + j] = -std::numeric_limits<float>::infinity();
        out_idx[r * k + j] = -1;
      }
    }
  }
}

// ---------------------------------------------------------------------------
// Exact search, Eq. (1) P:L43 with squared distances.
// xq [nq][d], xb [nb][d] fp32 row-major.  out_dist (fp32, rounded from double),
// out_dist64 (optional, may be NULL), out_ids int64: [nq][k].
// ---------------------------------------------------------------------------
static inline double l2_direct(const float* x, const float* y, int64_t d) {
  double s = 0.0;
  for (int64_t c = 0; c < d; ++c) {
    const double t = (double)x[c] - (double)y[c];
    s += t * t;
  }
  return s;
}

void orc_flat_l2_knn(const float* xq, int64_t nq, const float* xb, int64_t nb, int64_t d,
                     int64_t k, float* out_dist, double* out_dist64, int64_t* out_ids) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t j = 0; j < nq; ++j) {
    std::vector<Pair<double, int64_t>> p((size_t)nb);
    for (int64_t i = 0; i < nb; ++i) p[(size_t)i] = {l2_direct(xq + j * d, xb + i * d, d), i};
    std::sort(p.begin(), p.end(), pair_less<double, int64_t>);
    for (int64_t t = 0; t < k; ++t) {
      const bool have = t < nb;
      const double dv = have ? p[(size_t)t].v : std::numeric_limits<double>::infinity();
      out_dist[j * k + t] = (float)dv;
      if (out_dist64) out_dist64[j * k + t] = dv;
      out_ids[j * k + t] = have ? p[(size_t)t].i : -1;
    }
  }
}

// Distances for given pairs: out[j*m + t] = ||xq_j - xb_{ids[j*m+t]}||^2 (double);
// id < 0 gives +inf.
void orc_pair_l2(const float* xq, int64_t nq, const float* xb, int64_t d, const int64_t* ids,
                 int64_t m, double* out) {
#pragma omp parallel for
  for (int64_t j = 0; j < nq; ++j)
    for (int64_t t = 0; t < m; ++t) {
      const int64_t id = ids[j * m + t];
      out[j * m + t] = id < 0 ? std::numeric_limits<double>::infinity()
                              : l2_direct(xq + j * d, xb + id * d, d);
    }
}

// ---------------------------------------------------------------------------
// IVFADC add path, Eq. (3); product quantizer P:L86-90.
// coarse [nlist][d]; pq [M][256][dsub] with dsub = d/M, sub-vector m = dims
// [m*dsub, (m+1)*dsub).  For each y: list = argmin_c ||y - c||^2 (ties -> lower
// c); r = y - coarse[list]; code[m] = argmin_j ||r^m - pq[m][j]||^2 (ties ->
// lower j).  All in double.  Optional margins (may be NULL): the relative gap
// between the best and the second-best distance, (d2 - d1) / max(d2, tiny), for
// the coarse choice [n] and for each sub-quantizer choice [n][M]; a test uses
// them to excuse near-ties, never to compute anything.
// ---------------------------------------------------------------------------
void orc_ivfpq_encode(const float* coarse, const float* pq, int64_t d, int64_t nlist, int64_t M,
                      const float* y, int64_t n, int32_t* out_list, uint8_t* out_codes,
                      double* out_coarse_margin, double* out_code_margin) {
  const int64_t dsub = d / M;
  const double tiny = 1e-300;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n; ++i) {
    const float* yi = y + i * d;
    double best = std::numeric_limits<double>::infinity(), second = best;
    int64_t bl = -1;
    for (int64_t c = 0; c < nlist; ++c) {
      const double dist = l2_direct(yi, coarse + c * d, d);
      if (dist < best) {
        second = best;
        best = dist;
        bl = c;
      } else if (dist < second) {
        second = dist;
      }
    }
    out_list[i] = (int32_t)bl;
    if (out_coarse_margin) out_coarse_margin[i] = (second - best) / std::max(second, tiny);
    const float* cl = coarse + bl * d;
    for (int64_t m = 0; m < M; ++m) {
      double b1 = std::numeric_limits<double>::infinity(), b2 = b1;
      int64_t bj = -1;
      for (int64_t j = 0; j < 256; ++j) {
        const float* cw = pq + (m * 256 + j) * dsub;
        double s = 0.0;
        for (int64_t c = 0; c < dsub; ++c) {
          const double r = (double)yi[m * dsub + c] - (double)cl[m * dsub + c];
          const double t = r - (double)cw[c];
          s += t * t;
        }
        if (s < b1) {
          b2 = b1;
          b1 = s;
          bj = j;
        } else if (s < b2) {
          b2 = s;
        }
      }
      out_codes[i * M + m] = (uint8_t)bj;
      if (out_code_margin) out_code_margin[i * M + m] = (b2 - b1) / std::max(b2, tiny);
    }
  }
}

// ||x - (coarse[list] + concat_m pq[m][code_m])||^2 in double, Eq. (7) P:L276.
static inline double adc_reconstruct(const float* x, const float* cl, const float* pq,
                                     const uint8_t* code, int64_t M, int64_t dsub) {
  double s = 0.0;
  for (int64_t m = 0; m < M; ++m) {
    const float* cw = pq + (m * 256 + code[m]) * dsub;
    for (int64_t c = 0; c < dsub; ++c) {
      const double yhat = (double)cl[m * dsub + c] + (double)cw[c];
      const double t = (double)x[m * dsub + c] - yhat;
      s += t * t;
    }
  }
  return s;
}

// ---------------------------------------------------------------------------
// Alg. 4 IVFPQ-SEARCH.  Inverted file in CSR form: list L holds
// entries offsets[L] .. offsets[L+1]-1 of codes [ntotal][M] and ids [ntotal].
// Step 1 (Eq. 5): L_IVF = nprobe lowest ||x - c||^2 by (dist, c).
// Step 2 (Eq. 7): for every entry of every probed list the distance
//        by explicit reconstruction.
// Step 3 (Eq. 6): k lowest by (dist, id).
// Outputs: out_dist fp32 / out_dist64 (optional) / out_ids [nq][k], padded with
// (+inf, -1); out_probed int32 [nq][nprobe] and out_coarse64 [nq][nprobe]
// (optional) in ascending coarse distance.  If probed_in is non-NULL step 1 is
// skipped and those lists are scanned instead (used to check step 2-3 alone).
// ---------------------------------------------------------------------------
void orc_ivfpq_search(const float* coarse, const float* pq, int64_t d, int64_t nlist, int64_t M,
                      const int64_t* offsets, const uint8_t* codes, const int64_t* ids,
                      const float* xq, int64_t nq, int64_t nprobe, int64_t k,
                      const int32_t* probed_in, float* out_dist, double* out_dist64,
                      int64_t* out_ids, int32_t* out_probed, double* out_coarse64) {
  const int64_t dsub = d / M;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t q = 0; q < nq; ++q) {
    const float* x = xq + q * d;
    std::vector<int32_t> probes((size_t)nprobe);
    if (probed_in) {
      for (int64_t t = 0; t < nprobe; ++t) probes[(size_t)t] = probed_in[q * nprobe + t];
      if (out_probed)
        for (int64_t t = 0; t < nprobe; ++t) out_probed[q * nprobe + t] = probes[(size_t)t];
    } else {
      std::vector<Pair<double, int64_t>> cd((size_t)nlist);
      for (int64_t c = 0; c < nlist; ++c) cd[(size_t)c] = {l2_direct(x, coarse + c * d, d), c};
      std::sort(cd.begin(), cd.end(), pair_less<double, int64_t>);
      for (int64_t t = 0; t < nprobe; ++t) {
        const bool have = t < nlist;
        probes[(size_t)t] = have ? (int32_t)cd[(size_t)t].i : -1;
        if (out_probed) out_probed[q * nprobe + t] = probes[(size_t)t];
        if (out_coarse64)
          out_coarse64[q * nprobe + t] =
              have ? cd[(size_t)t].v : std::numeric_limits<double>::infinity();
      }
    }
    std::vector<Pair<double, int64_t>> cand;
    for (int64_t t = 0; t < nprobe; ++t) {
      const int64_t L = probes[(size_t)t];
      if (L < 0) continue;
      for (int64_t e = offsets[L]; e < offsets[L + 1]; ++e)
        cand.push_back({adc_reconstruct(x, coarse + L * d, pq, codes + e * M, M, dsub), ids[e]});
    }
    std::sort(cand.begin(), cand.end(), pair_less<double, int64_t>);
    for (int64_t t = 0; t < k; ++t) {
      const bool have = t < (int64_t)cand.size();
      const double dv = have ? cand[(size_t)t].v : std::numeric_limits<double>::infinity();
      out_dist[q * k + t] = (float)dv;
      if (out_dist64) out_dist64[q * k + t] = dv;
      out_ids[q * k + t] = have ? cand[(size_t)t].i : -1;
    }
  }
}

// ADC distance by reconstruction for given (query, list, code) triples.
void orc_adc_reconstruct(const float* coarse, const float* pq, int64_t d, int64_t M,
                         const float* x, const int32_t* list_no, const uint8_t* codes, int64_t n,
                         double* out) {
  const int64_t dsub = d / M;
  for (int64_t i = 0; i < n; ++i)
    out[i] = adc_reconstruct(x + i * d, coarse + (int64_t)list_no[i] * d, pq, codes + i * M, M, dsub);
}

// Eq. (10): tables T_m[j] = ||(x - c_L)^m - pq[m][j]||^2 for one
// (query, list) pair, then the distance of each code as sum_m T_m[code_m].
// tables_out (optional) [M][256].
void orc_adc_lut_sum(const float* coarse, const float* pq, int64_t d, int64_t M, const float* x,
                     int64_t list_no, const uint8_t* codes, int64_t n, double* out,
                     double* tables_out) {
  const int64_t dsub = d / M;
  std::vector<double> T((size_t)(M * 256));
  const float* cl = coarse + list_no * d;
  for (int64_t m = 0; m < M; ++m)
    for (int64_t j = 0; j < 256; ++j) {
      double s = 0.0;
      for (int64_t c = 0; c < dsub; ++c) {
        const double xt = (double)x[m * dsub + c] - (double)cl[m * dsub + c];
        const double t = xt - (double)pq[(m * 256 + j) * dsub + c];
        s += t * t;
      }
      T[(size_t)(m * 256 + j)] = s;
    }
  if (tables_out) std::memcpy(tables_out, T.data(), sizeof(double) * (size_t)(M * 256));
  for (int64_t i = 0; i < n; ++i) {
    double s = 0.0;
    for (int64_t m = 0; m < M; ++m) s += T[(size_t)(m * 256 + codes[i * M + m])];
    out[i] = s;
  }
}

// Eq. (11): ||q2||^2 + 2<q1, q2> (term 1) + ||x - q1||^2 (term 2)
// - 2 <x, q2> (term 3), for one (query, list) pair and n codes.
void orc_adc_eq11(const float* coarse, const float* pq, int64_t d, int64_t M, const float* x,
                  int64_t list_no, const uint8_t* codes, int64_t n, double* out) {
  const int64_t dsub = d / M;
  const float* cl = coarse + list_no * d;
  double term2 = 0.0;
  for (int64_t c = 0; c < d; ++c) {
    const double t = (double)x[c] - (double)cl[c];
    term2 += t * t;
  }
  for (int64_t i = 0; i < n; ++i) {
    double term1 = 0.0, term3 = 0.0;
    for (int64_t m = 0; m < M; ++m) {
      const float* cw = pq + (m * 256 + codes[i * M + m]) * dsub;
      for (int64_t c = 0; c < dsub; ++c) {
        const double q2 = (double)cw[c];
        term1 += q2 * q2 + 2.0 * (double)cl[m * dsub + c] * q2;
        term3 += (double)x[m * dsub + c] * q2;
      }
    }
    out[i] = term1 + term2 - 2.0 * term3;
  }
}

// ---------------------------------------------------------------------------
// Appendix, Eq. (13) and P:L575-577: count the elements of a sequence that are
// in the min-k of their own prefix ("successive min-k").  On a random
// permutation its expectation is k + k (H_l - H_k).  Used only as a pin of the
// analysis, not by any result.
// ---------------------------------------------------------------------------
int64_t orc_successive_mink_count(const float* a, int64_t n, int64_t k) {
  std::vector<float> heap;  // max-heap of the k smallest so far
  int64_t count = 0;
  for (int64_t i = 0; i < n; ++i) {
    if ((int64_t)heap.size() < k) {
      heap.push_back(a[i]);
      std::push_heap(heap.begin(), heap.end());
      ++count;
    } else if (a[i] < heap.front()) {
      std::pop_heap(heap.begin(), heap.end());
      heap.back() = a[i];
      std::push_heap(heap.begin(), heap.end());
      ++count;
    }
  }
  return count;
}

// ---------------------------------------------------------------------------
// One Lloyd iteration of k-means (section 6.2: "k-means ... the assignment
// is a k = 1 exact search").  The paper fixes nothing else; the library's stated rules
// (include/fs.h, fs_kmeans) are restated here: assignment = nearest centroid by the direct
// squared distance in double, ties to the lower centroid; new centroid = mean of its points
// (double, rounded to fp32 once); an EMPTY cluster c at iteration `iter` takes the point
// mix(mix(seed + 0x9E3779B97F4A7C15 (iter + 1)) + c) mod n, mix = the splitmix64 finaliser.
// margin (may be NULL): (d_second - d_best) / d_second of every point's assignment.
// ---------------------------------------------------------------------------
static inline uint64_t orc_mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

void orc_kmeans_step(const float* x, int64_t n, int64_t d, const float* cent_in, int64_t K, uint64_t seed,
                     int64_t iter, float* cent_out, int64_t* assign_out, double* margin_out) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n; ++i) {
    double best = std::numeric_limits<double>::infinity(), second = best;
    int64_t bc = -1;
    for (int64_t c = 0; c < K; ++c) {
      const double dist = l2_direct(x + i * d, cent_in + c * d, d);
      if (dist < best) {
        second = best;
        best = dist;
        bc = c;
      } else if (dist < second) {
        second = dist;
      }
    }
    assign_out[i] = bc;
    if (margin_out) margin_out[i] = (second - best) / std::max(second, 1e-300);
  }
  std::vector<double> sum((size_t)K * d, 0.0);
  std::vector<int64_t> cnt((size_t)K, 0);
  for (int64_t i = 0; i < n; ++i) {  // ascending point order
    const int64_t c = assign_out[i];
    ++cnt[c];
    for (int64_t j = 0; j < d; ++j) sum[c * d + j] += (double)x[i * d + j];
  }
  for (int64_t c = 0; c < K; ++c) {
    if (cnt[c] > 0) {
      for (int64_t j = 0; j < d; ++j) cent_out[c * d + j] = (float)(sum[c * d + j] / (double)cnt[c]);
    } else {
      const uint64_t src =
          orc_mix64(orc_mix64(seed + 0x9E3779B97F4A7C15ull * (uint64_t)(iter + 1)) + (uint64_t)c) % (uint64_t)n;
      for (int64_t j = 0; j < d; ++j) cent_out[c * d + j] = x[src * d + j];
    }
  }
}

}  // extern "C"
