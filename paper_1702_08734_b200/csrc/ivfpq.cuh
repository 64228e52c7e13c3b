// ivfpq.cuh -- the IVFADC index object behind fs_ivfpq_* (include/fs.h) and the
// internal interfaces between its translation units:
//   ivfpq.cu        object life cycle, quantizers, add (D1-D3), export, C ABI
//   ivfpq_search.cu search (C1-C5): LUT + list scan + pass-1 selection, pass 2
//   ivfpq_train.cu  k-means training of both quantizers
#pragma once

#include <vector>

#include "common.cuh"

namespace fs {

// Device buffer owned by the index (cudaMalloc / cudaFree), grown geometrically.
struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
  // Make room for `bytes`, keeping the first `keep` bytes.  Synchronises `s`.
  int ensure(size_t bytes, size_t keep, cudaStream_t s);
  void release();
  template <typename T>
  T* as() const { return static_cast<T*>(p); }
};

}  // namespace fs

// The opaque object of include/fs.h.
struct fs_ivfpq {
  int d = 0, nlist = 0, M = 0, dsub = 0;
  bool have_quantizers = false;
  fs::DevBuf coarse;  // [nlist][d] fp32
  fs::DevBuf cnorm;   // [nlist] fp32: ||c||^2 (B1 of the coarse search, precomputed)
  fs::DevBuf cprep;   // the centroids as a prepared database of the exact search (flat.cuh FlatPrep: norms, lo flag,
                      // lo plane), written whenever the centroids are: C1 and D1 skip that pass on every call
  fs::DevBuf pq;      // [M][256][dsub] fp32
  // Finalised inverted file, CSR over list number (codes and
  // ids in separate arrays, each list contiguous, append order kept).
  int64_t n_csr = 0;
  fs::DevBuf offsets;  // int64 [nlist+1]
  fs::DevBuf codes;    // uint8 [n_csr][M]; M = 8 / 16: byte i of the vector at position p of its list holds
                       // sub-quantizer i ^ (p mod M) (the lane order of the conflict-free scan, see permuted())
  fs::DevBuf ids;      // int64 [n_csr]
  fs::DevBuf s1;       // float [n_csr]: Eq. 11 term 1 of the stored vector, ||q2||^2 + 2 <q1, q2>
  std::vector<int64_t> offsets_host;

  // Vectors added since the last finalise, in arrival order.
  int64_t n_staged = 0;
  fs::DevBuf st_list;   // uint32 [n_staged]
  fs::DevBuf st_codes;  // uint8 [n_staged][M]
  fs::DevBuf st_ids;    // int64 [n_staged]
  fs::DevBuf st_s1;     // float [n_staged]

  // Code bytes scanned by the last search (device counter, read lazily).
  fs::DevBuf scanned;  // unsigned long long [1]
  // Stage boundaries of the last search on its stream: start, after C1, after C2-C4, end.
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  bool ev_valid = false;

  int64_t ntotal() const { return n_csr + n_staged; }
  // CSR codes stored pre-permuted for the fixed-point scan (the per-vector byte permutation is done once,
  // when the lists are built, instead of once per scanned vector); export undoes it.
  bool permuted() const { return M == 8 || M == 16; }
};

namespace fs {

// Stable radix sort of 32-bit keys with their arrival indices (ivfpq.cu): the workspace t holds the keys
// in its first n words on entry; stable_sort_ws(n) bytes.
size_t stable_sort_ws(int64_t n);
int stable_sort_by_key(char* t, int64_t n, int nbits, const uint32_t** keys_sorted, const uint32_t** order,
                       cudaStream_t s);

// Group staged vectors into the CSR lists (stable: append order kept).
int ivfpq_finalise(fs_ivfpq* ix, cudaStream_t s);

// D2: residual PQ encoding of n vectors with known coarse assignment.
int launch_pq_encode(const fs_ivfpq* ix, const float* y, int64_t n, const int64_t* assign,
                     uint8_t* codes_out, uint32_t* list_out, float* s1_out, cudaStream_t s);

// Lloyd k-means on device data x [n][d] -> cent [K][d] (ivfpq_train.cu).  init: start from evenly strided
// input points (else from cent as given); assign_out (or NULL): the assignment the last update used.
int kmeans_device(const float* x, int64_t n, int d, int K, int niter, uint64_t seed, float* cent,
                  cudaStream_t s, bool init = true, int64_t* assign_out = nullptr);
// Nearest centroid of each x (k = 1 exact search, chunked): assign int64 [n].
int assign_nearest(const float* x, int64_t n, const float* cent, const float* cent_norm, int K,
                   int d, int64_t* assign, cudaStream_t s, const void* cent_prep = nullptr);
// ||c||^2 and the prepared block of the index's centroids (after every change of them)
int ivfpq_prepare_coarse(fs_ivfpq* ix, cudaStream_t s);

int ivfpq_search_device(fs_ivfpq* ix, const float* xq, int64_t nq, int nprobe, int k,
                        float* out_dist, int64_t* out_ids, int32_t* out_probed, void* ws,
                        cudaStream_t s);
size_t ivfpq_search_ws(const fs_ivfpq* ix, int64_t nq, int nprobe, int k);

}  // namespace fs
