// ivfpq_train.cu -- Lloyd's k-means (fs_kmeans) and fs_ivfpq_train: training of the coarse quantizer
// q1 and of the residual product quantizer q2 ("trained via k-means"; section 6.2,
// the assignment step is the exact search with k = 1, whose selection is fused into the
// distance tiles -- flat_tc.cu -- so no n x K matrix is written).
//
// The paper leaves the initialisation and empty clusters unspecified (reading C-11); here:
//   init       centroid c = input point floor(c n / K) (evenly strided, distinct for n >= K)
//   assignment nearest centroid by the k = 1 exact search, ties to the lower centroid
//   update     DETERMINISTIC: the points are grouped by cluster with the stable radix sort of the
//              inverted-list builder, and one warp per cluster adds its points in ascending index order
//              in double precision (no float atomics: the same input gives the same quantizers bit for
//              bit, and the means match a double-precision reference to fp32 rounding)
//   empty      cluster c at iteration it is re-seeded from point
//              mix(mix(seed + 0x9E3779B97F4A7C15 (it + 1)) + c) mod n   (mix = the splitmix64 finaliser)
// oracle/oracle.cpp restates one step of this (orc_kmeans_step) for the parity test.
#include "flat.cuh"
#include "ivfpq.cuh"

namespace fs {

namespace {

__global__ void km_init_kernel(const float* __restrict__ x, int64_t n, int d, int K,
                               float* __restrict__ cent) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (int64_t)K * d) return;
  const int64_t c = e / d;
  const int j = (int)(e - c * d);
  const int64_t src = (c * n) / K;  // distinct for n >= K
  cent[e] = x[src * d + j];
}

__global__ void km_keys_kernel(const int64_t* __restrict__ assign, int64_t n, uint32_t* __restrict__ keys) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) keys[i] = (uint32_t)assign[i];
}

// first[c] = position of cluster c's first point in the sorted order (first[K] = n)
__global__ void km_bounds_kernel(const uint32_t* __restrict__ keys_sorted, int64_t n, int K, int64_t* __restrict__ first) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int64_t k1 = keys_sorted[p];
  const int64_t k0 = p > 0 ? (int64_t)keys_sorted[p - 1] : -1;
  for (int64_t c = k0 + 1; c <= k1; ++c) first[c] = p;
  if (p == n - 1)
    for (int64_t c = k1 + 1; c <= K; ++c) first[c] = n;
}

__device__ __forceinline__ uint64_t km_mix(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// One warp per cluster: the mean of its points (ascending point index, double accumulation), or the
// re-seed point when the cluster is empty.
__global__ void __launch_bounds__(256)
    km_update_kernel(const float* __restrict__ x, int64_t n, int d, int K, const uint32_t* __restrict__ order,
                     const int64_t* __restrict__ first, uint64_t seed, int iter, float* __restrict__ cent) {
  const int lane = threadIdx.x & 31;
  const int64_t c = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (c >= K) return;
  const int64_t b = first[c], e = first[c + 1];
  if (e == b) {
    const uint64_t src = km_mix(km_mix(seed + 0x9E3779B97F4A7C15ull * (uint64_t)(iter + 1)) + (uint64_t)c) % (uint64_t)n;
    for (int j = lane; j < d; j += 32) cent[c * d + j] = x[src * d + j];
    return;
  }
  const double inv = 1.0 / (double)(e - b);
  for (int j0 = 0; j0 < d; j0 += 32) {
    const int j = j0 + lane;
    double acc = 0.0;
    if (j < d)
      for (int64_t p = b; p < e; ++p) acc += (double)x[(int64_t)order[p] * d + j];
    if (j < d) cent[c * d + j] = (float)(acc * inv);
  }
}

__global__ void residual_kernel(const float* __restrict__ x, int64_t n, int d,
                                const float* __restrict__ cent, const int64_t* __restrict__ assign,
                                int j0, int dsub, float* __restrict__ out /*[n][dsub]*/) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n * dsub) return;
  const int64_t v = e / dsub;
  const int j = (int)(e - v * dsub);
  out[e] = x[v * d + j0 + j] - cent[assign[v] * d + j0 + j];
}

}  // namespace

int kmeans_device(const float* x, int64_t n, int d, int K, int niter, uint64_t seed, float* cent,
                  cudaStream_t s, bool init, int64_t* assign_out) {
  if (n < K) return set_error(FS_EINVAL, "k-means: %lld points for %d centroids", (long long)n, K);
  if (n >= (1LL << 32)) return set_error(FS_EUNSUPPORTED, "k-means: more than 2^32-1 points");
  DevBuf sortws, first, assign, cnorm;
  int rc;
  auto done = [&](int r) {
    cudaStreamSynchronize(s);
    sortws.release();
    first.release();
    assign.release();
    cnorm.release();
    return r;
  };
  const int64_t kd = (int64_t)K * d;
  if ((rc = sortws.ensure(stable_sort_ws(n), 0, s)) != FS_OK ||
      (rc = first.ensure((size_t)(K + 1) * sizeof(int64_t), 0, s)) != FS_OK ||
      (rc = assign.ensure((size_t)n * sizeof(int64_t), 0, s)) != FS_OK ||
      (rc = cnorm.ensure((size_t)K * sizeof(float), 0, s)) != FS_OK)
    return done(rc);
  if (init) {
    km_init_kernel<<<(unsigned)ceil_div(kd, 256), 256, 0, s>>>(x, n, d, K, cent);
    ++launch_counter();
  }
  int nbits = 0;
  while ((1LL << nbits) < K) ++nbits;
  for (int it = 0; it < niter; ++it) {
    if ((rc = launch_row_norms(cent, K, d, cnorm.as<float>(), s)) != FS_OK) return done(rc);
    if ((rc = assign_nearest(x, n, cent, cnorm.as<float>(), K, d, assign.as<int64_t>(), s)) != FS_OK)
      return done(rc);
    if (assign_out && it == niter - 1 &&
        cudaMemcpyAsync(assign_out, assign.p, (size_t)n * sizeof(int64_t), cudaMemcpyDeviceToDevice, s) != cudaSuccess)
      return done(set_error(FS_ECUDA, "fs_kmeans: copy of the assignments failed"));
    km_keys_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, s>>>(assign.as<int64_t>(), n, sortws.as<uint32_t>());
    ++launch_counter();
    const uint32_t *keys_sorted = nullptr, *order = nullptr;
    if ((rc = stable_sort_by_key(sortws.as<char>(), n, nbits, &keys_sorted, &order, s)) != FS_OK) return done(rc);
    km_bounds_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, s>>>(keys_sorted, n, K, first.as<int64_t>());
    km_update_kernel<<<(unsigned)ceil_div(K, 8), 256, 0, s>>>(x, n, d, K, order, first.as<int64_t>(), seed, it, cent);
    launch_counter() += 2;
  }
  cudaError_t e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return done(set_error(FS_ECUDA, "k-means failed: %s", cudaGetErrorString(e)));
  return done(FS_OK);
}

}  // namespace fs

extern "C" int fs_kmeans(const float* x, int64_t n, int d, int K, int niter, uint64_t seed, int init,
                         float* centroids, int64_t* assign, fs_stream stream) {
  using namespace fs;
  if (!x || !centroids) return set_error(FS_EINVAL, "fs_kmeans: NULL pointer");
  if (n < 1 || d < 1 || K < 1 || niter < 0) return set_error(FS_EINVAL, "fs_kmeans: need n, d, K >= 1 and niter >= 0");
  if (d > 2048) return set_error(FS_EUNSUPPORTED, "fs_kmeans: d > 2048");
  if (n < K) return set_error(FS_EINVAL, "fs_kmeans: fewer points than centroids");
  return kmeans_device(x, n, d, K, niter, seed, centroids, static_cast<cudaStream_t>(stream), init != 0, assign);
}

extern "C" int fs_ivfpq_train(fs_ivfpq* ix, const float* x, int64_t n, int niter, uint64_t seed,
                              fs_stream stream) {
  using namespace fs;
  if (!ix || !x) return set_error(FS_EINVAL, "fs_ivfpq_train: NULL pointer");
  if (niter < 0) return set_error(FS_EINVAL, "fs_ivfpq_train: niter < 0");
  if (ix->ntotal() > 0) return set_error(FS_ESTATE, "fs_ivfpq_train: index already holds vectors");
  if (n < ix->nlist || n < 256)
    return set_error(FS_EINVAL, "fs_ivfpq_train: need at least max(nlist, 256) training vectors");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int d = ix->d, M = ix->M, dsub = ix->dsub;
  int rc = kmeans_device(x, n, d, ix->nlist, niter, seed, ix->coarse.as<float>(), s);
  if (rc != FS_OK) return rc;
  if ((rc = ivfpq_prepare_coarse(ix, s)) != FS_OK) return rc;
  DevBuf assign, sub;
  if ((rc = assign.ensure((size_t)n * sizeof(int64_t), 0, s)) != FS_OK) return rc;
  if ((rc = sub.ensure((size_t)n * dsub * sizeof(float), 0, s)) != FS_OK) {
    assign.release();
    return rc;
  }
  rc = assign_nearest(x, n, ix->coarse.as<float>(), ix->cnorm.as<float>(), ix->nlist, d,
                      assign.as<int64_t>(), s, ix->cprep.p);
  for (int m = 0; m < M && rc == FS_OK; ++m) {
    residual_kernel<<<(unsigned)ceil_div(n * dsub, 256), 256, 0, s>>>(
        x, n, d, ix->coarse.as<float>(), assign.as<int64_t>(), m * dsub, dsub, sub.as<float>());
    ++launch_counter();
    rc = kmeans_device(sub.as<float>(), n, dsub, 256, niter, seed + 1 + m,
                       ix->pq.as<float>() + (size_t)m * 256 * dsub, s);
  }
  cudaStreamSynchronize(s);
  assign.release();
  sub.release();
  if (rc != FS_OK) return rc;
  ix->have_quantizers = true;
  return FS_OK;
}
