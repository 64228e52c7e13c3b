// ivfpq_train.cu -- fs_ivfpq_train: k-means training of the coarse quantizer q1
// and of the residual product quantizer q2 ("trained via k-means", P:L90;
// assignment = exact search with k = 1).
//
// Off the parity path (reading C-11): the oracle and the library share
// the resulting arrays through fs_ivfpq_get_quantizers.  The paper leaves the
// initialisation and empty clusters unspecified; here: initial centroids are
// evenly strided input points, Lloyd iterations assign with the k = 1 exact
// search (flat.cu) and accumulate the means with float atomics, and an empty
// cluster is re-seeded from a hashed input point.
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

__global__ void km_accumulate_kernel(const float* __restrict__ x, int64_t n, int d,
                                     const int64_t* __restrict__ assign, float* __restrict__ sums,
                                     unsigned int* __restrict__ counts) {
  const int lane = threadIdx.x & 31;
  const int64_t v = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (v >= n) return;
  const int64_t c = assign[v];
  for (int j = lane; j < d; j += 32) atomicAdd(&sums[c * d + j], x[v * d + j]);
  if (lane == 0) atomicAdd(&counts[c], 1u);
}

__device__ __forceinline__ uint64_t km_mix(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

__global__ void km_update_kernel(const float* __restrict__ x, int64_t n, int d, int K,
                                 const float* __restrict__ sums,
                                 const unsigned int* __restrict__ counts, uint64_t seed, int iter,
                                 float* __restrict__ cent) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (int64_t)K * d) return;
  const int64_t c = e / d;
  const int j = (int)(e - c * d);
  const unsigned int cnt = counts[c];
  if (cnt > 0) {
    cent[e] = sums[e] / (float)cnt;
  } else {
    const uint64_t src = km_mix(km_mix(seed + 0x9E3779B97F4A7C15ull * (uint64_t)(iter + 1)) + (uint64_t)c) % (uint64_t)n;
    cent[e] = x[src * d + j];
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
                  cudaStream_t s) {
  if (n < K) return set_error(FS_EINVAL, "k-means: %lld points for %d centroids", (long long)n, K);
  DevBuf sums, counts, assign, cnorm;
  int rc;
  auto done = [&](int r) {
    cudaStreamSynchronize(s);
    sums.release();
    counts.release();
    assign.release();
    cnorm.release();
    return r;
  };
  const int64_t kd = (int64_t)K * d;
  if ((rc = sums.ensure((size_t)kd * sizeof(float), 0, s)) != FS_OK ||
      (rc = counts.ensure((size_t)K * sizeof(unsigned int), 0, s)) != FS_OK ||
      (rc = assign.ensure((size_t)n * sizeof(int64_t), 0, s)) != FS_OK ||
      (rc = cnorm.ensure((size_t)K * sizeof(float), 0, s)) != FS_OK)
    return done(rc);
  km_init_kernel<<<(unsigned)ceil_div(kd, 256), 256, 0, s>>>(x, n, d, K, cent);
  ++launch_counter();
  for (int it = 0; it < niter; ++it) {
    if ((rc = launch_row_norms(cent, K, d, cnorm.as<float>(), s)) != FS_OK) return done(rc);
    if ((rc = assign_nearest(x, n, cent, cnorm.as<float>(), K, d, assign.as<int64_t>(), s)) != FS_OK)
      return done(rc);
    cudaMemsetAsync(sums.p, 0, (size_t)kd * sizeof(float), s);
    cudaMemsetAsync(counts.p, 0, (size_t)K * sizeof(unsigned int), s);
    km_accumulate_kernel<<<(unsigned)ceil_div(n, 8), 256, 0, s>>>(x, n, d, assign.as<int64_t>(),
                                                                 sums.as<float>(),
                                                                 counts.as<unsigned int>());
    km_update_kernel<<<(unsigned)ceil_div(kd, 256), 256, 0, s>>>(
        x, n, d, K, sums.as<float>(), counts.as<unsigned int>(), seed, it, cent);
    launch_counter() += 2;
  }
  cudaError_t e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return done(set_error(FS_ECUDA, "k-means failed: %s", cudaGetErrorString(e)));
  return done(FS_OK);
}

}  // namespace fs

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
  if ((rc = launch_row_norms(ix->coarse.as<float>(), ix->nlist, d, ix->cnorm.as<float>(), s)) != FS_OK)
    return rc;
  DevBuf assign, sub;
  if ((rc = assign.ensure((size_t)n * sizeof(int64_t), 0, s)) != FS_OK) return rc;
  if ((rc = sub.ensure((size_t)n * dsub * sizeof(float), 0, s)) != FS_OK) {
    assign.release();
    return rc;
  }
  rc = assign_nearest(x, n, ix->coarse.as<float>(), ix->cnorm.as<float>(), ix->nlist, d,
                      assign.as<int64_t>(), s);
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
