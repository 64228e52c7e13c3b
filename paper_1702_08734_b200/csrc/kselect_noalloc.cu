// kselect_noalloc.cu -- fs_kselect_noalloc: fs_kselect for callers that may not allocate (code under
// CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// The k-selection kernels need scratch memory: the row counter of the persistent CTAs, and for few long
// rows (A4) the sampled bound, the survivor count and the survivor lists; for k = 1 on few long
// rows the chunk minima.  fs_kselect takes it from the caller or from a stream-ordered temporary.  Here
// it is a file-scope __device__ array of FS_NOALLOC_SCRATCH_BYTES that every GPU which loads the
// library holds until the process exits; this entry point calls no cudaMalloc / cudaFree / allocating
// routine and rejects calls whose scratch need (fs_kselect_ws_bytes) is larger than the array.
//
// The array is shared by every call and keeps the last call's contents: the launch path clears the
// words that must start at zero (row counter, bounds, survivor counts) on the caller's stream before
// the kernels run, so calls in stream order are independent of what ran before; calls that overlap on
// the GPU (different streams, different host threads) race on it and must be serialised by the caller.
#include <mutex>

#include "common.cuh"

namespace fs {

// kselect.cu
size_t kselect_ws_bytes(int64_t n_rows, int64_t n, int k);
int kselect_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                   int32_t* out_idx, void* ws, cudaStream_t s, bool largest);

namespace {

static __device__ __align__(256) unsigned char g_noalloc_scratch[FS_NOALLOC_SCRATCH_BYTES];

// Device address of the array on the CURRENT device.  In host code the array's name is only a
// stand-in for the symbol, not a device address: the address comes from cudaGetSymbolAddress, asked
// once per device with that device current.
int scratch_address(void** out) {
  static std::mutex mu;
  static void* addr[64] = {};
  int dev = 0;
  FS_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return set_error(FS_EUNSUPPORTED, "fs_kselect_noalloc: device ordinal %d >= 64", dev);
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    FS_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return set_error(FS_ECUDA, "fs_kselect_noalloc: cudaGetSymbolAddress returned NULL");
    addr[dev] = p;
  }
  *out = addr[dev];
  return FS_OK;
}

}  // namespace
}  // namespace fs

extern "C" {

size_t fs_kselect_noalloc_max_scratch(void) { return (size_t)FS_NOALLOC_SCRATCH_BYTES; }

int fs_kselect_noalloc(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                       int32_t* out_idx, fs_stream stream) {
  if (n_rows < 0 || n < 0 || ld < n) return fs::set_error(FS_EINVAL, "fs_kselect_noalloc: need n_rows >= 0, 0 <= n <= ld");
  if (k < 1) return fs::set_error(FS_EINVAL, "fs_kselect_noalloc: k must be >= 1");
  if (k > FS_MAX_K) return fs::set_error(FS_EUNSUPPORTED, "fs_kselect_noalloc: k = %d > %d", k, FS_MAX_K);
  if (n >= (1LL << 31)) return fs::set_error(FS_EUNSUPPORTED, "fs_kselect_noalloc: n must be < 2^31");
  if (n_rows > 0 && (!out_val || !out_idx || (n > 0 && !rows)))
    return fs::set_error(FS_EINVAL, "fs_kselect_noalloc: NULL pointer");
  if (n_rows == 0) return FS_OK;
  const size_t need = fs::kselect_ws_bytes(n_rows, n, k);
  if (need > (size_t)FS_NOALLOC_SCRATCH_BYTES)
    return fs::set_error(FS_EUNSUPPORTED,
                         "fs_kselect_noalloc: this call needs %zu bytes of scratch, the built-in array holds %zu "
                         "(FS_NOALLOC_SCRATCH_BYTES); use fs_kselect with a caller workspace",
                         need, (size_t)FS_NOALLOC_SCRATCH_BYTES);
  void* ws = nullptr;
  const int rc = fs::scratch_address(&ws);
  if (rc != FS_OK) return rc;
  return fs::kselect_device(rows, n_rows, n, ld, k, out_val, out_idx, ws, static_cast<cudaStream_t>(stream), false);
}

}  // extern "C"
