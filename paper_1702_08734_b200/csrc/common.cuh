// common.cuh -- error handling, launch accounting and small helpers shared by
// the kernels of libfs.so (product path; shares nothing with oracle/).
#pragma once

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <string>

#include "../../include/fs.h"

namespace fs {

constexpr int kWarp = 32;
constexpr unsigned kFull = 0xffffffffu;

// thread-local state behind fs_last_error / fs_launch_count (api.cu)
std::string& last_error();
int64_t& launch_counter();
int set_error(int code, const char* fmt, ...);
int sm_count();  // SMs of the current device (cached)

#define FS_CUDA(call)                                                                  \
  do {                                                                                 \
    cudaError_t e_ = (call);                                                           \
    if (e_ != cudaSuccess)                                                             \
      return ::fs::set_error(FS_ECUDA, "%s failed: %s (%s:%d)", #call,                 \
                             cudaGetErrorString(e_), __FILE__, __LINE__);              \
  } while (0)

// Count a kernel launch and check it was accepted.
#define FS_LAUNCHED()                                                                  \
  do {                                                                                 \
    ++::fs::launch_counter();                                                          \
    cudaError_t e_ = cudaGetLastError();                                               \
    if (e_ != cudaSuccess)                                                             \
      return ::fs::set_error(FS_ECUDA, "kernel launch failed: %s (%s:%d)",             \
                             cudaGetErrorString(e_), __FILE__, __LINE__);              \
  } while (0)

static inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }
static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Stream-ordered temporary used when the caller passes ws == NULL.
struct TempWs {
  void* ptr = nullptr;
  cudaStream_t stream = nullptr;
  bool owned = false;
  int acquire(void* ws, size_t ws_bytes, size_t need, cudaStream_t s);
  ~TempWs();
};

}  // namespace fs
