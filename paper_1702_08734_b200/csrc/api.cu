// api.cu -- error string, version, launch accounting (include/fs.h, top part).
#include <cstdarg>

#include "common.cuh"

namespace fs {

std::string& last_error() {
  thread_local std::string s;
  return s;
}
int64_t& launch_counter() {
  thread_local int64_t c = 0;
  return c;
}
int set_error(int code, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  last_error() = buf;
  return code;
}
int sm_count() {  // SMs of the CURRENT device (cached per device)
  static int cache[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 148;
  if (dev >= 0 && dev < 64 && cache[dev] > 0) return cache[dev];
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
  if (dev >= 0 && dev < 64) cache[dev] = n;
  return n;
}

int TempWs::acquire(void* ws, size_t ws_bytes, size_t need, cudaStream_t s) {
  stream = s;
  if (need == 0) need = 16;
  if (ws != nullptr) {
    if (ws_bytes < need)
      return set_error(FS_ENOMEM, "workspace too small: %zu bytes given, %zu needed", ws_bytes, need);
    ptr = ws;
    owned = false;
    return FS_OK;
  }
  cudaError_t e = cudaMallocAsync(&ptr, need, s);
  if (e != cudaSuccess) {
    ptr = nullptr;
    return set_error(FS_ENOMEM, "cudaMallocAsync(%zu) failed: %s", need, cudaGetErrorString(e));
  }
  owned = true;
  return FS_OK;
}
TempWs::~TempWs() {
  if (owned && ptr) cudaFreeAsync(ptr, stream);
}

}  // namespace fs

extern "C" {
const char* fs_last_error(void) { return fs::last_error().c_str(); }
const char* fs_version(void) { return "fs 0.1 (sm_100a)"; }
int64_t fs_launch_count(void) { return fs::launch_counter(); }
void fs_reset_launch_count(void) { fs::launch_counter() = 0; }
}
