// kselect.cu -- fs_kselect: batched k-selection: entry points, the k = 1
// reduction (A5) and the host-buffer variant.  k >= 2 lives in kselect_row.cu.
//
//   A5 k = 1   kselect_k1_kernel: min / argmin reduction on packed (value, index) keys, one warp per
//              (row, chunk), plain streaming 128-bit loads ("a parallel reduction is used
//              for the k = 1 case, not WarpSelect").  Few long rows are cut into P chunks
//              whose minima kselect_k1_final_kernel reduces again.
#include <cstdlib>
#include <mutex>

#include "common.cuh"
#include "select.cuh"

namespace fs {

struct K1Args {
  const float* vals;  // [n_rows][ld]
  int64_t n_rows, n, ld;
  int P;              // chunks per row
  int64_t chunk;      // elements per chunk (multiple of 4)
  float* out_val;     // P == 1: [n_rows]
  int32_t* out_idx;
  uint64_t* out_keys;  // P > 1: [n_rows][P] chunk minima as keys
  int largest;         // 1: arg max (the kernels reduce -v)
};

__device__ __forceinline__ float4 ld_stream4(const float* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
               : "l"(p));
  return r;
}

template <int WARPS, bool LG>
__global__ void __launch_bounds__(WARPS * 32) kselect_k1_kernel(const K1Args a) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t item = (int64_t)blockIdx.x * WARPS + warp;
  if (item >= a.n_rows * a.P) return;
  const int64_t row = item / a.P;
  const int c = (int)(item - row * a.P);
  const int64_t start = (int64_t)c * a.chunk;
  int64_t len = a.n - start;
  if (len > a.chunk) len = a.chunk;
  if (len < 0) len = 0;
  const float* p = a.vals + row * a.ld + start;
  const uint32_t base = (uint32_t)start;
  int64_t head = (4 - (int)(((uintptr_t)p >> 2) & 3)) & 3;  // scalars before the 16-byte aligned body
  if (head > len) head = len;
  const int64_t nvec = (len - head) >> 2;
  uint64_t best = kSentinelKey;
  if (lane < head) best = umin64(best, make_key(LG ? -p[lane] : p[lane], base + lane));
  const float* pv = p + head;
  const uint32_t vbase = base + (uint32_t)head;
  // Per lane a running float minimum decides whether the exact key compare is
  // needed at all: "!(v > m)" is true for v <= m and for NaN.
  float m = __uint_as_float(0x7FFFFFFFu);
  auto take = [&](float raw, uint32_t idx) {
    const float v = LG ? -raw : raw;  // arg max = arg min of the negated values, ties still to the lower index
    if (!(v > m)) {
      const uint64_t key = make_key(v, idx);
      if (key < best) {
        best = key;
        m = key_val(key);
      }
    }
  };
  constexpr int U = 4;
  int64_t v0 = 0;
  for (; v0 + U * 32 <= nvec; v0 += U * 32) {
    float4 x[U];
#pragma unroll
    for (int u = 0; u < U; ++u) x[u] = ld_stream4(pv + ((v0 + u * 32 + lane) << 2));
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const uint32_t i0 = vbase + (uint32_t)((v0 + u * 32 + lane) << 2);
      take(x[u].x, i0);
      take(x[u].y, i0 + 1);
      take(x[u].z, i0 + 2);
      take(x[u].w, i0 + 3);
    }
  }
  for (int64_t v = v0 + lane; v < nvec; v += 32) {
    const float4 x = ld_stream4(pv + (v << 2));
    const uint32_t i0 = vbase + (uint32_t)(v << 2);
    take(x.x, i0);
    take(x.y, i0 + 1);
    take(x.z, i0 + 2);
    take(x.w, i0 + 3);
  }
  const int64_t done = head + (nvec << 2);
  if (done + lane < len) take(p[done + lane], base + (uint32_t)(done + lane));
#pragma unroll
  for (int s = 16; s >= 1; s >>= 1) best = umin64(best, shfl_xor64(best, s));
  if (lane == 0) {
    if (a.P > 1) {
      a.out_keys[item] = best;
    } else if (best == kSentinelKey) {
      a.out_val[item] = __uint_as_float(LG ? 0xFF800000u : 0x7F800000u);
      a.out_idx[item] = -1;
    } else {
      const uint32_t idx = key_idx(best);
      a.out_val[item] = a.vals[row * a.ld + idx];
      a.out_idx[item] = (int32_t)idx;
    }
  }
}

// The minimum of a row's P chunk minima: one warp per row.
__global__ void __launch_bounds__(128) kselect_k1_final_kernel(const uint64_t* __restrict__ keys, int64_t n_rows, int P,
                                                                const float* __restrict__ rows, int64_t ld,
                                                                float* __restrict__ out_val, int32_t* __restrict__ out_idx,
                                                                int largest) {
  const int lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (row >= n_rows) return;
  uint64_t best = kSentinelKey;
  for (int i = lane; i < P; i += 32) best = umin64(best, keys[row * P + i]);
#pragma unroll
  for (int s = 16; s >= 1; s >>= 1) best = umin64(best, shfl_xor64(best, s));
  if (lane == 0) {
    if (best == kSentinelKey) {
      out_val[row] = __uint_as_float(largest ? 0xFF800000u : 0x7F800000u);
      out_idx[row] = -1;
    } else {
      const uint32_t idx = key_idx(best);
      out_val[row] = rows[row * ld + idx];  // original bits (+-0, NaN payload)
      out_idx[row] = (int32_t)idx;
    }
  }
}

// ---------------------------------------------------------------------------
// Host side: plan of the k = 1 call and launches.
// ---------------------------------------------------------------------------
namespace {

constexpr int kWarpsPerCtaK1 = 4;

struct Plan {
  int P;          // chunks per row
  int64_t chunk;  // elements per chunk (multiple of 4)
  size_t bytes;   // workspace: [n_rows][P] keys when P > 1
};

// Rows are cut into chunks only when there are too few rows to occupy the GPU (16 warps per SM), and
// never below 4 096 elements per chunk.
Plan make_plan(int64_t n_rows, int64_t n) {
  Plan p;
  const int64_t resident = (int64_t)sm_count() * 16;
  const int64_t min_chunk = 4096;
  int64_t P = 1;
  if (n_rows > 0 && n_rows * 2 <= resident && n >= 2 * min_chunk) {
    P = resident / n_rows;
    const int64_t pmax = n / min_chunk;
    if (P > pmax) P = pmax;
    if (P < 1) P = 1;
  }
  int64_t chunk = ceil_div(n > 0 ? n : 1, P);
  chunk = (chunk + 3) / 4 * 4;
  P = n > 0 ? ceil_div(n, chunk) : 1;
  p.P = (int)P;
  p.chunk = chunk;
  p.bytes = P > 1 ? align_up((size_t)n_rows * P * sizeof(uint64_t), 256) : 16;
  return p;
}

int validate(const void* rows, int64_t n_rows, int64_t n, int64_t ld, int k, const void* ov,
             const void* oi) {
  if (n_rows < 0 || n < 0 || ld < n) return set_error(FS_EINVAL, "fs_kselect: need n_rows >= 0, 0 <= n <= ld");
  if (k < 1) return set_error(FS_EINVAL, "fs_kselect: k must be >= 1");
  if (k > FS_MAX_K) return set_error(FS_EUNSUPPORTED, "fs_kselect: k = %d > %d", k, FS_MAX_K);
  if (n >= (1LL << 31)) return set_error(FS_EUNSUPPORTED, "fs_kselect: n must be < 2^31");
  if (n_rows > 0 && (!ov || !oi || (n > 0 && !rows)))
    return set_error(FS_EINVAL, "fs_kselect: NULL pointer");
  return FS_OK;
}

}  // namespace

// Device staging of the host entry point: one grow-only allocation, three streams, events per slice.
struct HostStage {
  void* p = nullptr;
  size_t bytes = 0;
  cudaStream_t s_in = nullptr, s_run = nullptr, s_out = nullptr;
  cudaEvent_t ev_in[8] = {}, ev_run[8] = {};
  int ensure(size_t need) {
    if (!s_in) {
      if (cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking) != cudaSuccess ||
          cudaStreamCreateWithFlags(&s_run, cudaStreamNonBlocking) != cudaSuccess ||
          cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking) != cudaSuccess)
        return set_error(FS_ECUDA, "fs_kselect_host: cudaStreamCreate failed");
      for (int i = 0; i < 8; ++i)
        if (cudaEventCreateWithFlags(&ev_in[i], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ev_run[i], cudaEventDisableTiming) != cudaSuccess)
          return set_error(FS_ECUDA, "fs_kselect_host: cudaEventCreate failed");
    }
    if (need > bytes) {
      if (p) cudaFree(p);
      p = nullptr;
      bytes = 0;
      const cudaError_t e = cudaMalloc(&p, need);
      if (e != cudaSuccess) return set_error(FS_ECUDA, "fs_kselect_host: cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e));
      bytes = need;
    }
    return FS_OK;
  }
};

// kselect_row.cu: k >= 2
size_t kselect_rows_ws_bytes(int64_t n_rows, int64_t n, int k);
int kselect_rows_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                        int32_t* out_idx, void* ws, cudaStream_t s, bool largest);

// Selection over device rows; also used by the flat and IVFPQ drivers.
size_t kselect_ws_bytes(int64_t n_rows, int64_t n, int k) {
  return k >= 2 ? kselect_rows_ws_bytes(n_rows, n, k) : make_plan(n_rows, n).bytes;
}

int kselect_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                   int32_t* out_idx, void* ws, cudaStream_t s, bool largest) {
  if (k >= 2) return kselect_rows_device(rows, n_rows, n, ld, k, out_val, out_idx, ws, s, largest);
  const Plan p = make_plan(n_rows, n);
  K1Args a;
  a.vals = rows;
  a.n_rows = n_rows;
  a.n = n;
  a.ld = ld;
  a.P = p.P;
  a.chunk = p.chunk;
  a.out_val = out_val;
  a.out_idx = out_idx;
  a.out_keys = p.P > 1 ? reinterpret_cast<uint64_t*>(ws) : nullptr;
  a.largest = largest ? 1 : 0;
  const int64_t items = n_rows * p.P;
  if (items == 0) return FS_OK;
  const int64_t grid = ceil_div(items, kWarpsPerCtaK1);
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "too many rows for one launch");
  if (largest)
    kselect_k1_kernel<kWarpsPerCtaK1, true><<<(unsigned)grid, kWarpsPerCtaK1 * 32, 0, s>>>(a);
  else
    kselect_k1_kernel<kWarpsPerCtaK1, false><<<(unsigned)grid, kWarpsPerCtaK1 * 32, 0, s>>>(a);
  FS_LAUNCHED();
  if (p.P > 1) {
    kselect_k1_final_kernel<<<(unsigned)ceil_div(n_rows, 4), 128, 0, s>>>(a.out_keys, n_rows, p.P, rows, ld, out_val,
                                                                        out_idx, a.largest);
    FS_LAUNCHED();
  }
  return FS_OK;
}

}  // namespace fs

extern "C" {

size_t fs_kselect_ws_bytes(int64_t n_rows, int64_t n, int k) {
  if (n_rows < 0 || n < 0 || k < 1 || k > FS_MAX_K) return 0;
  return fs::kselect_ws_bytes(n_rows, n, k);
}

static int kselect_entry(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                         int32_t* out_idx, void* ws, size_t ws_bytes, fs_stream stream, bool largest) {
  int rc = fs::validate(rows, n_rows, n, ld, k, out_val, out_idx);
  if (rc != FS_OK) return rc;
  if (n_rows == 0) return FS_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  fs::TempWs t;
  rc = t.acquire(ws, ws_bytes, fs::kselect_ws_bytes(n_rows, n, k), s);
  if (rc != FS_OK) return rc;
  return fs::kselect_device(rows, n_rows, n, ld, k, out_val, out_idx, t.ptr, s, largest);
}

int fs_kselect(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
               int32_t* out_idx, void* ws, size_t ws_bytes, fs_stream stream) {
  return kselect_entry(rows, n_rows, n, ld, k, out_val, out_idx, ws, ws_bytes, stream, false);
}

int fs_kselect_largest(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                       int32_t* out_idx, void* ws, size_t ws_bytes, fs_stream stream) {
  return kselect_entry(rows, n_rows, n, ld, k, out_val, out_idx, ws, ws_bytes, stream, true);
}

int fs_kselect_host(const float* rows_host, int64_t n_rows, int64_t n, int64_t ld, int k,
                    float* out_val_host, int32_t* out_idx_host) {
  int rc = fs::validate(rows_host, n_rows, n, ld, k, out_val_host, out_idx_host);
  if (rc != FS_OK) return rc;
  if (n_rows == 0) return FS_OK;
  // Rows go through in up to 8 slices on three streams: slice c + 1 is copied in while slice c is
  // selected and slice c - 1 is copied out (PCIe is full duplex).  Device staging comes from a
  // grow-only arena that lives as long as the library (no cudaMalloc / cudaFree per call).
  static std::mutex mu;
  std::lock_guard<std::mutex> lock(mu);
  static fs::HostStage st;
  const int64_t n_slices = n_rows < 8 ? n_rows : 8;
  const int64_t per = (n_rows + n_slices - 1) / n_slices;
  const size_t in_b = (size_t)n_rows * ld * sizeof(float), out_n = (size_t)n_rows * k;
  size_t ws_b = 0;
  for (int64_t r0 = 0; r0 < n_rows; r0 += per) {
    const size_t b = fs::kselect_ws_bytes(n_rows - r0 < per ? n_rows - r0 : per, n, k);
    ws_b = b > ws_b ? b : ws_b;
  }
  const size_t o_rows = 0, o_val = fs::align_up(in_b, 256), o_idx = o_val + fs::align_up(out_n * sizeof(float), 256),
               o_ws = o_idx + fs::align_up(out_n * sizeof(int32_t), 256), total = o_ws + fs::align_up(ws_b, 256);
  if ((rc = st.ensure(total)) != FS_OK) return rc;
  char* base = static_cast<char*>(st.p);
  float* d_rows = reinterpret_cast<float*>(base + o_rows);
  float* d_val = reinterpret_cast<float*>(base + o_val);
  int32_t* d_idx = reinterpret_cast<int32_t*>(base + o_idx);
  cudaError_t e = cudaSuccess;
  auto ck = [&](cudaError_t err, const char* what) {
    if (err != cudaSuccess && rc == FS_OK) rc = fs::set_error(FS_ECUDA, "%s failed: %s", what, cudaGetErrorString(err));
    return err == cudaSuccess;
  };
  int slice = 0;
  for (int64_t r0 = 0; r0 < n_rows && rc == FS_OK; r0 += per, ++slice) {
    const int64_t nr = n_rows - r0 < per ? n_rows - r0 : per;
    if (!ck(cudaMemcpyAsync(d_rows + r0 * ld, rows_host + r0 * ld, (size_t)nr * ld * sizeof(float),
                            cudaMemcpyHostToDevice, st.s_in), "cudaMemcpyAsync H2D")) break;
    if (!ck(cudaEventRecord(st.ev_in[slice], st.s_in), "cudaEventRecord")) break;
    if (!ck(cudaStreamWaitEvent(st.s_run, st.ev_in[slice], 0), "cudaStreamWaitEvent")) break;
    rc = fs::kselect_device(d_rows + r0 * ld, nr, n, ld, k, d_val + r0 * k, d_idx + r0 * k, base + o_ws, st.s_run, false);
    if (rc != FS_OK) break;
    if (!ck(cudaEventRecord(st.ev_run[slice], st.s_run), "cudaEventRecord")) break;
    if (!ck(cudaStreamWaitEvent(st.s_out, st.ev_run[slice], 0), "cudaStreamWaitEvent")) break;
    if (!ck(cudaMemcpyAsync(out_val_host + r0 * k, d_val + r0 * k, (size_t)nr * k * sizeof(float),
                            cudaMemcpyDeviceToHost, st.s_out), "cudaMemcpyAsync D2H")) break;
    if (!ck(cudaMemcpyAsync(out_idx_host + r0 * k, d_idx + r0 * k, (size_t)nr * k * sizeof(int32_t),
                            cudaMemcpyDeviceToHost, st.s_out), "cudaMemcpyAsync D2H")) break;
  }
  e = cudaStreamSynchronize(st.s_in);
  ck(e, "cudaStreamSynchronize");
  e = cudaStreamSynchronize(st.s_run);
  ck(e, "cudaStreamSynchronize");
  e = cudaStreamSynchronize(st.s_out);
  ck(e, "cudaStreamSynchronize");
  return rc;
}

}  // extern "C"
