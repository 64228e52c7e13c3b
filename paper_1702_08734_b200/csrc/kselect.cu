// kselect.cu -- fs_kselect: batched k-selection.
//
//   A1 stream + first-level filter   kselect_warp_kernel main loop
//   A2 restore invariants            warp_flush<NQ,NB> in select.cuh
//   A3 output                        final flush + gather of the original bits
//   A4 long rows                     rows are cut into P chunks, one warp each; the
//                                    P*k partial results are selected again
//   A5 k = 1                         kselect_k1_kernel: min/argmin reduction
//
// One warp owns one work item (a row, or a chunk of a row); lane j reads elements
// 4j..4j+3 of each 128-element group with one 128-bit load (the vectorised form
// of "lane j reads a_{32i+j}"), four groups in flight per lane.
#include "common.cuh"
#include "select.cuh"

namespace fs {

struct KSelArgs {
  const float* vals;     // [n_rows][ld] values to select from
  const int32_t* in_idx; // optional [n_rows][ld]: index each value stands for (pass >= 2); -1 = skip
  int64_t n_rows, n, ld;
  int P;                 // chunks per row
  int64_t chunk;         // elements per chunk (multiple of 4)
  const float* gather;   // original rows: out_val = gather[row*gather_ld + idx]
  int64_t gather_ld;
  float* out_val;        // [n_rows][P][k]
  int32_t* out_idx;
  int k;
};

__device__ __forceinline__ float4 ld_stream4(const float* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
               : "l"(p));
  return r;
}

// ---------------------------------------------------------------------------
// General k: one warp per (row, chunk).
// ---------------------------------------------------------------------------
template <int NQ, int NB, int WARPS>
__global__ void __launch_bounds__(WARPS * 32) kselect_warp_kernel(const KSelArgs a) {
  extern __shared__ __align__(16) uint64_t smem_keys[];
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
  const int32_t* pi = a.in_idx ? a.in_idx + row * a.ld + start : nullptr;
  const uint32_t base = (uint32_t)start;

  WarpSelect<NQ, NB> q;
  q.init(smem_keys + warp * warp_select_smem_keys<NB>(), lane);

  // One element per lane with explicit validity (head, tail, and the indexed pass).
  auto scalar_round = [&](int64_t e) {
    bool ok = e < len;
    float v = 0.f;
    uint32_t idx = 0;
    if (ok) {
      v = p[e];
      if (pi) {
        const int32_t t = pi[e];
        ok = t >= 0;
        idx = (uint32_t)t;
      } else {
        idx = base + (uint32_t)e;
      }
    }
    const uint64_t key = make_key(v, idx);
    q.push(ok && q.maybe(v) && q.wants(key), key);
  };

  if (pi) {
    for (int64_t e0 = 0; e0 < len; e0 += 32) scalar_round(e0 + lane);
  } else {
    // peel to 16-byte alignment
    int64_t head = (4 - (int)(((uintptr_t)p >> 2) & 3)) & 3;
    if (head > len) head = len;
    if (head) scalar_round(lane < head ? lane : len);
    const float* pv = p + head;
    const int64_t nvec = (len - head) >> 2;
    const uint32_t vbase = base + (uint32_t)head;

    auto consume = [&](const float4& x, int64_t v) {
      const bool any = q.maybe(x.x) | q.maybe(x.y) | q.maybe(x.z) | q.maybe(x.w);
      if (__any_sync(kFull, any)) {
        const uint32_t i0 = vbase + (uint32_t)(v << 2);
        const float xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll 1
        for (int t = 0; t < 4; ++t) {
          const float xv = t == 0 ? xs[0] : t == 1 ? xs[1] : t == 2 ? xs[2] : xs[3];
          const uint64_t key = make_key(xv, i0 + t);
          q.push(q.maybe(xv) && q.wants(key), key);
        }
      }
    };

    constexpr int U = 4;
    int64_t v0 = 0;
    for (; v0 + U * 32 <= nvec; v0 += U * 32) {
      float4 x[U];
#pragma unroll
      for (int u = 0; u < U; ++u) x[u] = ld_stream4(pv + ((v0 + u * 32 + lane) << 2));
#pragma unroll 1
      for (int u = 0; u < U; ++u) {
        const float4 xu = u == 0 ? x[0] : u == 1 ? x[1] : u == 2 ? x[2] : x[3];
        consume(xu, v0 + u * 32 + lane);
      }
    }
    for (; v0 < nvec; v0 += 32) {
      const int64_t v = v0 + lane;
      const bool ok = v < nvec;
      float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
      if (ok) x = ld_stream4(pv + (v << 2));
      const uint32_t i0 = vbase + (uint32_t)(v << 2);
#pragma unroll 1
      for (int t = 0; t < 4; ++t) {
        const float xv = t == 0 ? x.x : t == 1 ? x.y : t == 2 ? x.z : x.w;
        const uint64_t key = make_key(xv, i0 + t);
        q.push(ok && q.maybe(xv) && q.wants(key), key);
      }
    }
    const int64_t done = head + (nvec << 2);
    if (done < len) scalar_round(done + lane);
  }
  q.finish();

  // A3: W is the answer; element i = r*32 + lane.
  const float* g = a.gather + row * a.gather_ld;
  float* ov = a.out_val + item * a.k;
  int32_t* oi = a.out_idx + item * a.k;
#pragma unroll
  for (int r = 0; r < NQ; ++r) {
    const int i = r * 32 + lane;
    if (i < a.k) {
      const uint64_t key = q.W[r];
      if (key == kSentinelKey) {
        ov[i] = __uint_as_float(0x7F800000u);
        oi[i] = -1;
      } else {
        const uint32_t idx = key_idx(key);
        ov[i] = g[idx];
        oi[i] = (int32_t)idx;
      }
    }
  }
}

// ---------------------------------------------------------------------------
// k = 1: min / argmin reduction on packed keys, one warp per (row, chunk).
// ---------------------------------------------------------------------------
template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) kselect_k1_kernel(const KSelArgs a) {
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
  const int32_t* pi = a.in_idx ? a.in_idx + row * a.ld + start : nullptr;
  const uint32_t base = (uint32_t)start;
  uint64_t best = kSentinelKey;

  if (pi) {
    for (int64_t e = lane; e < len; e += 32) {
      const int32_t t = pi[e];
      if (t >= 0) best = umin64(best, make_key(p[e], (uint32_t)t));
    }
  } else {
    int64_t head = (4 - (int)(((uintptr_t)p >> 2) & 3)) & 3;
    if (head > len) head = len;
    if (lane < head) best = umin64(best, make_key(p[lane], base + lane));
    const float* pv = p + head;
    const int64_t nvec = (len - head) >> 2;
    const uint32_t vbase = base + (uint32_t)head;
    // Per lane a running float minimum decides whether the exact key compare is
    // needed at all: "!(v > m)" is true for v <= m and for NaN.
    float m = __uint_as_float(0x7FFFFFFFu);
    auto take = [&](float v, uint32_t idx) {
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
  }
#pragma unroll
  for (int s = 16; s >= 1; s >>= 1) best = umin64(best, shfl_xor64(best, s));
  if (lane == 0) {
    if (best == kSentinelKey) {
      a.out_val[item] = __uint_as_float(0x7F800000u);
      a.out_idx[item] = -1;
    } else {
      const uint32_t idx = key_idx(best);
      a.out_val[item] = a.gather[row * a.gather_ld + idx];
      a.out_idx[item] = (int32_t)idx;
    }
  }
}

// ---------------------------------------------------------------------------
// Host side: plan of passes (A4) and launches.
// ---------------------------------------------------------------------------
namespace {

constexpr int kWarpsPerCta = 4;

struct Pass {
  int64_t n;  // elements per row entering this pass
  int P;      // chunks per row
  int64_t chunk;
};

// Rows are cut into chunks until one warp per row is enough to occupy the GPU or
// a chunk would fall under max(4096, 8k) elements (below that the k outputs per
// chunk dominate).  Returns the passes; the last one has P == 1.
int plan_passes(int64_t n_rows, int64_t n, int k, Pass* out) {
  const int64_t target_items = (int64_t)sm_count() * 16;
  const int64_t min_chunk = k * 8 > 4096 ? (int64_t)k * 8 : 4096;
  int np = 0;
  while (np < 7) {
    int64_t P = 1;
    if (n_rows < target_items && n >= 2 * min_chunk) {
      P = ceil_div(target_items, n_rows);
      const int64_t pmax = n / min_chunk;
      if (P > pmax) P = pmax;
      if (P < 1) P = 1;
    }
    int64_t chunk = ceil_div(n, P);
    chunk = (chunk + 3) / 4 * 4;
    if (chunk < 4) chunk = 4;
    P = n > 0 ? ceil_div(n, chunk) : 1;
    out[np++] = Pass{n, (int)P, chunk};
    if (P == 1) break;
    n = P * k;
  }
  if (out[np - 1].P != 1) out[np++] = Pass{n, 1, (n + 3) / 4 * 4 > 4 ? (n + 3) / 4 * 4 : 4};
  return np;
}

template <int NQ, int NB>
int launch_warp(const KSelArgs& a, cudaStream_t s) {
  const int64_t items = a.n_rows * a.P;
  if (items == 0) return FS_OK;
  const size_t smem = (size_t)kWarpsPerCta * warp_select_smem_keys<NB>() * sizeof(uint64_t);
  const int64_t grid = ceil_div(items, kWarpsPerCta);
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "too many rows for one launch");
  kselect_warp_kernel<NQ, NB, kWarpsPerCta><<<(unsigned)grid, kWarpsPerCta * 32, smem, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
}

int launch_pass(const KSelArgs& a, cudaStream_t s) {
  const int k = a.k;
  if (k == 1) {
    const int64_t items = a.n_rows * a.P;
    if (items == 0) return FS_OK;
    const int64_t grid = ceil_div(items, kWarpsPerCta);
    if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "too many rows for one launch");
    kselect_k1_kernel<kWarpsPerCta><<<(unsigned)grid, kWarpsPerCta * 32, 0, s>>>(a);
    FS_LAUNCHED();
    return FS_OK;
  }
  if (k <= 32) return launch_warp<1, 1>(a, s);
  if (k <= 64) return launch_warp<2, 2>(a, s);
  if (k <= 128) return launch_warp<4, 4>(a, s);
  if (k <= 256) return launch_warp<8, 8>(a, s);
  if (k <= 512) return launch_warp<16, 8>(a, s);
  return launch_warp<32, 8>(a, s);
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

// Selection over device rows; also used by the flat and IVFPQ drivers.
size_t kselect_ws_bytes(int64_t n_rows, int64_t n, int k) {
  Pass ps[8];
  const int np = plan_passes(n_rows, n, k, ps);
  size_t tot = 0;
  for (int i = 0; i + 1 < np; ++i)
    tot += align_up((size_t)n_rows * ps[i].P * k * sizeof(float), 256) +
           align_up((size_t)n_rows * ps[i].P * k * sizeof(int32_t), 256);
  return tot;
}

int kselect_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                   int32_t* out_idx, void* ws, cudaStream_t s) {
  Pass ps[8];
  const int np = plan_passes(n_rows, n, k, ps);
  char* w = static_cast<char*>(ws);
  const float* cur_val = rows;
  const int32_t* cur_idx = nullptr;
  int64_t cur_ld = ld;
  for (int i = 0; i < np; ++i) {
    KSelArgs a;
    a.vals = cur_val;
    a.in_idx = cur_idx;
    a.n_rows = n_rows;
    a.n = ps[i].n;
    a.ld = cur_ld;
    a.P = ps[i].P;
    a.chunk = ps[i].chunk;
    a.gather = rows;
    a.gather_ld = ld;
    a.k = k;
    const bool last = (i == np - 1);
    if (last) {
      a.out_val = out_val;
      a.out_idx = out_idx;
    } else {
      a.out_val = reinterpret_cast<float*>(w);
      w += align_up((size_t)n_rows * ps[i].P * k * sizeof(float), 256);
      a.out_idx = reinterpret_cast<int32_t*>(w);
      w += align_up((size_t)n_rows * ps[i].P * k * sizeof(int32_t), 256);
    }
    const int rc = launch_pass(a, s);
    if (rc != FS_OK) return rc;
    cur_val = a.out_val;
    cur_idx = a.out_idx;
    cur_ld = (int64_t)ps[i].P * k;
  }
  return FS_OK;
}

}  // namespace fs

extern "C" {

size_t fs_kselect_ws_bytes(int64_t n_rows, int64_t n, int k) {
  if (n_rows < 0 || n < 0 || k < 1 || k > FS_MAX_K) return 0;
  return fs::kselect_ws_bytes(n_rows, n, k);
}

int fs_kselect(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
               int32_t* out_idx, void* ws, size_t ws_bytes, fs_stream stream) {
  int rc = fs::validate(rows, n_rows, n, ld, k, out_val, out_idx);
  if (rc != FS_OK) return rc;
  if (n_rows == 0) return FS_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  fs::TempWs t;
  rc = t.acquire(ws, ws_bytes, fs::kselect_ws_bytes(n_rows, n, k), s);
  if (rc != FS_OK) return rc;
  return fs::kselect_device(rows, n_rows, n, ld, k, out_val, out_idx, t.ptr, s);
}

int fs_kselect_host(const float* rows_host, int64_t n_rows, int64_t n, int64_t ld, int k,
                    float* out_val_host, int32_t* out_idx_host) {
  int rc = fs::validate(rows_host, n_rows, n, ld, k, out_val_host, out_idx_host);
  if (rc != FS_OK) return rc;
  if (n_rows == 0) return FS_OK;
  float* d_rows = nullptr;
  float* d_val = nullptr;
  int32_t* d_idx = nullptr;
  const size_t in_b = (size_t)n_rows * ld * sizeof(float), out_n = (size_t)n_rows * k;
  cudaStream_t s = nullptr;
  rc = FS_OK;
  auto fail = [&](cudaError_t e, const char* what) {
    rc = fs::set_error(FS_ECUDA, "%s failed: %s", what, cudaGetErrorString(e));
  };
  cudaError_t e;
  if ((e = cudaMalloc(&d_rows, in_b ? in_b : 16)) != cudaSuccess) fail(e, "cudaMalloc");
  if (rc == FS_OK && (e = cudaMalloc(&d_val, out_n * sizeof(float))) != cudaSuccess) fail(e, "cudaMalloc");
  if (rc == FS_OK && (e = cudaMalloc(&d_idx, out_n * sizeof(int32_t))) != cudaSuccess) fail(e, "cudaMalloc");
  if (rc == FS_OK && in_b &&
      (e = cudaMemcpyAsync(d_rows, rows_host, in_b, cudaMemcpyHostToDevice, s)) != cudaSuccess)
    fail(e, "cudaMemcpyAsync H2D");
  if (rc == FS_OK) rc = fs_kselect(d_rows, n_rows, n, ld, k, d_val, d_idx, nullptr, 0, s);
  if (rc == FS_OK && (e = cudaMemcpyAsync(out_val_host, d_val, out_n * sizeof(float),
                                          cudaMemcpyDeviceToHost, s)) != cudaSuccess)
    fail(e, "cudaMemcpyAsync D2H");
  if (rc == FS_OK && (e = cudaMemcpyAsync(out_idx_host, d_idx, out_n * sizeof(int32_t),
                                          cudaMemcpyDeviceToHost, s)) != cudaSuccess)
    fail(e, "cudaMemcpyAsync D2H");
  if ((e = cudaStreamSynchronize(s)) != cudaSuccess && rc == FS_OK) fail(e, "cudaStreamSynchronize");
  cudaFree(d_rows);
  cudaFree(d_val);
  cudaFree(d_idx);
  return rc;
}

}  // extern "C"
