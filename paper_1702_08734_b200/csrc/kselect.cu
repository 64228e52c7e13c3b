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
#include "tselect.cuh"

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
// General k: one warp per (row, chunk); threshold-filtered selection (tselect.cuh).
// ---------------------------------------------------------------------------
template <int NQ>
__global__ void __launch_bounds__(TSelCfg<NQ>::WARPS * 32) kselect_warp_kernel(const KSelArgs a) {
  constexpr int WARPS = TSelCfg<NQ>::WARPS;
  constexpr int LCAP = TSelCfg<NQ>::LCAP;
  constexpr int U = 8;          // 128-bit loads in flight per lane
  constexpr int SAMPLE = 1024;  // elements of the row used to place the first bound
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

  TSel<NQ> q;
  q.init(smem_keys + (size_t)warp * (32 * LCAP), lane);

  if (pi) {
    // pass >= 2: (value, index) pairs in arbitrary index order; index -1 = padding
    for (int64_t e0 = 0; e0 < len; e0 += 32) {
      const int64_t e = e0 + lane;
      bool ok = e < len;
      float v = 0.f;
      int32_t t = -1;
      if (ok) {
        v = p[e];
        t = pi[e];
      }
      q.push(ok && t >= 0, v, (uint32_t)t);
      if (q.crowded()) q.flush(false);
    }
    q.flush(false);
  } else {
    int64_t head = (4 - (int)(((uintptr_t)p >> 2) & 3)) & 3;
    if (head > len) head = len;
    const float* pv = p + head;
    const int64_t nvec = (len - head) >> 2;
    const uint32_t vbase = base + (uint32_t)head;
    const int64_t done = head + (nvec << 2);
    // elements of the sample that should pass so that ~MSTAR of the chunk do
    float rho = (float)TSelCfg<NQ>::MSTAR * (float)SAMPLE / (float)(len > 0 ? len : 1);
    if (rho < 12.f) rho = 12.f;
    const int rho_lo = (int)rho, rho_hi = (int)(rho * 1.25f) + 1;
    const bool can_sample = nvec >= U * 32 && rho_hi < SAMPLE / 2;
    const int64_t want = a.k < len ? a.k : len;

    auto push4 = [&](const float4& x, int64_t v, bool ok) {
      const uint32_t i0 = vbase + (uint32_t)(v << 2);
      q.push(ok, x.x, i0);
      q.push(ok, x.y, i0 + 1);
      q.push(ok, x.z, i0 + 2);
      q.push(ok, x.w, i0 + 3);
    };

#pragma unroll 1
    for (int attempt = 0; attempt < 2; ++attempt) {
      const bool sampled = attempt == 0 && can_sample;
      q.reset();
      if (head) q.push(lane < head, lane < head ? p[lane] : 0.f, base + lane);
      if (sampled) {
        // counting bisection in the order image over the first SAMPLE elements:
        // find o with rho_lo <= #(v <= o) <= rho_hi.  No call while x[] is live.
        float4 x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ld_stream4(pv + ((int64_t)(u * 32 + lane) << 2));
        uint32_t lo = 0u, hi = 0xFF800000u, pick = 0xFF800000u;
#pragma unroll 1
        for (int it = 0; it < 34 && hi - lo > 1u; ++it) {
          const uint32_t mid = lo + ((hi - lo) >> 1);
          const float tf = ord_f32(mid);
          int cme = 0;
#pragma unroll
          for (int u = 0; u < U; ++u)
            cme += (x[u].x <= tf) + (x[u].y <= tf) + (x[u].z <= tf) + (x[u].w <= tf);
          const int cw = __reduce_add_sync(kFull, cme);
          if (cw < rho_lo) {
            lo = mid;
          } else {
            hi = mid;
            pick = mid;
            if (cw <= rho_hi) break;
          }
        }
        q.set_sampled_bound(pick);
      }
      // Stream.  A batch stops early when a lane queue runs full; the restore
      // step is called at ONE site where no loaded data is live, and the batch
      // restarts behind the last 128-bit group that was consumed.
      int64_t v0 = 0;
      while (v0 + U * 32 <= nvec) {
        float4 x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ld_stream4(pv + ((v0 + u * 32 + lane) << 2));
        int used = U;
        bool full = false;
#pragma unroll
        for (int u = 0; u < U; ++u) {
          if (!full) {
            push4(x[u], v0 + u * 32 + lane, true);
            full = q.crowded();
            if (full) used = u + 1;
          }
        }
        v0 += used * 32;
        if (full) q.flush(true);
      }
      for (; v0 < nvec; v0 += 32) {
        const int64_t v = v0 + lane;
        const bool ok = v < nvec;
        float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
        if (ok) x = ld_stream4(pv + (v << 2));
        push4(x, v, ok);
        if (q.crowded()) q.flush(true);
      }
      if (done < len) {
        const bool ok = done + lane < len;
        q.push(ok, ok ? p[done + lane] : 0.f, base + (uint32_t)(done + lane));
      }
      q.flush(true);
      // the sampled bound let fewer than k elements through: scan again with the
      // adaptive bound only (exact in every case)
      if (!sampled || q.exact || q.total >= want) break;
    }
  }

  // A3: buf[swz<NQ>(i)] is the i-th smallest key.  The value is rebuilt from the
  // key's order image, except for the two images that are not injective (+-0 and
  // NaN), which are re-read from the row so that the original bits come back.
  const float* g = a.gather + row * a.gather_ld;
  float* ov = a.out_val + item * a.k;
  int32_t* oi = a.out_idx + item * a.k;
  for (int i = lane; i < a.k; i += 32) {
    const uint64_t key = q.buf[swz<NQ>(i)];
    if (key == kSentinelKey) {
      ov[i] = __uint_as_float(0x7F800000u);
      oi[i] = -1;
    } else {
      const uint32_t idx = key_idx(key), o = (uint32_t)(key >> 32);
      ov[i] = (o == 0x80000000u || o == 0xFFFFFFFFu) ? g[idx] : ord_f32(o);
      oi[i] = (int32_t)idx;
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

template <int NQ>
int launch_warp(const KSelArgs& a, cudaStream_t s) {
  constexpr int WARPS = TSelCfg<NQ>::WARPS;
  const int64_t items = a.n_rows * a.P;
  if (items == 0) return FS_OK;
  const size_t smem = (size_t)WARPS * 32 * TSelCfg<NQ>::LCAP * sizeof(uint64_t);
  static bool attr_done = false;
  if (!attr_done) {
    FS_CUDA(cudaFuncSetAttribute(kselect_warp_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)smem));
    FS_CUDA(cudaFuncSetAttribute(kselect_warp_kernel<NQ>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 cudaSharedmemCarveoutMaxShared));
    attr_done = true;
  }
  const int64_t grid = ceil_div(items, WARPS);
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "too many rows for one launch");
  kselect_warp_kernel<NQ><<<(unsigned)grid, WARPS * 32, smem, s>>>(a);
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
  if (k <= 32) return launch_warp<1>(a, s);
  if (k <= 64) return launch_warp<2>(a, s);
  if (k <= 128) return launch_warp<4>(a, s);
  if (k <= 256) return launch_warp<8>(a, s);
  if (k <= 512) return launch_warp<16>(a, s);
  return launch_warp<32>(a, s);
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
