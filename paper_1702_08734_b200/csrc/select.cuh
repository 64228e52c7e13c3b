// select.cuh -- warp-level k-selection state kept in registers.
//
// What it computes is the paper's WarpSelect contract: after any
// prefix of the input the warp queue W holds the k smallest elements seen,
// sorted ascending in a lane-stride register array.  How it
// gets there differs from the paper's Maxwell design:
//   * every comparison is on one packed 64-bit key (order-preserving transform
//     of the fp32 bits, then the index), so ties resolve to the lower index
//     everywhere and a single unsigned compare orders (value, index);
//   * the first-level filter is one compare against the warp queue's tail
//     W[k-1] (kept broadcast in a register) instead of per-lane thread queues
//     (P:L218); accepted elements are compacted by ballot/popc into a per-warp
//     shared-memory batch of C candidates, so a sort+merge event always
//     processes a full batch rather than firing when any one lane's queue fills
//     (P:L230-232);
//   * the batch is sorted with a bitonic network in a BLOCKED register layout
//     (lane l holds elements l*NB..l*NB+NB-1): 15 cross-lane shuffle steps for
//     any batch size instead of 5 per merge stage in lane-stride layout; it is
//     then merged into W with the half-cleaner "W[K-1-i] = min(W[K-1-i], B[i])"
//     followed by a log2(K)-step bitonic merge (power-of-two sizes with
//     sentinel padding instead of the odd-size networks of Alg. 1-2,
//     P:L146-208).
#pragma once

#include <cstdint>

#include "common.cuh"

namespace fs {

constexpr uint64_t kSentinelKey = ~0ull;  // (NaN-rank, index -1): sorts after every real key

// Order-preserving map fp32 -> uint32: a < b  <=>  ord(a) < ord(b) for non-NaN
// a, b, with -0 == +0; every NaN maps to 0xFFFFFFFF (after +inf).
__device__ __forceinline__ uint32_t f32_ord(float v) {
  uint32_t b = __float_as_uint(v);
  if (v != v) return 0xFFFFFFFFu;
  if (b == 0x80000000u) b = 0u;
  return b ^ ((uint32_t)((int32_t)b >> 31) | 0x80000000u);
}
// Inverse (up to -0 -> +0 and NaN payload): used for the float pre-filter and
// for values computed on chip (distances), never for copies of caller data.
__device__ __forceinline__ float ord_f32(uint32_t o) {
  const uint32_t b = (o & 0x80000000u) ? (o ^ 0x80000000u) : ~o;
  return __uint_as_float(b);
}
__device__ __forceinline__ uint64_t make_key(float v, uint32_t idx) {
  return ((uint64_t)f32_ord(v) << 32) | idx;
}
__device__ __forceinline__ uint32_t key_idx(uint64_t k) { return (uint32_t)k; }
__device__ __forceinline__ float key_val(uint64_t k) { return ord_f32((uint32_t)(k >> 32)); }

__device__ __forceinline__ uint64_t umin64(uint64_t a, uint64_t b) { return a < b ? a : b; }
__device__ __forceinline__ uint64_t umax64(uint64_t a, uint64_t b) { return a < b ? b : a; }
__device__ __forceinline__ uint64_t shfl_xor64(uint64_t v, int m) {
  return __shfl_xor_sync(kFull, v, m);
}

// Bitonic sort of 32*NB keys held in BLOCKED layout: element e = lane*NB + r.
template <int NB>
__device__ __forceinline__ void sort_blocked(uint64_t (&B)[NB], int lane) {
  constexpr int N = 32 * NB;
#pragma unroll
  for (int sz = 2; sz <= N; sz <<= 1) {
#pragma unroll
    for (int j = sz >> 1; j >= 1; j >>= 1) {
      if (j >= NB) {  // partner in lane ^ (j / NB), same register
        const int lj = j / NB;
        const bool lower = (lane & lj) == 0;
        const bool asc = (sz >= N) ? true : (((lane * NB) & sz) == 0);
#pragma unroll
        for (int r = 0; r < NB; ++r) {
          const uint64_t o = shfl_xor64(B[r], lj);
          B[r] = (asc == lower) ? umin64(B[r], o) : umax64(B[r], o);
        }
      } else {  // partner register r ^ j in the same lane
#pragma unroll
        for (int r = 0; r < NB; ++r) {
          if ((r & j) == 0) {
            const bool asc =
                (sz >= N) ? true : ((sz < NB) ? ((r & sz) == 0) : (((lane * NB) & sz) == 0));
            const uint64_t lo = umin64(B[r], B[r | j]), hi = umax64(B[r], B[r | j]);
            B[r] = asc ? lo : hi;
            B[r | j] = asc ? hi : lo;
          }
        }
      }
    }
  }
}

// Bitonic merge of a bitonic sequence of 32*NQ keys in LANE-STRIDE layout
// (element e = r*32 + lane) into ascending order.
template <int NQ>
__device__ __forceinline__ void merge_lane_stride(uint64_t (&W)[NQ], int lane) {
#pragma unroll
  for (int j = NQ / 2; j >= 1; j >>= 1) {
#pragma unroll
    for (int r = 0; r < NQ; ++r) {
      if ((r & j) == 0) {
        const uint64_t lo = umin64(W[r], W[r | j]), hi = umax64(W[r], W[r | j]);
        W[r] = lo;
        W[r | j] = hi;
      }
    }
  }
#pragma unroll
  for (int lj = 16; lj >= 1; lj >>= 1) {
    const bool lower = (lane & lj) == 0;
#pragma unroll
    for (int r = 0; r < NQ; ++r) {
      const uint64_t o = shfl_xor64(W[r], lj);
      W[r] = lower ? umin64(W[r], o) : umax64(W[r], o);
    }
  }
}

// Merge another ascending queue of 32*NQ keys (lane-stride in memory: element e at other[e]) into the
// ascending lane-stride queue W, keeping the 32*NQ smallest: half-cleaner against the reversed other
// queue, then the bitonic merge.  Warp-collective.
template <int NQ>
__device__ __forceinline__ void merge_sorted_queue(uint64_t (&W)[NQ], const uint64_t* other, int lane) {
#pragma unroll
  for (int r = 0; r < NQ; ++r) W[NQ - 1 - r] = umin64(W[NQ - 1 - r], other[r * 32 + (31 - lane)]);
  merge_lane_stride<NQ>(W, lane);
}

// Shared-memory words (uint64) one warp's candidate batch needs.
template <int NB>
__host__ __device__ constexpr int warp_select_smem_keys() {
  return 32 * NB + 2 * NB + 2;  // C keys + padding of the conflict-free blocked layout
}

// Sort one warp's batch of cnt (<= 32*NB) candidate keys in buf and merge it
// into the warp queue W (32*NQ keys, lane-stride, ascending): this lane's r-th
// key is Wmem[r * wstride] (wstride = 1 for a lane-private array, 32 for a
// shared/global array addressed as base + lane).  Returns the new threshold
// W[K-1].  Deliberately NOT inlined: one copy of the networks per (NQ, NB); W
// goes through memory (NQ loads + NQ stores per call against the ~10^3
// instructions of the networks).  Warp-collective.
template <int NQ, int NB>
__device__ __noinline__ uint64_t warp_flush(uint64_t* Wmem, int wstride, uint64_t* buf, int cnt) {
  const int lane = threadIdx.x & 31;
  constexpr int NM = NB < NQ ? NB : NQ;  // batch registers that can reach the queue
  __syncwarp();
  uint64_t B[NB];
#pragma unroll
  for (int r = 0; r < NB; ++r) {
    const int e = r * 32 + lane;  // any bijection slot -> (lane, reg) will do: unsorted
    B[r] = e < cnt ? buf[e] : kSentinelKey;
  }
  sort_blocked<NB>(B, lane);
  __syncwarp();
  // blocked (sorted position e = lane*NB + r) -> shared, padded against bank conflicts
#pragma unroll
  for (int r = 0; r < NB; ++r) {
    const int e = lane * NB + r;
    buf[e + (e >> 4)] = B[r];
  }
  __syncwarp();
  uint64_t W[NQ];
#pragma unroll
  for (int r = 0; r < NQ; ++r) W[r] = Wmem[r * wstride];
  // half-cleaner against the reversed batch: W[K-1-i] = min(W[K-1-i], B[i]), i < min(C, K)
#pragma unroll
  for (int r = 0; r < NM; ++r) {
    const int i = r * 32 + (31 - lane);
    W[NQ - 1 - r] = umin64(W[NQ - 1 - r], buf[i + (i >> 4)]);
  }
  __syncwarp();
  merge_lane_stride<NQ>(W, lane);
#pragma unroll
  for (int r = 0; r < NQ; ++r) Wmem[r * wstride] = W[r];
  return __shfl_sync(kFull, W[NQ - 1], 31);
}

// Queue-length class of k: K = 32 << kclass >= k.
__host__ __device__ inline int k_class(int k) {
  int c = 0;
  while ((32 << c) < k) ++c;
  return c;
}

// Run-time dispatch for kernels whose body does not depend on the queue length
// (the fused distance kernels): batch of 64 candidates (NB = 2).
__device__ __forceinline__ uint64_t warp_flush_b64(int kclass, uint64_t* Wmem, int wstride,
                                                    uint64_t* buf, int cnt) {
  switch (kclass) {
    case 0: return warp_flush<1, 2>(Wmem, wstride, buf, cnt);
    case 1: return warp_flush<2, 2>(Wmem, wstride, buf, cnt);
    case 2: return warp_flush<4, 2>(Wmem, wstride, buf, cnt);
    case 3: return warp_flush<8, 2>(Wmem, wstride, buf, cnt);
    case 4: return warp_flush<16, 2>(Wmem, wstride, buf, cnt);
    default: return warp_flush<32, 2>(Wmem, wstride, buf, cnt);
  }
}

// Per-warp selection state.  K = 32*NQ >= k is the queue length, C = 32*NB the
// candidate batch.  All member functions are warp-collective (full mask).
template <int NQ, int NB>
struct WarpSelect {
    static constexpr int K = 32 * NQ;
  static constexpr int C = 32 * NB;

  uint64_t W[NQ];    // lane-stride, ascending; kSentinelKey marks empty slots
  uint64_t thr;      // W[kq] (default the tail W[K-1]), broadcast: a key must be < thr to matter
  float thr_val;     // float image of thr for the one-instruction pre-filter
  float sub_val;     // float image of W[ks] (set_k): lets several warps that share a stream bound each other
  uint64_t* buf;     // this warp's shared-memory batch
  int cnt;           // keys in the batch (warp-uniform)
  int lane;
  int kq, ks;        // sorted positions (0-based) whose keys are published as thr / sub_val

  __device__ __forceinline__ void init(uint64_t* smem_buf, int lane_) {
    buf = smem_buf;
    lane = lane_;
    kq = K - 1;
    ks = K - 1;
    reset();
  }
  // Select exactly k <= K: the bound becomes the k-th smallest key instead of the K-th (fewer
  // candidates pass), and sub_val follows the ceil(k / parts)-th smallest: if each of `parts` queues
  // over disjoint parts of a stream holds that many keys <= x, their union holds k keys <= x, so
  // max over the queues of sub_val bounds the union's k-th smallest.
  __device__ __forceinline__ void set_k(int k, int parts) {
    kq = k - 1;
    ks = (k + parts - 1) / parts - 1;
  }
  __device__ __forceinline__ void reset() {
#pragma unroll
    for (int r = 0; r < NQ; ++r) W[r] = kSentinelKey;
    thr = kSentinelKey;
    thr_val = __uint_as_float(0x7FFFFFFFu);  // NaN: "!(v > thr_val)" passes everything
    sub_val = __uint_as_float(0x7F800000u);
    cnt = 0;
  }
  // Cheap necessary condition for "key(v, idx) < thr" (exact test: wants()).
  __device__ __forceinline__ bool maybe(float v) const { return !(v > thr_val); }
  __device__ __forceinline__ bool wants(uint64_t key) const { return key < thr; }

  // Append key on the lanes where pred holds.
  __device__ __forceinline__ void push(bool pred, uint64_t key) {
    const unsigned m = __ballot_sync(kFull, pred);
    if (m == 0) return;
    if (pred) buf[cnt + __popc(m & ((1u << lane) - 1u))] = key;
    cnt += __popc(m);
    if (cnt > C - 32) flush();
  }
  __device__ __forceinline__ void flush() {
    thr = warp_flush<NQ, NB>(W, 1, buf, cnt);
    if (kq != K - 1) {  // (W went through memory for the call: the indexed reads are plain loads)
      thr = __shfl_sync(kFull, W[kq >> 5], kq & 31);
      const uint64_t sk = __shfl_sync(kFull, W[ks >> 5], ks & 31);
      sub_val = sk == kSentinelKey ? __uint_as_float(0x7F800000u) : key_val(sk);
    }
    thr_val = key_val(thr);
    cnt = 0;
  }
  __device__ __forceinline__ void finish() {
    if (cnt > 0) flush();
  }
};

}  // namespace fs
