// tselect.cuh -- threshold-filtered warp k-selection (fs_kselect, rows A1-A3).
//
// Contract = the paper's WarpSelect: after any prefix of the input the
// state holds the k smallest (value, index) keys seen.  The mechanism is re-cut for
// B200, where the instruction budget per streamed element is small (~20 lane
// instructions at 60 % of HBM peak) and shared memory is large:
//
//   * first-level filter: ONE float compare per element against the
//     current bound, exactly as in the paper; an accepted element is appended to
//     a LANE-PRIVATE queue in shared memory (slot (j, lane) -> word j*32+lane:
//     the "thread queue" of P:L218, but LCAP-deep and outside the register file),
//     with no ballot, shuffle or branch on the hot path;
//   * restore step: only when some lane's queue is full (rare) or at
//     the end of the row.  The ragged queues are compacted in place, sorted in
//     blocks of <= 1024 keys with a bitonic network on registers in BLOCKED layout
//     (15 cross-lane steps for any size; power-of-two sizes with sentinel padding
//     instead of the odd-size networks of Alg. 1-2) and min-merged to the k
//     smallest; the k-th key becomes the new exact bound;
//   * the initial bound is not +inf: the first 1024 elements of the row are used
//     as a sample, and a counting bisection on them picks a value that about
//     m* = 1.5k..6k elements of the whole row are expected to pass, so a typical
//     row needs exactly one restore step.  If fewer than k elements passed, the
//     row is scanned again with the paper's adaptive bound (+inf start); the
//     result is exact either way.
//
// Every ordering decision is on the packed 64-bit key of select.cuh, so ties go
// to the lower index everywhere (reading K-1/K-7).
#pragma once

#include "select.cuh"

namespace fs {

// ---- sorting networks on registers, blocked layout (element e = lane*NB + r) ----
// Bitonic sort in the "flip" form: a merge stage of size sz first compares e with
// e ^ (sz - 1) (the mirrored element of the other sorted half), then runs the usual
// half-cleaners e <-> e ^ j, j = sz/4 .. 1.  Every comparator then points the same
// way (smaller key to the smaller position), so the in-register steps have
// compile-time directions and the code stays small.
__device__ __forceinline__ void cmpex_up(uint64_t& a, uint64_t& b) {
  const uint64_t lo = umin64(a, b), hi = umax64(a, b);
  a = lo;
  b = hi;
}

template <int NB>
__device__ __forceinline__ void local_halfcleaners(uint64_t (&B)[NB], int jmax) {
#pragma unroll
  for (int j = NB / 2; j >= 1; j >>= 1) {
    if (j <= jmax) {
#pragma unroll
      for (int r = 0; r < NB; ++r)
        if ((r & j) == 0) cmpex_up(B[r], B[r | j]);
    }
  }
}

template <int NB>
__device__ __forceinline__ void sort_blocked_rt(uint64_t (&B)[NB], int lane) {
  // stages inside a lane
#pragma unroll
  for (int sz = 2; sz <= NB; sz <<= 1) {
#pragma unroll
    for (int r = 0; r < NB; ++r)
      if ((r & (sz >> 1)) == 0) cmpex_up(B[r], B[r ^ (sz - 1)]);
#pragma unroll
    for (int j = sz >> 2; j >= 1; j >>= 1) {
#pragma unroll
      for (int r = 0; r < NB; ++r)
        if ((r & j) == 0) cmpex_up(B[r], B[r | j]);
    }
  }
  // stages across lanes: sz = szl * NB
#pragma unroll 1
  for (int szl = 2; szl <= 32; szl <<= 1) {
    {  // flip: partner lane ^ (szl - 1), mirrored register
      const bool low = (lane & (szl >> 1)) == 0;
      if (NB == 1) {
        const uint64_t o = shfl_xor64(B[0], szl - 1);
        B[0] = low ? umin64(B[0], o) : umax64(B[0], o);
      } else {
#pragma unroll
        for (int r = 0; r < NB / 2; ++r) {
          const uint64_t o1 = shfl_xor64(B[NB - 1 - r], szl - 1);
          const uint64_t o2 = shfl_xor64(B[r], szl - 1);
          B[r] = low ? umin64(B[r], o1) : umax64(B[r], o1);
          B[NB - 1 - r] = low ? umin64(B[NB - 1 - r], o2) : umax64(B[NB - 1 - r], o2);
        }
      }
    }
#pragma unroll 1
    for (int lj = szl >> 2; lj >= 1; lj >>= 1) {
      const bool low = (lane & lj) == 0;
#pragma unroll
      for (int r = 0; r < NB; ++r) {
        const uint64_t o = shfl_xor64(B[r], lj);
        B[r] = low ? umin64(B[r], o) : umax64(B[r], o);
      }
    }
    local_halfcleaners<NB>(B, NB / 2);
  }
}

// B bitonic over all 32*NB elements (blocked) -> ascending.
template <int NB>
__device__ __forceinline__ void merge_blocked_rt(uint64_t (&B)[NB], int lane) {
#pragma unroll 1
  for (int lj = 16; lj >= 1; lj >>= 1) {
    const bool low = (lane & lj) == 0;
#pragma unroll
    for (int r = 0; r < NB; ++r) {
      const uint64_t o = shfl_xor64(B[r], lj);
      B[r] = low ? umin64(B[r], o) : umax64(B[r], o);
    }
  }
  local_halfcleaners<NB>(B, NB / 2);
}

// Conflict-free placement of a blocked array in shared memory without padding:
// position e = l*NB + r is stored at l*NB + (r ^ g(l)); for a fixed r the 16
// lanes of a half-warp then hit 16 different 8-byte bank pairs.
__device__ __forceinline__ int swz_rt(int lognb, int e) {
  const int nb = 1 << lognb;
  const int l = e >> lognb, r = e & (nb - 1);
  const int g = lognb >= 4 ? (l & 15) : ((l >> (4 - lognb)) & (nb - 1));
  return (l << lognb) + (r ^ g);
}
template <int NB>
__device__ __forceinline__ int swz(int e) {
  constexpr int L = NB == 1 ? 0 : NB == 2 ? 1 : NB == 4 ? 2 : NB == 8 ? 3 : NB == 16 ? 4 : 5;
  return swz_rt(L, e);
}

// Sort base[0..n) (dense, any order; n <= 32*NB) -> base[swz<NB>(e)] = e-th
// smallest, sentinel-padded to 32*NB.  Warp-collective.
template <int NB>
__device__ __noinline__ void sort_block(uint64_t* base, int n) {
  const int lane = threadIdx.x & 31;
  uint64_t B[NB];
#pragma unroll
  for (int r = 0; r < NB; ++r) {
    const int e = r * 32 + lane;
    B[r] = e < n ? base[e] : kSentinelKey;
  }
  __syncwarp();
  sort_blocked_rt<NB>(B, lane);
#pragma unroll
  for (int r = 0; r < NB; ++r) base[swz<NB>(lane * NB + r)] = B[r];
  __syncwarp();
}

// MAXN: largest n the caller can have (prunes the tiers that get instantiated).
template <int MAXN>
__device__ __forceinline__ int sort_block_any(uint64_t* base, int n) {  // returns log2(NB)
  if (MAXN <= 32 || n <= 32) { sort_block<1>(base, n); return 0; }
  if (MAXN <= 64 || n <= 64) { sort_block<2>(base, n); return 1; }
  if (MAXN <= 128 || n <= 128) { sort_block<4>(base, n); return 2; }
  if (MAXN <= 256 || n <= 256) { sort_block<8>(base, n); return 3; }
  if (MAXN <= 512 || n <= 512) { sort_block<16>(base, n); return 4; }
  sort_block<32>(base, n);
  return 5;
}

// buf[0..m) dense keys -> buf[swz<NQ>(i)], i < K = 32*NQ: the K smallest ascending
// (sentinel padded).  Needs room for ceil(m/BLK) blocks of BLK keys.  Returns the
// K-th key (kSentinelKey if m < K).  Warp-collective.
template <int NQ, int CAP>
__device__ __noinline__ uint64_t select_topk(uint64_t* buf, int m) {
  // sort-block size: 512 keys (16 per lane) keeps the register count of the whole
  // call tree at 128 for k <= 512; only the k = 1024 class sorts 1024 at a time
  constexpr int LBLK = NQ == 32 ? 10 : 9;
  constexpr int BLK = 1 << LBLK;
  constexpr int K = 32 * NQ;
  constexpr int LQ = NQ == 1 ? 0 : NQ == 2 ? 1 : NQ == 4 ? 2 : NQ == 8 ? 3 : NQ == 16 ? 4 : 5;
  const int lane = threadIdx.x & 31;
  const int nblk = m > BLK ? ((m + BLK - 1) >> LBLK) : 1;
  int tiers = 0;  // log2(NB) of block b in bits [4b, 4b+4)
#pragma unroll 1
  for (int b = 0; b < nblk; ++b) {
    int nb = m - (b << LBLK);
    if (nb > BLK) nb = BLK;
    tiers |= sort_block_any<(CAP < BLK ? CAP : BLK)>(buf + (b << LBLK), nb) << (4 * b);
  }
  const int t0 = tiers & 15;
  if (nblk == 1 && t0 == LQ) return buf[swz<NQ>(K - 1)];
  uint64_t W[NQ];
#pragma unroll
  for (int r = 0; r < NQ; ++r) {
    const int i = lane * NQ + r;
    W[r] = (i < (32 << t0)) ? buf[swz_rt(t0, i)] : kSentinelKey;
  }
#pragma unroll 1
  for (int b = 1; b < nblk; ++b) {
    const uint64_t* bb = buf + (b << LBLK);
    const int t = (tiers >> (4 * b)) & 15;
#pragma unroll
    for (int r = 0; r < NQ; ++r) {
      const int p = K - 1 - (lane * NQ + r);
      const uint64_t o = (p < (32 << t)) ? bb[swz_rt(t, p)] : kSentinelKey;
      W[r] = umin64(W[r], o);
    }
    merge_blocked_rt<NQ>(W, lane);
  }
  __syncwarp();
#pragma unroll
  for (int r = 0; r < NQ; ++r) buf[swz<NQ>(lane * NQ + r)] = W[r];
  __syncwarp();
  return __shfl_sync(kFull, W[NQ - 1], 31);
}

// Per-class sizes: LCAP = depth of each lane queue (capacity 32*LCAP keys, a
// multiple of the 1024-key sort block where it exceeds one), MSTAR = number of
// elements the sampled bound is aimed to let through.
template <int NQ> struct TSelCfg;
template <> struct TSelCfg<1> { static constexpr int LCAP = 16, MSTAR = 192, WARPS = 4; };
template <> struct TSelCfg<2> { static constexpr int LCAP = 32, MSTAR = 288, WARPS = 4; };
template <> struct TSelCfg<4> { static constexpr int LCAP = 32, MSTAR = 448, WARPS = 4; };
template <> struct TSelCfg<8> { static constexpr int LCAP = 48, MSTAR = 704, WARPS = 4; };
template <> struct TSelCfg<16> { static constexpr int LCAP = 64, MSTAR = 960, WARPS = 2; };
template <> struct TSelCfg<32> { static constexpr int LCAP = 96, MSTAR = 1536, WARPS = 1; };

__device__ __forceinline__ float ord_next_up(uint32_t o) {
  // smallest float strictly above the value with order image o; NaN ("accept
  // everything" under !(v >= x)) when there is none
  return o >= 0xFF800000u ? __uint_as_float(0x7FFFFFFFu) : ord_f32(o + 1u);
}

struct TSelFlushOut {
  uint64_t kth;  // K-th smallest key (kSentinelKey if fewer than K survive)
  int m;         // keys that entered the selection
};

// Compacts the ragged lane queues of one warp in place (rows [0, wrows) hold keys
// already, the rest raw (bits, index) pairs), drops what the exact bound excludes,
// and selects: on return buf[swz<NQ>(i)], i < K, are the K smallest ascending.
// A free function taking values so that the caller's state stays in registers.
template <int NQ>
__device__ __noinline__ TSelFlushOut tsel_flush(uint64_t* buf, int cnt, int wrows, uint64_t thr_key) {
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  int maxc = cnt;
#pragma unroll
  for (int s = 16; s >= 1; s >>= 1) {
    const int o = __shfl_xor_sync(kFull, maxc, s);
    maxc = o > maxc ? o : maxc;
  }
  int m = 0;
  for (int j = 0; j < maxc; ++j) {
    bool valid = j < cnt;
    uint64_t key = kSentinelKey;
    if (valid) {
      const uint64_t e = buf[j * 32 + lane];
      key = j < wrows ? e : make_key(__uint_as_float((uint32_t)e), (uint32_t)(e >> 32));
      valid = key != kSentinelKey && key <= thr_key;
    }
    const unsigned b = __ballot_sync(kFull, valid);  // also orders this row's reads before the writes
    if (valid) buf[m + __popc(b & lt)] = key;
    m += __popc(b);
    __syncwarp();
  }
  TSelFlushOut out;
  out.kth = select_topk<NQ, 32 * TSelCfg<NQ>::LCAP>(buf, m);
  out.m = m;
  return out;
}

template <int NQ>
struct TSel {
  static constexpr int K = 32 * NQ;
  static constexpr int LCAP = TSelCfg<NQ>::LCAP;

  uint64_t* buf;     // this warp's 32*LCAP slots
  uint64_t thr_key;  // exact bound once `exact`; kSentinelKey before
  float thr_x;       // an element enters iff !(v >= thr_x)
  int cnt;           // entries in this lane's queue (rows [0, wrows) are shared, see flush)
  int wrows;         // rows that already hold keys (the current top-K), 0 or NQ
  int total;         // valid keys after the last flush (<= K)
  int lane;
  bool exact;        // thr_key is the K-th smallest key of everything seen so far

  __device__ __forceinline__ void init(uint64_t* b, int lane_) {
    buf = b;
    lane = lane_;
    reset();
  }
  __device__ __forceinline__ void reset() {
    thr_key = kSentinelKey;
    thr_x = __uint_as_float(0x7FFFFFFFu);
    cnt = 0;
    wrows = 0;
    total = 0;
    exact = false;
  }
  // Sampled bound (inclusive): everything with order image <= o passes.
  __device__ __forceinline__ void set_sampled_bound(uint32_t o) { thr_x = ord_next_up(o); }

  __device__ __forceinline__ void push(bool ok, float v, uint32_t idx) {
    if (ok && !(v >= thr_x)) {
      buf[cnt * 32 + lane] = ((uint64_t)idx << 32) | __float_as_uint(v);  // raw (bits, index)
      ++cnt;
    }
  }
  __device__ __forceinline__ bool crowded() const { return __any_sync(kFull, cnt > LCAP - 4); }

  // Restore step.  monotone: every future element has a larger index than all
  // elements seen so far, so ties with the bound can never win (strict bound).
  __device__ __forceinline__ void flush(bool monotone) {
    const TSelFlushOut o = tsel_flush<NQ>(buf, cnt, wrows, thr_key);
    total = o.m < K ? o.m : K;
    if (o.m >= K) {
      thr_key = o.kth;
      exact = true;
      const uint32_t ov = (uint32_t)(o.kth >> 32);
      thr_x = monotone ? ord_f32(ov) : ord_next_up(ov);
    }
    wrows = NQ;
    cnt = NQ;
  }
};

}  // namespace fs
