// tselect.cuh -- threshold-filtered warp k-selection (fs_kselect, rows A1-A3).
//
// Contract = the paper's WarpSelect: after any prefix of the input the
// state holds the k smallest (value, index) keys seen.  The mechanism is re-cut for
// B200, where the instruction budget per streamed element is small (~35 warp
// instructions per 32 elements at 60 % of HBM peak) and shared memory is large:
//
//   * first-level filter: ONE float compare per element against the
//     current bound, exactly as in the paper; an accepted element is appended to
//     a LANE-PRIVATE queue in shared memory (slot (j, lane) -> word j*32+lane:
//     the "thread queue" of P:L218, but LCAP-deep and outside the register file),
//     with no ballot, shuffle or branch on the hot path;
//   * restore step: only when some lane's queue is nearly full (rare)
//     or at the end of the row.  The ragged queues are compacted in place and the
//     exact k-th smallest key is found by RADIX SELECTION (6-bit digits, lane-
//     private 16-bit counters in shared memory: no atomics, no bank conflicts);
//     the k winners are compacted again and the k-th key becomes the new bound.
//     No sorting network runs here: the paper's sort+merge of thread queues and
//     warp queue (Alg. 1-3) is replaced by counting, which is O(m) with a small
//     constant and a small code footprint (the unrolled networks of a k = 1024
//     queue do not fit the instruction cache, profiles/r01);
//   * output: ONE bitonic network on registers (blocked layout, 15
//     cross-lane steps for any size; power-of-two sizes with sentinel padding
//     instead of the odd-size networks of Alg. 1-2) sorts the k winners at the
//     very end of the row;
//   * the initial bound is not +inf: the first 1024 elements of the row are used
//     as a sample, and a counting bisection on them picks a value that about
//     m* = 1.25k..6k elements of the whole row are expected to pass, so a typical
//     row needs exactly one restore step.  If fewer than k elements passed, the
//     row is scanned again with the paper's adaptive bound (+inf start); the
//     result is exact either way.
//
// Every ordering decision is on the packed 64-bit key of select.cuh, so ties go
// to the lower index everywhere (reading K-1/K-7).
#pragma once

#include "select.cuh"

namespace fs {

// ---- sorting network on registers, blocked layout (element e = lane*NB + r) ----
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
__device__ __forceinline__ void local_halfcleaners(uint64_t (&B)[NB]) {
#pragma unroll
  for (int j = NB / 2; j >= 1; j >>= 1) {
#pragma unroll
    for (int r = 0; r < NB; ++r)
      if ((r & j) == 0) cmpex_up(B[r], B[r | j]);
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
    local_halfcleaners<NB>(B);
  }
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
__device__ __forceinline__ void sort_block_inl(uint64_t* base, int n) {
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

// ---- radix selection -------------------------------------------------------------
// Scratch of one warp: 2^RB bins x 32 lanes x 16-bit counters, also used as a 64-key
// staging area.  Counter of (bin d, lane l) lives in 32-bit word
// (d >> 1) * 32 + l, half (d & 1): a lane only ever touches its own words (no
// races, no atomics) and the 32 lanes of an access hit 32 different banks.
// RB = digit width: 5 bits (2 KB of counters) wherever shared memory per warp decides the
// occupancy -- also for k = 1024, where 9 resident warps per SM instead of 8 outweigh the extra
// counting passes (0.907 -> 0.839 ms at cfg2, 0.362 -> 0.306 ms on the 2^27 row); 6 bits for k = 512.
template <int RB>
constexpr int sel_scratch_bytes() { return (1 << RB) * 32 * 2; }

// One counting pass over keys[0..m): among the keys whose bits [dec, 64) equal
// those of prefix (all keys when dec >= 64), histogram the digit (key >> s) & 63
// (s >= dec - 6, so the digit covers every undecided bit above s; decided bits that
// fall into it are the same for all counted keys) and locate the digit holding the
// rank-th smallest (rank 1-based).  Returns the digit; below = keys in smaller
// digits, cnt = keys in that digit.  Warp-collective.
template <int RB>
__device__ __forceinline__ int radix_pass(const uint64_t* keys, int m, uint64_t prefix, int s, int dec,
                                          int rank, uint32_t* scratch, int& below, int& cnt) {
  const int lane = threadIdx.x & 31;
  constexpr int kRadixBins = 1 << RB;
#pragma unroll
  for (int t = 0; t < kRadixBins / 2; ++t) scratch[t * 32 + lane] = 0u;
  __syncwarp();
  uint16_t* h16 = reinterpret_cast<uint16_t*>(scratch);
  for (int i = lane; i < m; i += 32) {
    const uint64_t key = keys[i];
    const bool in = dec >= 64 || ((key ^ prefix) >> dec) == 0;
    if (in) {
      const uint32_t d = (uint32_t)(key >> s) & (kRadixBins - 1);
      uint16_t* h = h16 + ((((d >> 1) * 32 + lane) << 1) | (d & 1));
      *h = (uint16_t)(*h + 1);
    }
  }
  __syncwarp();
  // lane L owns digits 2L and 2L+1: sum word row L over the 32 source lanes (rotated: no conflicts)
  uint32_t acc = 0;
  if (lane < kRadixBins / 2) {
#pragma unroll 8
    for (int t = 0; t < 32; ++t) acc += scratch[lane * 32 + ((lane + t) & 31)];
  }
  const int c0 = (int)(acc & 0xFFFFu), c1 = (int)(acc >> 16);
  int incl = c0 + c1;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(kFull, incl, o);
    if (lane >= o) incl += v;
  }
  const int excl = incl - (c0 + c1);
  const bool mine = excl < rank && rank <= incl;
  const unsigned who = __ballot_sync(kFull, mine);
  const int src = __ffs(who) - 1;  // exactly one lane when 1 <= rank <= (keys counted)
  int d, b, c;
  if (rank <= excl + c0) {
    d = 2 * lane;
    b = excl;
    c = c0;
  } else {
    d = 2 * lane + 1;
    b = excl + c0;
    c = c1;
  }
  d = __shfl_sync(kFull, d, src);
  below = __shfl_sync(kFull, b, src);
  cnt = __shfl_sync(kFull, c, src);
  __syncwarp();
  return d;
}

// Exact rank-th smallest (1-based, 1 <= rank <= m) of the DISTINCT keys[0..m).
// diff = OR over i of (keys[i] ^ keys[0]) (bits in which the keys differ at all).
// Warp-collective; scratch = kSelScratchBytes of this warp.
template <int RB>
__device__ __noinline__ uint64_t radix_select_kth(const uint64_t* keys, int m, int rank, uint64_t diff,
                                                  uint32_t* scratch) {
  const int lane = threadIdx.x & 31;
  if (diff == 0) return keys[0];  // m == 1 (keys are distinct)
  const int top = 63 - __clzll((long long)diff);
  constexpr int kRadixBits = RB;
  int s = top - (kRadixBits - 1);
  if (s < 0) s = 0;
  uint64_t prefix = keys[0];  // bits above `top` are common to all keys
  prefix = (top >= 63) ? 0ull : (prefix >> (top + 1)) << (top + 1);
  int dec = 64;  // lowest decided bit; the common bits above `top` need no test
  while (true) {
    int below, cnt;
    const int d = radix_pass<RB>(keys, m, prefix, s, dec, rank, scratch, below, cnt);
    dec = s;
    rank -= below;
    prefix |= (uint64_t)d << s;
    if (s == 0) return prefix;
    if (cnt <= 64) {
      // stage the <= 64 keys of the digit, sort them, take the rank-th
      uint64_t* st = reinterpret_cast<uint64_t*>(scratch);
      int n = 0;
      for (int i0 = 0; i0 < m; i0 += 32) {
        const int i = i0 + lane;
        uint64_t key = 0;
        bool in = false;
        if (i < m) {
          key = keys[i];
          in = ((key ^ prefix) >> s) == 0;
        }
        const unsigned b = __ballot_sync(kFull, in);
        if (in) st[n + __popc(b & ((1u << lane) - 1u))] = key;
        n += __popc(b);
      }
      __syncwarp();
      sort_block<2>(st, n);
      const uint64_t r = st[swz<2>(rank - 1)];
      __syncwarp();
      return r;
    }
    s -= kRadixBits;
    if (s < 0) s = 0;
  }
}

// Per-class sizes: LCAP = depth of each lane queue (capacity 32*LCAP keys; sized for
// the mean + 4 sigma of a lane's share of the sampled bound's m*, see sample_target),
// RB = radix digit width, WARPS per CTA.
template <int NQ> struct TSelCfg;
#ifndef FS_K1_LCAP
#define FS_K1_LCAP 28
#endif
#ifndef FS_K4_LCAP
#define FS_K4_LCAP 28
#endif
template <> struct TSelCfg<1> { static constexpr int LCAP = FS_K1_LCAP, RB = 5, WARPS = 1; };
template <> struct TSelCfg<2> { static constexpr int LCAP = 32, RB = 5, WARPS = 1; };
template <> struct TSelCfg<4> { static constexpr int LCAP = FS_K4_LCAP, RB = 5, WARPS = 1; };
template <> struct TSelCfg<8> { static constexpr int LCAP = 48, RB = 5, WARPS = 1; };
template <> struct TSelCfg<16> { static constexpr int LCAP = 60, RB = 6, WARPS = 1; };
#ifndef FS_K32_LCAP
#define FS_K32_LCAP 72
#endif
#ifndef FS_K32_RB
#define FS_K32_RB 5
#endif
template <> struct TSelCfg<32> { static constexpr int LCAP = FS_K32_LCAP, RB = FS_K32_RB, WARPS = 1; };

// How many of the S sample elements the sampled bound should let through so that at
// least k of the len elements pass with ~3 sigma confidence: the count c of sample
// elements under a value has standard deviation ~sqrt(c), so c - 3 sqrt(c) >= k S/len.
__device__ __forceinline__ float sample_target(int k, int S, int64_t len) {
  const float c0 = (float)k * (float)S / (float)(len > 0 ? len : 1);
  const float r = 0.5f * (3.f + sqrtf(9.f + 4.f * c0));
  return r * r;
}

__device__ __forceinline__ float ord_next_up(uint32_t o) {
  // smallest float strictly above the value with order image o; NaN ("accept
  // everything" under !(v >= x)) when there is none
  return o >= 0xFF800000u ? __uint_as_float(0x7FFFFFFFu) : ord_f32(o + 1u);
}

struct TSelFlushOut {
  uint64_t kth;  // k-th smallest key (kSentinelKey if fewer than k survive)
  int m;         // keys kept: min(k, keys that entered the selection)
};

// Restore step.  Compacts the ragged lane queues of one warp in place (rows
// [0, wrows) hold keys already, the rest raw (bits, index) pairs), drops what the
// exact bound excludes, and selects: on return buf[0..out.m) are the k smallest
// keys (dense, unordered).  A free function taking values so that the caller's
// state stays in registers.  Warp-collective.
template <int RB>
__device__ __noinline__ TSelFlushOut tsel_flush(uint64_t* buf, uint32_t* scratch, int cnt, int wrows,
                                                uint64_t thr_key, int k) {
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  int maxc = cnt;
#pragma unroll
  for (int s = 16; s >= 1; s >>= 1) {
    const int o = __shfl_xor_sync(kFull, maxc, s);
    maxc = o > maxc ? o : maxc;
  }
  int m = 0;
  uint64_t kor = 0ull, kand = ~0ull;
  for (int j = 0; j < maxc; ++j) {
    bool valid = j < cnt;
    uint64_t key = kSentinelKey;
    if (valid) {
      const uint64_t e = buf[j * 32 + lane];
      key = j < wrows ? e : make_key(__uint_as_float((uint32_t)e), (uint32_t)(e >> 32));
      valid = key != kSentinelKey && key <= thr_key;
    }
    const unsigned b = __ballot_sync(kFull, valid);  // also orders this row's reads before the writes
    if (valid) {
      buf[m + __popc(b & lt)] = key;
      kor |= key;
      kand &= key;
    }
    m += __popc(b);
    __syncwarp();
  }
  TSelFlushOut out;
  if (m <= k) {
    out.kth = (m == k && m > 0) ? 0ull : kSentinelKey;
    out.m = m;
    if (m == k && m > 0) {  // all kept: the bound is their maximum
      uint64_t mx = 0;
      for (int i = lane; i < m; i += 32) mx = umax64(mx, buf[i]);
#pragma unroll
      for (int s = 16; s >= 1; s >>= 1) mx = umax64(mx, shfl_xor64(mx, s));
      out.kth = mx;
    }
    return out;
  }
  // bits in which the keys differ at all: set in some key and clear in some key
  const uint32_t olo = __reduce_or_sync(kFull, (uint32_t)kor), ohi = __reduce_or_sync(kFull, (uint32_t)(kor >> 32));
  const uint32_t alo = __reduce_and_sync(kFull, (uint32_t)kand), ahi = __reduce_and_sync(kFull, (uint32_t)(kand >> 32));
  const uint64_t diff = (((uint64_t)ohi << 32) | olo) & ~(((uint64_t)ahi << 32) | alo);
  const uint64_t kth = radix_select_kth<RB>(buf, m, k, diff, scratch);
  // keep the keys <= kth (exactly k of them: keys are distinct)
  int w = 0;
  for (int i0 = 0; i0 < m; i0 += 32) {
    const int i = i0 + lane;
    uint64_t key = 0;
    bool keep = false;
    if (i < m) {
      key = buf[i];
      keep = key <= kth;
    }
    const unsigned b = __ballot_sync(kFull, keep);
    if (keep) buf[w + __popc(b & lt)] = key;
    w += __popc(b);
    __syncwarp();
  }
  out.kth = kth;
  out.m = w;
  return out;
}

template <int NQ>
struct TSel {
  static constexpr int LCAP = TSelCfg<NQ>::LCAP;

  uint64_t* buf;      // this warp's 32*LCAP slots
  uint32_t* scratch;  // this warp's sel_scratch_bytes<RB>()
  uint64_t thr_key;   // exact bound once `exact`; kSentinelKey before
  float thr_x;        // an element enters iff !(v >= thr_x)
  int cnt;            // entries in this lane's queue (rows [0, wrows) are shared, see flush)
  int wrows;          // rows that already hold keys (the current top-k)
  int total;          // valid keys after the last flush (<= k)
  int k;
  int lane;
  bool exact;         // thr_key is the k-th smallest key of everything seen so far

  __device__ __forceinline__ void init(uint64_t* b, uint32_t* sc, int lane_, int k_) {
    buf = b;
    scratch = sc;
    lane = lane_;
    k = k_;
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
  __device__ __forceinline__ void push_raw(float v, uint32_t idx) {  // caller checked the bound and the room
    buf[cnt * 32 + lane] = ((uint64_t)idx << 32) | __float_as_uint(v);
    ++cnt;
  }
  // room for `need` more entries in every lane?
  __device__ __forceinline__ bool crowded(int need) const { return __any_sync(kFull, cnt > LCAP - need); }

  // Restore step.  monotone: every future element has a larger index than all
  // elements seen so far, so ties with the bound can never win (strict bound).
  __device__ __forceinline__ void flush(bool monotone) {
    const TSelFlushOut o = tsel_flush<TSelCfg<NQ>::RB>(buf, scratch, cnt, wrows, thr_key, k);
    total = o.m;
    if (o.m >= k) {
      thr_key = o.kth;
      exact = true;
      const uint32_t ov = (uint32_t)(o.kth >> 32);
      thr_x = monotone ? ord_f32(ov) : ord_next_up(ov);
    }
    // the kept keys occupy rows [0, wrows); pad the last row with sentinels
    wrows = (o.m + 31) >> 5;
    if (wrows * 32 - 32 + lane >= o.m && wrows > 0) buf[(wrows - 1) * 32 + lane] = kSentinelKey;
    cnt = wrows;
    __syncwarp();
  }
};

}  // namespace fs
