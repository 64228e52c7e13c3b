// kselect_row.cu -- fs_kselect for k >= 2: one CTA per row, counting selection.
//
// The contract is the paper's (WarpSelect P:L210-248): the k smallest (value, index) keys of
// every row, ascending, ties by lower index, bit-exact.  The mechanism is cut for B200, where a row of
// 16 384 floats has a budget of a few thousand issue slots per SM at 60 % of the HBM rate:
//
//   A1  a producer warp streams the 16-byte aligned body of the row through a ring of 16 KB stages with
//       cp.async.bulk (TMA bulk copy, mbarrier full / empty pairs); the ring holds a whole cfg2 row and
//       runs ahead into the next rows, which the producer draws from an atomic counter.  Eight consumer
//       warps read a stage with 128-bit shared-memory loads and apply the first-level filter:
//       ONE float compare per element against a bound.
//   bound: not the running k-th (P:L232 restores it after every overflow) but a SAMPLED one: the first
//       2 048 elements of the row are a sample; a SCOUT warp, one row ahead of the consumers, runs a
//       counting search over it (interpolation with a bisection safeguard) for a value that c sample
//       elements pass, with c - 3 sqrt(c) >= k S / n, so that >= k elements of the row pass with ~3 sigma
//       confidence and ~k + 3.3 sqrt(k n / S) are expected to (1 333 for k = 1 024, n = 16 384).
//   A2/A3  the survivors (appended to a dense shared-memory array of raw entries, one atomic per lane that
//       holds any) are ordered by COUNTING,
//       not by merge networks (Alg. 1-3): a monotone linear map sends the values between the sample
//       minimum and the bound to 2 048 buckets (1 024 for k <= 256); one shared-memory atomic per survivor gives the bucket
//       histogram and the survivor's slot in its bucket, one block-wide exclusive scan gives the bucket
//       starts and the bucket that holds rank k, a scatter groups the keys by bucket, and every key of a
//       bucket at or under that one counts the keys of ITS bucket that are smaller (buckets hold ~0.7
//       keys on average): rank = bucket start + that count, exact whatever the distribution, ties on the
//       full 64-bit (value, index) key.  Keys of rank < k go straight to their place in the output.
//       Skewed buckets (heavy ties) switch to a block-wide bitonic sort of the kept keys.
//   exactness: if the sampled bound lets fewer than k elements through, or more than the candidate slots
//       (a head of the row that does not represent it: sorted rows, runs of equal values), the row -- still
//       in L2 -- gets a second look: a STRIDED sample of it is searched the same way and the row filtered
//       again with that bound (loads batched eight per thread); failing that, two passes with the first
//       bound rescaled by what was counted; failing that, the paper's own scheme -- chunks of the row merged
//       into a running top-k with the exact k-th key as the bound -- using the same counting step as the
//       restore operation.  Rare (5 - 15 of cfg2's 10 000 rows take the second look), exact.
//   A4  long rows (few rows, n >= 2^18): a 65 536-element strided sample gives a 4-sigma bound
//       (kselect_sample_kernel), the whole row is streamed once by every SM with that bound and the
//       few survivors (~40 k of 2^27) are appended to a per-row list (kselect_filter_kernel), which this
//       file's row kernel then selects from as if it were a row (values + original indices).
#include <cmath>

#include "common.cuh"
#include "select.cuh"
#include "sm100.cuh"

namespace fs {
namespace {

using namespace sm100;

constexpr int RW = 8;                // consumer warps
constexpr int RT = RW * 32;          // consumer threads
constexpr int RTHREADS = RT + 64;    // + producer warp + scout warp
constexpr int RANK_MAX_BUCKET = 512;  // larger buckets among the kept ones -> bitonic sort instead (in-bucket counting is
                                      // c^2 / 256 compares per thread: ~8 us at c = 256, the block-wide sort ~100 us)

// Capacity class: CAPT candidate slots and buckets per row, NST ring stages, CTAs per SM.
// AL ("aliased"): the counting step's arrays (grouped keys, histogram, slots) live in the last HOLD ring
// stages of the row itself -- the consumers have filtered them and simply do not hand them back to the
// producer until the row's selection is done -- so the shared memory they took goes to the ring: the
// k <= 1 024 class streams through 16 KB stages like the k <= 256 class instead of 8 KB ones (cfg2 k = 1 024:
// 0.272 -> 0.258 ms).  The k <= 256 class keeps arrays of its own: a fourth 16 KB stage bought this way made
// it 1 - 3 % slower (the ring is already deep enough; the held stage delays the next row's prefetch).
template <int CAPT, bool AL> struct RowCfg;
template <> struct RowCfg<1024, false> { static constexpr int SEG = 4096, NST = 3, CTAS = 3, HOLD = 0; };  // k <= 256: 72 KB
template <> struct RowCfg<2048, false> {  // k <= 1 024, rows of fewer than two 16 KB stages: 8 KB stages, 72 KB
  static constexpr int SEG = 2048, NST = 3, CTAS = 3, HOLD = 0;
};
template <> struct RowCfg<4096, false> { static constexpr int SEG = 4096, NST = 4, CTAS = 1, HOLD = 0; };  // survivor lists: 160 KB
template <> struct RowCfg<2048, true> { static constexpr int SEG = 4096, NST = 3, CTAS = 3, HOLD = 2; };   // 65 KB

struct RowArgs {
  const float* vals;      // [n_rows][ld] values to select from
  int64_t n_rows, n, ld;
  int k;
  const unsigned int* len;  // per-row length (long rows: survivors of the filter pass) or NULL: n
  const unsigned int* len_nan;  // with len: how many of them are NaN (they pass every bound)
  int64_t len_cap;          // rows with len[row] > len_cap or < min(k, n_orig) take the exact slow path on orig
  const uint32_t* map;      // [n_rows][ld] index of vals[row][i] in the original row, or NULL: i
  const float* orig;        // original rows (ties of +-0 / NaN re-read their bits here; slow path of mapped rows)
  int64_t n_orig, orig_ld;
  float* out_val;           // [n_rows][k]
  int32_t* out_idx;
  unsigned int* work;       // row counter of the persistent CTAs (zero before the launch)
  int largest;              // 1: the k LARGEST ("other comparators"): the kernels select on -v
};

struct StageDesc {
  int64_t row;   // -1: no more rows
  int64_t len;   // elements of the row
  int seg;       // stage number inside the row
  int nseg;      // stages of the row
  int cnt;       // floats in the stage (multiple of 4)
  int last;      // last stage of the row
  int fallback;  // mapped row whose list is unusable: slow path on the original row
};

struct RowBound {
  float thr_x;       // an element enters iff !(v >= thr_x); NaN: everything enters
  float lo, hi;      // value range of the counting map (sample minimum, inclusive bound)
  int sampled;
};

struct RowSharedBase {       // what the selection steps use
  RowBound fb;               // bound of a row's second look (strided sample)
  RowBound cur;              // the bound of the row the consumers are on, and its length: parked here from row
  long long cur_len;         // begin to row end instead of riding through the stages in five registers
  unsigned int redu[2][RW];
  int cnt, ovf;              // candidates appended, overflow flag
  int kb, kept, maxc;        // counting step: boundary bucket, keys in buckets <= kb, largest such bucket
  int nan_cnt;               // counting step: NaN keys among the candidates (counted only when rank k is in their bucket)
  unsigned long long thr_key;  // slow path: exact k-th key so far
  int wsum[RW];
};
template <int NST>
struct RowShared : RowSharedBase {  // + the ring's barriers and stage records
  uint64_t full[NST], empty[NST], bnd[NST];
  StageDesc desc[NST];
  RowBound bound[NST];
};

template <int CAPT, bool AL>
struct RowSmem {
  static constexpr int NST = RowCfg<CAPT, AL>::NST, SEG = RowCfg<CAPT, AL>::SEG, HOLD = RowCfg<CAPT, AL>::HOLD;
  static constexpr size_t cand = (size_t)CAPT * sizeof(uint64_t);
  static constexpr size_t hist = (size_t)(CAPT + 8) * sizeof(uint32_t);
  static constexpr size_t bs = (size_t)CAPT * sizeof(uint32_t);
  // a stage of the aliased classes has 128 bytes behind its data: the histogram is CAPT + 8 words
  static constexpr size_t stride = (size_t)SEG * sizeof(float) + (AL ? 128 : 0);
  static constexpr size_t ring = (size_t)NST * stride;
  static constexpr size_t o_cand = ring, o_sorted = o_cand + cand, o_hist = o_sorted + cand, o_bs = o_hist + hist,
                          o_sh = AL ? o_cand + cand : o_bs + bs;
  static constexpr size_t total = o_sh + sizeof(RowShared<NST>) + 128;
  // aliased: grouped keys | histogram | slots in one held stage (HOLD = 1), or keys in the stage before the
  // last and histogram | slots in the last (HOLD = 2)
  static constexpr size_t a_hist = HOLD == 1 ? cand : 0, a_bs = a_hist + hist;
  static_assert(!AL || (a_bs + bs <= stride && cand <= stride), "the counting arrays must fit the held stages");
  static_assert(a_bs % 16 == 0 && stride % 128 == 0, "alignment");
};

// mbarrier wait of the producer and scout warps: the blocking try_wait form.  (A test_wait + nanosleep poll
// was measured too: nanosleep(300) returns almost at once, the two warps then issue 18 % of the kernel's
// instructions, and the calls are 1 - 2 % slower; nanosleep(3000) delays the refills and costs 70 %.  The
// polls are 17 % of the issued instructions -- YIELD / TRYWAIT / BRA every ~25 clocks -- but take no slot a
// working warp wants: try_wait with a suspend-time hint of 2 / 20 us (ptxas: NANOSLEEP.SYNCS between polls)
// removes them and changes no call's time, profiles/r02_kselect.md.)
__device__ __forceinline__ void mbar_wait_park(uint64_t* bar, uint32_t parity) { mbar_wait(bar, parity); }

// The k-largest variant runs the same selection on the negated values (-v < -w <=> v > w; f32_ord folds
// +-0 and NaN, so NaN still sorts last and ties still go to the lower index).  LG is the kernels'
// compile-time switch for the streaming loads, sg the run-time sign mask of the rarely taken paths.
template <bool LG> __device__ __forceinline__ float fl(float v) { return LG ? -v : v; }
__device__ __forceinline__ float flip(float v, uint32_t sg) { return __uint_as_float(__float_as_uint(v) ^ sg); }
template <bool LG> __device__ __forceinline__ float4 ldn4(const float4* p) {
  const float4 x = *p;
  return make_float4(fl<LG>(x.x), fl<LG>(x.y), fl<LG>(x.z), fl<LG>(x.w));
}

__device__ __forceinline__ void cbar() { asm volatile("bar.sync 1, %0;" ::"n"(RT) : "memory"); }

// bucket of a value under the monotone map value -> [0, NBK): non-decreasing in the key order for any lo and
// any scale >= 0 (FADD, FMUL by a non-negative number, FMNMX and F2I are monotone); NaN -- the value itself or
// inf * 0 -- comes out of fminf as NBK - 1 (NaN sorts last); -0 and +0 share a bucket
template <int NBK>
__device__ __forceinline__ int bucket_of_val(float v, float lo, float scale) {
  const float t = fminf((v - lo) * scale, (float)(NBK - 1));
  const int b = __float2int_rz(t);
  return b < 0 ? 0 : b;
}
// the same bucket from a key: its order image gives the value back (up to -0 -> +0 and the NaN payload)
template <int NBK>
__device__ __forceinline__ int bucket_of(uint64_t key, float lo, float scale) {
  return bucket_of_val<NBK>(ord_f32((uint32_t)(key >> 32)), lo, scale);
}

template <int CAPT>
struct RowCtx {
  const RowArgs* a;
  float* ring;
  uint64_t* cand;
  uint64_t* sorted;
  uint32_t* hist;
  uint32_t* bs;
  RowSharedBase* s;
  int tid, warp, lane;
};

template <int CAPT>
__device__ __forceinline__ void emit_out(const RowCtx<CAPT>& c, int64_t row, int r, uint64_t key) {
  const RowArgs& a = *c.a;
  const uint32_t idx = key_idx(key), o = (uint32_t)(key >> 32);
  // the value is rebuilt from the order image except for the two images that are not injective
  // (+-0 and NaN), which are re-read from the row (original bits, A3)
  const float v = (o == 0x80000000u || o == 0xFFFFFFFFu) ? a.orig[row * a.orig_ld + idx]
                                                        : flip(ord_f32(o), a.largest ? 0x80000000u : 0u);
  a.out_val[row * a.k + r] = v;
  a.out_idx[row * a.k + r] = (int32_t)idx;
}

// Block-wide bitonic sort of sorted[0..n2) (n2 a power of two <= CAPT), ascending.
template <int CAPT>
__device__ void block_bitonic(const RowCtx<CAPT>& c, int n2) {
  for (int sz = 2; sz <= n2; sz <<= 1) {
    for (int j = sz >> 1; j >= 1; j >>= 1) {
      for (int t = c.tid; t < (n2 >> 1); t += RT) {
        const int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));
        const int hi = lo | j;
        const bool asc = (lo & sz) == 0;
        const uint64_t x = c.sorted[lo], y = c.sorted[hi];
        if ((x > y) == asc) {
          c.sorted[lo] = y;
          c.sorted[hi] = x;
        }
      }
      cbar();
    }
  }
}

// The counting step over cand[0..m): ranks the keys and either writes the `want` smallest to the
// output of `row` (padding up to k) or, RESTORE, leaves them in cand[0..want) in ascending order and
// publishes the want-th smallest in s->thr_key.  RAW: cand holds (index << 32 | value bits) as the
// filter wrote them (position in vals, translated through mp when the row is a survivor list);
// otherwise keys.  lo / hi: value range of the map (have_range), else taken from the candidates.
// The histogram must be zero on entry and is left dirty.  All consumer threads; ends with a barrier.
// bounded: the candidates are what a bound let through, not the whole row.  NaN passes every bound (the
// filters test "less than or unordered"), so m >= want does not yet mean that the `want` smallest keys of the
// ROW are among the candidates: if fewer than `want` of them are real values, elements above the bound would
// have come before the NaNs.  The step then returns false before it writes anything (the caller goes on to
// its next, wider method); the check costs nothing unless rank `want` falls into the bucket NaN lives in.
template <int CAPT, bool RESTORE, bool RAW>
__device__ bool count_select(const RowCtx<CAPT>& c, int64_t row, int m, int want, bool have_range, float lo, float hi,
                             const uint32_t* mp, bool bounded = false) {
  constexpr int NBK = CAPT, BPT = NBK / RT;  // buckets per thread in the scan
  auto* s = c.s;
  const int tid = c.tid, lane = c.lane, warp = c.warp;
  if (tid == 0) {
    s->kb = NBK - 1;
    s->kept = m;
    s->maxc = 0;
    s->nan_cnt = 0;
  }
  // The passes below are issue-bound, not latency-bound (three CTAs per SM overlap them): U > 1 keys per
  // thread in flight was measured 7 % (U = 2) and 27 % (U = 4) slower at k = 1 024.
  constexpr int U = 1;
  const bool raw = RAW && have_range;  // raw entries become keys inside the histogram pass
  if (RAW && !have_range) {            // no range given: keys first (the range is taken from them)
    for (int i = tid; i < m; i += RT) {
      const uint64_t e = c.cand[i];
      const uint32_t pos = (uint32_t)(e >> 32);
      c.cand[i] = make_key(__uint_as_float((uint32_t)e), mp ? mp[pos] : pos);
    }
  }
  if (!have_range) {  // range of the candidates' order images (NaN image left out of the maximum)
    uint32_t mn = 0xFFFFFFFFu, mx = 0u;
    for (int i = tid; i < m; i += RT) {
      const uint32_t o = (uint32_t)(c.cand[i] >> 32);
      mn = o < mn ? o : mn;
      if (o != 0xFFFFFFFFu) mx = o > mx ? o : mx;
    }
    mn = __reduce_min_sync(kFull, mn);
    mx = __reduce_max_sync(kFull, mx);
    if (lane == 0) {
      s->redu[0][warp] = mn;
      s->redu[1][warp] = mx;
    }
    cbar();
#pragma unroll
    for (int w = 0; w < RW; ++w) {
      mn = s->redu[0][w] < mn ? s->redu[0][w] : mn;
      mx = s->redu[1][w] > mx ? s->redu[1][w] : mx;
    }
    lo = ord_f32(mn);
    hi = ord_f32(mx);
  }
  const float span = hi - lo;
  const float scale = (span > 0.f && span < 3.0e38f) ? (float)NBK / span : 0.f;
  // 1. histogram: one shared-memory atomic per key gives the bucket count and the key's slot
  for (int i0 = tid; i0 < m; i0 += U * RT) {
    uint64_t key[U];
    int bk[U];
    unsigned int slot[U];
#pragma unroll
    for (int u = 0; u < U; ++u) key[u] = i0 + u * RT < m ? c.cand[i0 + u * RT] : 0ull;
    if (RAW && raw) {  // the raw entry still has the value's own bits: bucket from them, then the key
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const uint32_t pos = (uint32_t)(key[u] >> 32);
        const uint32_t idx = (mp && i0 + u * RT < m) ? mp[pos] : pos;
        const float v = __uint_as_float((uint32_t)key[u]);
        bk[u] = bucket_of_val<NBK>(v, lo, scale);
        key[u] = make_key(v, idx);
      }
    } else {
#pragma unroll
      for (int u = 0; u < U; ++u) bk[u] = bucket_of<NBK>(key[u], lo, scale);
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (i0 + u * RT < m) slot[u] = atomicAdd(&c.hist[bk[u]], 1u);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (i0 + u * RT < m) {
        if (RAW && raw) c.cand[i0 + u * RT] = key[u];
        c.bs[i0 + u * RT] = (uint32_t)bk[u] | (slot[u] << 12);
      }
    }
  }
  cbar();
  // 2. exclusive scan of the counts (BPT per thread), boundary bucket, largest kept bucket
  {
    unsigned int cn[BPT], ex[BPT], run = 0;
#pragma unroll
    for (int q = 0; q < BPT / 4; ++q) {
      const uint4 p = reinterpret_cast<const uint4*>(c.hist)[(BPT / 4) * tid + q];
      cn[4 * q] = p.x;
      cn[4 * q + 1] = p.y;
      cn[4 * q + 2] = p.z;
      cn[4 * q + 3] = p.w;
    }
#pragma unroll
    for (int j = 0; j < BPT; ++j) {
      ex[j] = run;
      run += cn[j];
    }
    unsigned int incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int v = __shfl_up_sync(kFull, incl, o);
      if (lane >= o) incl += v;
    }
    if (lane == 31) s->wsum[warp] = (int)incl;
    cbar();
    unsigned int base = incl - run;
#pragma unroll
    for (int w = 0; w < RW; ++w)
      if (w < warp) base += (unsigned int)s->wsum[w];
    unsigned int mxc = 0;
#pragma unroll
    for (int j = 0; j < BPT; ++j) {
      ex[j] += base;
      if ((int)ex[j] < want) {
        mxc = cn[j] > mxc ? cn[j] : mxc;
        if ((int)(ex[j] + cn[j]) >= want) {  // rank want-1 lives here
          s->kb = tid * BPT + j;
          s->kept = (int)(ex[j] + cn[j]);
        }
      }
    }
#pragma unroll
    for (int q = 0; q < BPT / 4; ++q)
      reinterpret_cast<uint4*>(c.hist)[(BPT / 4) * tid + q] = make_uint4(ex[4 * q], ex[4 * q + 1], ex[4 * q + 2], ex[4 * q + 3]);
    if (tid == RT - 1) c.hist[NBK] = base + run;  // = m: end of the last bucket
    mxc = __reduce_max_sync(kFull, mxc);
    if (lane == 0 && mxc > 0) atomicMax(&s->maxc, (int)mxc);
  }
  cbar();
  if (bounded && s->kb == NBK - 1) {  // (uniform) rank `want` is in the last bucket: count the NaN keys
    int nn = 0;
    for (int i = tid; i < m; i += RT) nn += (uint32_t)(c.cand[i] >> 32) == 0xFFFFFFFFu ? 1 : 0;
    nn = __reduce_add_sync(kFull, nn);
    if (lane == 0 && nn) atomicAdd(&s->nan_cnt, nn);
    cbar();
    if (m - s->nan_cnt < want) return false;
  }
  // 3. scatter the keys of the buckets up to the boundary one, grouped by bucket
  const int kb = s->kb, kept = s->kept;
  for (int i0 = tid; i0 < m; i0 += U * RT) {
    uint32_t e[U], h[U];
    uint64_t key[U];
    bool ok[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const bool in = i0 + u * RT < m;
      e[u] = in ? c.bs[i0 + u * RT] : 0xFFFu;
      key[u] = in ? c.cand[i0 + u * RT] : 0ull;
      ok[u] = in && (int)(e[u] & 0xFFFu) <= kb;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) h[u] = ok[u] ? c.hist[e[u] & 0xFFFu] : 0u;
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (ok[u]) c.sorted[h[u] + (e[u] >> 12)] = key[u];
  }
  cbar();
  // 4. rank inside the bucket (or sort everything kept when some bucket is crowded) and emit
  if (s->maxc <= RANK_MAX_BUCKET) {
    for (int p0 = tid; p0 < kept; p0 += U * RT) {
      uint64_t key[U];
      int s0[U], cn[U], r[U], mc = 0;
#pragma unroll
      for (int u = 0; u < U; ++u) key[u] = p0 + u * RT < kept ? c.sorted[p0 + u * RT] : 0ull;
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int b = bucket_of<NBK>(key[u], lo, scale);
        const bool in = p0 + u * RT < kept;
        s0[u] = in ? (int)c.hist[b] : 0;
        cn[u] = in ? (int)c.hist[b + 1] - s0[u] : 0;
        r[u] = s0[u];
        mc = cn[u] > mc ? cn[u] : mc;
      }
      if (mc > 1) {  // a key alone in its bucket has its rank already
        for (int j = 0; j < mc; ++j) {
#pragma unroll
          for (int u = 0; u < U; ++u)
            if (j < cn[u]) r[u] += c.sorted[s0[u] + j] < key[u] ? 1 : 0;
        }
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        if (p0 + u * RT < kept && r[u] < want) {
          if (RESTORE) {
            c.cand[r[u]] = key[u];
            if (r[u] == want - 1) s->thr_key = key[u];
          } else {
            emit_out<CAPT>(c, row, r[u], key[u]);
          }
        }
      }
    }
  } else {
    int n2 = 2;
    while (n2 < kept) n2 <<= 1;
    for (int p = kept + tid; p < n2; p += RT) c.sorted[p] = kSentinelKey;
    cbar();
    block_bitonic<CAPT>(c, n2);
    for (int p = tid; p < want; p += RT) {
      const uint64_t key = c.sorted[p];
      if (RESTORE) {
        c.cand[p] = key;
        if (p == want - 1) s->thr_key = key;
      } else {
        emit_out<CAPT>(c, row, p, key);
      }
    }
  }
  if (!RESTORE) {
    const RowArgs& a = *c.a;
    for (int r = want + tid; r < a.k; r += RT) {  // fewer than k elements: (+inf, -1) padding
      a.out_val[row * a.k + r] = __uint_as_float(a.largest ? 0xFF800000u : 0x7F800000u);
      a.out_idx[row * a.k + r] = -1;
    }
  }
  cbar();
  return true;
}

template <int CAPT>
__device__ __forceinline__ void zero_hist(const RowCtx<CAPT>& c) {
  uint4* h4 = reinterpret_cast<uint4*>(c.hist);
#pragma unroll
  for (int i = 0; i < CAPT / (4 * RT); ++i) h4[i * RT + c.tid] = make_uint4(0, 0, 0, 0);
  if (c.tid < 2) h4[CAPT / 4 + c.tid] = make_uint4(0, 0, 0, 0);
}

// Second look at a row whose sampled bound let the wrong number of elements through: the row (still in
// L2) is filtered again against thr_x (an element enters iff !(v >= thr_x)) into raw entries.  s->cnt
// holds the number that passed (entries beyond CAPT are not stored); the caller decides what follows.
template <int CAPT>
__device__ void refilter_row(const RowCtx<CAPT>& c, const float* src, int64_t len, float thr_x) {
  auto* s = c.s;
  if (c.tid == 0) s->cnt = 0;
  cbar();
  const unsigned lt = (1u << c.lane) - 1u;
  const uint32_t sg = c.a->largest ? 0x80000000u : 0u;
  constexpr int XU = 8;  // loads in flight per thread: the row comes from L2, one load at a time would cost its latency
  const int64_t nblk = (len + 32 * XU - 1) / (32 * XU);
  for (int64_t blk = c.warp; blk < nblk; blk += RW) {
    const int64_t e0 = blk * (32 * XU) + c.lane;
    float v[XU];
#pragma unroll
    for (int u = 0; u < XU; ++u) v[u] = e0 + 32 * u < len ? flip(__ldg(src + e0 + 32 * u), sg) : 0.f;
#pragma unroll
    for (int u = 0; u < XU; ++u) {
      const int64_t e = e0 + 32 * u;
      const bool pass = e < len && !(v[u] >= thr_x);
      const unsigned b = __ballot_sync(kFull, pass);
      if (b == 0u) continue;
      int base = 0;
      if (c.lane == 0) base = atomicAdd(&s->cnt, __popc(b));
      base = __shfl_sync(kFull, base, 0);
      const int pos = base + __popc(b & lt);
      if (pass && pos < CAPT) c.cand[pos] = ((uint64_t)(uint32_t)e << 32) | __float_as_uint(v[u]);
    }
  }
  cbar();
}

// Exact selection of one row by the paper's scheme: chunks of the row are merged into a
// running top-k whose k-th key is the bound for what follows; the merge is count_select<RESTORE>.
template <int CAPT>
__device__ void slow_row(const RowCtx<CAPT>& c, int64_t row, const float* src, int64_t len, const uint32_t* map) {
  auto* s = c.s;
  const RowArgs& a = *c.a;
  const int k = a.k;
  const int want_all = (int64_t)k < len ? k : (int)len;
  const uint32_t sg = a.largest ? 0x80000000u : 0u;
  zero_hist<CAPT>(c);
  if (c.tid == 0) {
    s->cnt = 0;
    s->thr_key = kSentinelKey;
  }
  cbar();
  const int64_t chunk = CAPT - k;  // k <= CAPT / 2
  if (len == 0) {
    count_select<CAPT, false, false>(c, row, 0, 0, false, 0.f, 0.f, nullptr);
    return;
  }
  for (int64_t e0 = 0; e0 < len; e0 += chunk) {
    const int64_t e1 = e0 + chunk < len ? e0 + chunk : len;
    const unsigned long long thr = s->thr_key;
    for (int64_t e = e0 + c.tid; e < e1; e += RT) {
      const uint64_t key = make_key(flip(src[e], sg), map ? map[e] : (uint32_t)e);
      if (key < thr) c.cand[atomicAdd(&s->cnt, 1)] = key;
    }
    cbar();
    const int m = s->cnt;
    if (e1 >= len) {
      count_select<CAPT, false, false>(c, row, m, m < want_all ? m : want_all, false, 0.f, 0.f, nullptr);
    } else if (m > k) {
      count_select<CAPT, true, false>(c, row, m, k, false, 0.f, 0.f, nullptr);
      zero_hist<CAPT>(c);
      if (c.tid == 0) s->cnt = k;
      cbar();
    }
  }
}

// How many of the S sample elements the sampled bound should let through so that at least k of the
// len elements pass with ~z sigma confidence: c - z sqrt(c) >= k S / len.
__device__ __forceinline__ float sample_target(float z, int k, int S, int64_t len) {
  const float c0 = (float)k * (float)S / (float)(len > 0 ? len : 1);
  const float r = 0.5f * (z + sqrtf(z * z + 4.f * c0));
  return r * r;
}

// The scout warp's job for one row: a bound from the first S = 2 048 (or 1 024) elements of the row's
// first stage, by a counting search over the sample (interpolation with a bisection safeguard).
template <int CAPT, bool LG>
__device__ __forceinline__ RowBound scout_bound(const float* st, int cnt, int64_t len, int k, int lane) {
  RowBound b;
  b.thr_x = __uint_as_float(0x7FFFFFFFu);
  b.lo = b.hi = 0.f;
  b.sampled = 0;
  // 2 048 sample elements for rows of cfg2's length (the scout's work is on the issue budget of the SM), the
  // whole first stage for long lists, whose bound needs the resolution
  const int S = (cnt >= 4096 && len > 32768) ? 4096 : (cnt >= 2048 ? 2048 : 1024);
  const float rho = sample_target(3.f, k, S, len);
  const int rho_lo = (int)rho + 1;
  int w = rho_lo >> 3;
  w = w < 8 ? 8 : w;
  const int rho_hi = rho_lo + w;  // a window of >= 8 counts is found in a few probes
  // the survivors expected at the top of the window, plus 3 sigma of the sampling error, must fit
  const float top = (float)rho_hi + 3.f * sqrtf((float)rho_hi);
  if (!(cnt >= 1024 && rho_hi < S / 2 && len > CAPT && top * (float)len <= (float)CAPT * (float)S)) return b;
  const int nq = S / 128;  // float4 per lane
  const float4* s4 = reinterpret_cast<const float4*>(st);
  float mn = __uint_as_float(0x7F800000u), mx = __uint_as_float(0xFF800000u);
  bool has_nan = false;
#pragma unroll 4
  for (int j = 0; j < nq; ++j) {
    const float4 x = ldn4<LG>(s4 + j * 32 + lane);
    mn = fminf(fminf(mn, x.x), fminf(fminf(x.y, x.z), x.w));
    mx = fmaxf(fmaxf(mx, x.x), fmaxf(fmaxf(x.y, x.z), x.w));
    has_nan |= (x.x != x.x) | (x.y != x.y) | (x.z != x.z) | (x.w != x.w);
  }
  const uint32_t omn = __reduce_min_sync(kFull, f32_ord(mn));
  uint32_t omx = __reduce_max_sync(kFull, f32_ord(mx));
  if (__any_sync(kFull, has_nan)) omx = 0xFFFFFFFFu;
  // bracket [lo, hi] in the order image with counts clo < rho_lo, chi > rho_hi; probes interpolate
  // linearly in the value domain (3 of 4 steps) or bisect the order image (every 4th: termination)
  uint32_t lo = omn > 0u ? omn - 1u : 0u, hi = omx, pick = 0xFF800000u;
  if (hi > 0xFF800000u) hi = 0xFF800000u;  // NaN in the sample: the +inf image is the widest bound
  int clo = 0, chi = S;
  const float target = 0.5f * (float)(rho_lo + rho_hi);
  if (hi <= lo) hi = lo;  // degenerate (constant sample): pick stays +inf
#pragma unroll 1
  for (int it = 0; it < 48 && hi - lo > 1u; ++it) {
    uint32_t mid = lo + ((hi - lo) >> 1);
    if ((it & 3) != 3) {
      const float vlo = ord_f32(lo), vhi = ord_f32(hi);
      const float t = vlo + (vhi - vlo) * ((target - (float)clo) / (float)(chi - clo));
      const uint32_t m2 = f32_ord(t);
      if (t == t && m2 > lo && m2 < hi) mid = m2;
    }
    const float tf = ord_f32(mid);
    int cme = 0;
    // After a few probes without a hit the distribution is probably discrete (ties): the probe then also
    // finds the sample values next to it, and the bracket snaps to them, so that runs of equal values
    // cost one probe each instead of a bisection down to one ulp.
    const bool snap = it >= 4;
    float vb = __uint_as_float(0xFF800000u), va = __uint_as_float(0x7F800000u);  // max <= tf, min > tf
    if (!snap) {
#pragma unroll 4
      for (int j = 0; j < nq; ++j) {
        const float4 x = ldn4<LG>(s4 + j * 32 + lane);
        cme += (x.x <= tf) + (x.y <= tf) + (x.z <= tf) + (x.w <= tf);
      }
    } else {
#pragma unroll 2
      for (int j = 0; j < nq; ++j) {
        const float4 x = ldn4<LG>(s4 + j * 32 + lane);
        const float e[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          if (e[t] <= tf) {
            ++cme;
            vb = fmaxf(vb, e[t]);
          } else if (e[t] == e[t]) {
            va = fminf(va, e[t]);
          }
        }
      }
    }
    const int cw = __reduce_add_sync(kFull, cme);
    uint32_t nlo = mid, nhi = mid;
    if (snap) {
      const uint32_t ob = __reduce_max_sync(kFull, f32_ord(vb)), oa = __reduce_min_sync(kFull, f32_ord(va));
      if (cw > 0 && ob <= mid) nhi = ob;                  // the count at ob is the count at mid
      if (cw < S && oa > mid && oa > 0u) nlo = oa - 1u;   // and so is the count just under oa
    }
    if (cw < rho_lo) {
      lo = nlo > lo ? nlo : lo;
      clo = cw;
    } else {
      hi = nhi < hi ? nhi : hi;
      chi = cw;
      pick = hi;
      if (cw <= rho_hi) break;
    }
  }
  if (pick == 0xFF800000u && hi < 0xFF800000u && hi > lo) pick = hi;  // window never hit: hi passes >= rho_lo
  if (pick >= 0xFF800000u) return b;  // no usable bound: the row behaves as an unsampled one
  b.thr_x = ord_f32(pick + 1u);  // inclusive bound `pick`: everything with order image <= pick passes
  b.lo = ord_f32(omn);
  b.hi = ord_f32(pick);
  b.sampled = 1;
  return b;
}

template <int CAPT, bool AL, bool LG>
__global__ void __launch_bounds__(RTHREADS, RowCfg<CAPT, AL>::CTAS) kselect_row_kernel(const RowArgs a) {
  using CF = RowCfg<CAPT, AL>;
  constexpr int NST = CF::NST, SEG = CF::SEG, HOLD = CF::HOLD, VPT = SEG / (4 * RT);  // float4 per thread and stage
  using SM = RowSmem<CAPT, AL>;
  constexpr uint32_t STRIDE = (uint32_t)SM::stride;  // bytes from one stage to the next
  extern __shared__ __align__(128) unsigned char smem_raw[];
  RowCtx<CAPT> c;
  c.a = &a;
  c.ring = reinterpret_cast<float*>(smem_raw);
  c.cand = reinterpret_cast<uint64_t*>(smem_raw + SM::o_cand);
  c.sorted = reinterpret_cast<uint64_t*>(smem_raw + SM::o_sorted);  // aliased classes: set at every row end
  c.hist = reinterpret_cast<uint32_t*>(smem_raw + SM::o_hist);
  c.bs = reinterpret_cast<uint32_t*>(smem_raw + SM::o_bs);
  auto* s = reinterpret_cast<RowShared<NST>*>(smem_raw + SM::o_sh);
  c.s = s;
  c.tid = threadIdx.x;
  c.warp = threadIdx.x >> 5;
  c.lane = threadIdx.x & 31;
  auto stage_ptr = [&](int slot) { return reinterpret_cast<float*>(smem_raw + (size_t)slot * STRIDE); };
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < NST; ++i) {
      mbar_init(&s->full[i], 1);
      mbar_init(&s->empty[i], RW + 1);
      mbar_init(&s->bnd[i], 1);
    }
    s->cnt = 0;
    s->ovf = 0;
    fence_mbar_init();
  }
  __syncthreads();

  if (c.warp == RW) {
    // ---------------- producer: rows -> ring stages ----------------
    if (c.lane != 0) return;
    uint32_t stage = 0;
    int64_t row = blockIdx.x;
    auto acquire = [&]() {
      const int slot = (int)(stage % NST);
      mbar_wait_park(&s->empty[slot], ((stage / NST) & 1u) ^ 1u);
      return slot;
    };
    while (row < a.n_rows) {
      int64_t len = a.n;
      int fallback = 0;
      if (a.len) {
        const int64_t l = (int64_t)a.len[row];
        const int64_t need = (int64_t)a.k < a.n_orig ? a.k : a.n_orig;
        // NaNs pass the long-row bound too: only the real values of the list count towards the k it must hold
        const int64_t real = l - (a.len_nan ? (int64_t)a.len_nan[row] : 0);
        if (l > a.len_cap || real < need) {
          fallback = 1;
          len = 0;
        } else {
          len = l;
        }
      }
      const float* p = a.vals + row * a.ld;
      int64_t head = (4 - (int64_t)(((uintptr_t)p >> 2) & 3)) & 3;
      if (head > len) head = len;
      const int64_t body = ((len - head) >> 2) << 2;
      const int64_t nseg = body > 0 ? (body + SEG - 1) / SEG : 1;
      for (int64_t seg = 0; seg < nseg; ++seg) {
        const int slot = acquire();
        const int64_t left = body - seg * SEG;
        const int cnt = (int)(left < SEG ? left : SEG);
        StageDesc& d = s->desc[slot];
        d.row = row;
        d.len = len;
        d.seg = (int)seg;
        d.nseg = (int)nseg;
        d.cnt = cnt;
        d.last = seg == nseg - 1;
        d.fallback = fallback;
        if (cnt > 0) {
          mbar_expect_tx(&s->full[slot], (uint32_t)cnt * 4u);
          bulk_load(stage_ptr(slot), p + head + seg * SEG, (uint32_t)cnt * 4u, &s->full[slot]);
        } else {
          mbar_arrive(&s->full[slot]);
        }
        ++stage;
      }
      row = (int64_t)atomicAdd(a.work, 1u) + gridDim.x;
    }
    const int slot = acquire();
    s->desc[slot].row = -1;
    mbar_arrive(&s->full[slot]);
    return;
  }

  if (c.warp == RW + 1) {
    // ---------------- scout: the bound of every row, ahead of the consumers ----------------
    uint32_t stage = 0;
    for (;;) {
      const int slot = (int)(stage % NST);
      mbar_wait_park(&s->full[slot], (stage / NST) & 1u);
      const int64_t row = s->desc[slot].row;
      if (row < 0) break;
      if (s->desc[slot].seg == 0) {
        const RowBound b = scout_bound<CAPT, LG>(stage_ptr(slot), s->desc[slot].cnt, s->desc[slot].len, a.k, c.lane);
        if (c.lane == 0) s->bound[slot] = b;
      }
      __syncwarp();
      if (c.lane == 0) {
        mbar_arrive(&s->bnd[slot]);    // every stage, so that its phases run with the ring's
        mbar_arrive(&s->empty[slot]);  // the scout is done reading the stage
      }
      ++stage;
    }
    return;
  }

  // ---------------- consumers ----------------
  const int tid = c.tid, lane = c.lane;
  const int k = a.k;
  const uint32_t cnt_addr = smem_addr(&s->cnt), ring_sa = smem_addr(c.ring), cand_sa = smem_addr(c.cand);
  uint32_t stage = 0;
  float row_thr = 0.f;  // the row's bound (RowBound::thr_x)
  int head = 0;
  for (;;) {
    const int slot = (int)(stage % NST);
    const uint32_t par = (stage / NST) & 1u;
    mbar_wait(&s->full[slot], par);
    const int64_t row = s->desc[slot].row;
    if (row < 0) break;
    const int seg = s->desc[slot].seg, dcnt = s->desc[slot].cnt, dlast = s->desc[slot].last, dfb = s->desc[slot].fallback;
    const bool held = AL && seg >= s->desc[slot].nseg - HOLD;  // a stage the row's counting step will use
    if (seg == 0) {
      // ---- row begin ----
      const int64_t len = s->desc[slot].len;
      const float* p = a.vals + row * a.ld;
      head = (4 - (int)(((uintptr_t)p >> 2) & 3)) & 3;
      if (head > len) head = (int)len;
      if (!AL) zero_hist<CAPT>(c);
      mbar_wait(&s->bnd[slot], par);
      const RowBound bd = s->bound[slot];
      row_thr = bd.thr_x;
      if (tid == 0) {
        s->cur = bd;
        s->cur_len = len;
      }
      // head and tail scalars around the aligned body (plain loads)
      const int64_t body = ((len - head) >> 2) << 2;
      const int64_t ntail = len - head - body;
      if (tid < head + ntail) {
        const int64_t e = tid < head ? tid : head + body + (tid - head);
        const float v = fl<LG>(p[e]);
        if (!(v >= bd.thr_x)) {
          const int pos = atomicAdd(&s->cnt, 1);
          if (pos < CAPT)
            c.cand[pos] = ((uint64_t)(uint32_t)e << 32) | __float_as_uint(v);
          else
            s->ovf = 1;
        }
      }
    }
    // ---- A1: first-level filter over this stage (4 VPT elements per thread) ----
    if (dcnt > 0) {
      const int nvec = dcnt >> 2;
      const float thr_x = fl<LG>(row_thr);  // -v < t  <=>  v > -t
      const uint32_t st_sa = ring_sa + (uint32_t)slot * STRIDE + (uint32_t)tid * 16u;
      float4 x[VPT];
      uint32_t mask = 0u;
      // pass = !(v >= bound) = "less than or unordered": one FSET and one LOP3 per element
#define FS_TEST(V, BIT)                                                                                            \
  do {                                                                                                             \
    if (LG)                                                                                                        \
      asm("{\n\t.reg .b32 t;\n\tset.gtu.u32.f32 t, %1, %2;\n\tlop3.b32 %0, t, %3, %0, 0xEA;\n\t}" : "+r"(mask) : "f"(V), \
          "f"(thr_x), "r"(BIT));                                                                                   \
    else                                                                                                           \
      asm("{\n\t.reg .b32 t;\n\tset.ltu.u32.f32 t, %1, %2;\n\tlop3.b32 %0, t, %3, %0, 0xEA;\n\t}" : "+r"(mask) : "f"(V), \
          "f"(thr_x), "r"(BIT));                                                                                   \
  } while (0)
      if (nvec == SEG / 4) {
#pragma unroll
        for (int u = 0; u < VPT; ++u) {
          asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                       : "=f"(x[u].x), "=f"(x[u].y), "=f"(x[u].z), "=f"(x[u].w)
                       : "r"(st_sa + (uint32_t)u * (RT * 16u)));
        }
#pragma unroll
        for (int u = 0; u < VPT; ++u) {
          FS_TEST(x[u].x, 1u << (4 * u));
          FS_TEST(x[u].y, 2u << (4 * u));
          FS_TEST(x[u].z, 4u << (4 * u));
          FS_TEST(x[u].w, 8u << (4 * u));
        }
      } else {
#pragma unroll
        for (int u = 0; u < VPT; ++u) {
          x[u] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (u * RT + tid < nvec) {
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                         : "=f"(x[u].x), "=f"(x[u].y), "=f"(x[u].z), "=f"(x[u].w)
                         : "r"(st_sa + (uint32_t)u * (RT * 16u)));
            FS_TEST(x[u].x, 1u << (4 * u));
            FS_TEST(x[u].y, 2u << (4 * u));
            FS_TEST(x[u].z, 4u << (4 * u));
            FS_TEST(x[u].w, 8u << (4 * u));
          }
        }
      }
#undef FS_TEST
      {
        // every lane that holds survivors reserves its own slots with one shared-memory atomic: the order of the
        // raw entries does not matter (the counting step ranks them by key), and a warp-wide prefix sum per
        // stage cost as much as the filter itself (measured: k = 32 0.170 -> 0.157 ms, k = 1 024 0.326 -> 0.308)
        if (mask != 0u) {
          const int cm = __popc(mask);
          int base;
          asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(base) : "r"(cnt_addr), "r"(cm) : "memory");
          if (base + cm > CAPT) {
            s->ovf = 1;
          } else {
            uint32_t addr = cand_sa + (uint32_t)base * 8u;
            const uint32_t ib = (uint32_t)head + (uint32_t)seg * SEG + (uint32_t)tid * 4u;
            while (mask) {
              const int j = __ffs(mask) - 1;
              mask &= mask - 1u;
              const uint32_t off = (uint32_t)(j >> 2) * (RT * 4u) + (uint32_t)(j & 3);
              uint32_t bits;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(bits) : "r"(st_sa + off * 4u));
              if (LG) bits ^= 0x80000000u;
              asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(addr), "r"(bits), "r"(ib + off) : "memory");
              addr += 8u;
            }
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0 && !held) mbar_arrive(&s->empty[slot]);
    ++stage;
    if (dlast) {
      // ---- row end: counting step, or the exact slow path ----
      cbar();
      if (AL) {  // every consumer is done with the row's stages: the held ones become the counting arrays
        unsigned char* sa = smem_raw + (size_t)slot * STRIDE;
        unsigned char* sb = smem_raw + (size_t)((slot + NST - 1) % NST) * STRIDE;
        c.sorted = reinterpret_cast<uint64_t*>(HOLD == 2 ? sb : sa);
        c.hist = reinterpret_cast<uint32_t*>(sa + SM::a_hist);
        c.bs = reinterpret_cast<uint32_t*>(sa + SM::a_bs);
        zero_hist<CAPT>(c);
        cbar();
      }
      const int m = s->cnt;
      const RowBound bd = s->cur;
      const int64_t len = s->cur_len;
      const int want = (int64_t)k < len ? k : (int)len;
      // the row's base and map again: carried through the stages they cost four registers, and the k <= 1 024
      // class with 16 KB stages then spills (44 bytes; 3 % of the cfg2 k = 1 024 call)
      const float* p = a.vals + row * a.ld;
      const uint32_t* mp = a.map ? a.map + row * a.ld : nullptr;
      bool fell_back = false;
      if constexpr (CAPT == 4096) {  // only survivor lists of long rows can be unusable as a whole
        if (dfb) {
          slow_row<CAPT>(c, row, a.orig + row * a.orig_ld, a.n_orig, nullptr);
          fell_back = true;
        }
      }
      // One counting step over what a bound let through.  It refuses (false, nothing written) when the
      // candidates hold fewer than `want` real values and NaNs -- which pass every bound -- made up the number;
      // the histogram it leaves behind is cleared before the next attempt.
      bool done = false, dirty = false;
      auto select = [&](int mm, bool have_range, float lo, float hi, bool bounded) {
        if (dirty) {
          zero_hist<CAPT>(c);
          cbar();
        }
        dirty = true;
        return count_select<CAPT, false, true>(c, row, mm, want, have_range, lo, hi, mp, bounded);
      };
      if (!fell_back && !(s->ovf || m < want || m > CAPT))
        done = select(m, bd.sampled != 0, bd.lo, bd.hi, bd.sampled != 0);
      if (!fell_back && !done) {
        // The sample (the head of the row) did not represent the row: sorted rows, runs of equal values, NaNs.
        // Second look: a STRIDED sample of the row (it is in L2) searched the same way, one more filter pass
        // with its bound; then, if the first bound spanned a range, two passes with that bound rescaled by
        // what the pass before counted; then the paper's scheme, which needs nothing from the distribution.
        {
          const int S2 = (CAPT >= 2048 && len > 32768) ? 4096 : 2048;  // what scout_bound takes from 2 CAPT floats
          const int64_t stride = len / S2;
          if (stride >= 2) {
            float* smp = reinterpret_cast<float*>(c.sorted);
            for (int i = tid; i < S2; i += RT) smp[i] = __ldg(p + (int64_t)i * stride);
            cbar();
            if (c.warp == 0) {
              const RowBound b2 = scout_bound<CAPT, LG>(smp, S2, len, k, lane);
              if (lane == 0) s->fb = b2;
            }
            cbar();
            const RowBound b2 = s->fb;
            if (b2.sampled) {
              refilter_row<CAPT>(c, p, len, b2.thr_x);
              const int m2 = s->cnt;
              if (m2 >= want && m2 <= CAPT) done = select(m2, true, b2.lo, b2.hi, true);
            }
          }
        }
        if (!done && bd.sampled && bd.hi > bd.lo) {
          float hi = bd.hi;
          int seen = m;
          for (int attempt = 0; attempt < 2 && !done; ++attempt) {
            float f = 1.3f * (float)want / (float)(seen > 0 ? seen : 1);
            f = f > 16.f ? 16.f : f;
            hi = bd.lo + (hi - bd.lo) * f;  // along the line through (lo, 0) and (hi, seen)
            refilter_row<CAPT>(c, p, len, ord_f32(f32_ord(hi) + 1u));
            seen = s->cnt;
            if (seen >= want && seen <= CAPT) done = select(seen, false, 0.f, 0.f, true);
          }
        }
        if (!done) slow_row<CAPT>(c, row, p, len, mp);
      }
      if (tid == 0) {
        s->cnt = 0;
        s->ovf = 0;
      }
      cbar();
      if (AL && lane == 0) {  // the held stages go back to the producer
        mbar_arrive(&s->empty[slot]);
        if (HOLD == 2) mbar_arrive(&s->empty[(slot + NST - 1) % NST]);
      }
    }
  }
}

// ---------------------------------------------------------------------------
// A4: long rows.  Step 1: bound from a strided sample of 65 536 elements.
// ---------------------------------------------------------------------------
constexpr int LS_PIECES = 64, LS_PIECE = 1024, LS_S = LS_PIECES * LS_PIECE;
constexpr int LS_REG = 32;  // sample values per thread kept in registers; the rest in shared memory ([j][tid])
constexpr size_t kSampleSmem = (size_t)(LS_PIECES - LS_REG) * LS_PIECE * sizeof(float);

template <bool LG>
__global__ void __launch_bounds__(1024) kselect_sample_kernel(const float* __restrict__ rows, int64_t n, int64_t ld,
                                                               int k, float* __restrict__ thr_out) {
  extern __shared__ __align__(16) float ls_x[];  // [LS_PIECES - LS_REG][1024]
  __shared__ int red[2][32];
  __shared__ unsigned int redu[2][32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float* p = rows + (int64_t)blockIdx.x * ld;
  const int64_t stride = n / LS_PIECES;  // >= LS_PIECE: pieces do not overlap
  float x[LS_REG];
#pragma unroll
  for (int j = 0; j < LS_REG; ++j) x[j] = fl<LG>(p[j * stride + tid]);
  float mn = x[0], mx = x[0];
  bool has_nan = false;
#pragma unroll 8
  for (int j = LS_REG; j < LS_PIECES; ++j) {
    const float v = fl<LG>(p[j * stride + tid]);
    ls_x[(j - LS_REG) * LS_PIECE + tid] = v;
    mn = fminf(mn, v);
    mx = fmaxf(mx, v);
    has_nan |= v != v;
  }
#pragma unroll
  for (int j = 0; j < LS_REG; ++j) {
    mn = fminf(mn, x[j]);
    mx = fmaxf(mx, x[j]);
    has_nan |= x[j] != x[j];
  }
  uint32_t omn = __reduce_min_sync(kFull, f32_ord(mn)), omx = __reduce_max_sync(kFull, f32_ord(mx));
  const unsigned nanw = __ballot_sync(kFull, has_nan);
  if (lane == 0) {
    redu[0][warp] = omn;
    redu[1][warp] = nanw ? 0xFFFFFFFFu : omx;
  }
  __syncthreads();
  for (int w = 0; w < 32; ++w) {
    omn = redu[0][w] < omn ? redu[0][w] : omn;
    omx = redu[1][w] > omx ? redu[1][w] : omx;
  }
  const float c0 = (float)k * (float)LS_S / (float)n;
  const float r = 0.5f * (4.f + sqrtf(16.f + 4.f * c0));  // 4 sigma: a miss costs a whole-row slow path
  const int rho_lo = (int)(r * r) + 1, rho_hi = rho_lo + (rho_lo >> 3) + 2;
  uint32_t lo = omn > 0u ? omn - 1u : 0u, hi = omx, pick = 0xFF800000u;
  if (hi > 0xFF800000u) hi = 0xFF800000u;
  int clo = 0, chi = LS_S;
  const float target = 0.5f * (float)(rho_lo + rho_hi);
  if (hi <= lo) hi = lo;
#pragma unroll 1
  for (int it = 0; it < 64 && hi - lo > 1u; ++it) {
    uint32_t mid = lo + ((hi - lo) >> 1);
    if ((it & 3) != 3) {
      const float vlo = ord_f32(lo), vhi = ord_f32(hi);
      const float t = vlo + (vhi - vlo) * ((target - (float)clo) / (float)(chi - clo));
      const uint32_t m2 = f32_ord(t);
      if (t == t && m2 > lo && m2 < hi) mid = m2;
    }
    const float tf = ord_f32(mid);
    int cme = 0;
#pragma unroll
    for (int j = 0; j < LS_REG; ++j) cme += x[j] <= tf;
#pragma unroll 8
    for (int j = 0; j < LS_PIECES - LS_REG; ++j) cme += ls_x[j * LS_PIECE + tid] <= tf;
    cme = __reduce_add_sync(kFull, cme);
    if (lane == 0) red[it & 1][warp] = cme;
    __syncthreads();
    int cw = 0;
    for (int w = 0; w < 32; ++w) cw += red[it & 1][w];
    if (cw < rho_lo) {
      lo = mid;
      clo = cw;
    } else {
      hi = mid;
      chi = cw;
      pick = mid;
      if (cw <= rho_hi) break;
    }
  }
  if (pick == 0xFF800000u && hi < 0xFF800000u && hi > lo) pick = hi;
  if (tid == 0) thr_out[blockIdx.x] = pick >= 0xFF800000u ? __uint_as_float(0x7FFFFFFFu) : ord_f32(pick + 1u);
}

// Step 2: every element of the row once, against the bound; survivors (value, index) to the row's list.
__device__ __forceinline__ float4 ld_stream4(const float* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
               : "l"(p));
  return r;
}

constexpr int LF_THREADS = 256, LF_UNROLL = 8;

template <bool LG>
__global__ void __launch_bounds__(LF_THREADS) kselect_filter_kernel(const float* __restrict__ rows, int64_t n, int64_t ld,
                                                                     const float* __restrict__ thr,
                                                                     float* __restrict__ cval, uint32_t* __restrict__ cidx,
                                                                     unsigned int* __restrict__ count,
                                                                     unsigned int* __restrict__ nan_count, int64_t cap) {
  const int64_t row = blockIdx.y;
  const float* p = rows + row * ld;
  const float thr_x = thr[row];
  float* cv = cval + row * cap;
  uint32_t* ci = cidx + row * cap;
  auto take = [&](float v, int64_t e) {
    if (!(fl<LG>(v) >= thr_x)) {
      if (v != v) atomicAdd(nan_count + row, 1u);
      const unsigned int pos = atomicAdd(count + row, 1u);
      if ((int64_t)pos < cap) {
        cv[pos] = v;
        ci[pos] = (uint32_t)e;
      }
    }
  };
  int64_t head = (4 - (int64_t)(((uintptr_t)p >> 2) & 3)) & 3;
  if (head > n) head = n;
  const int64_t nvec = (n - head) >> 2;
  const float* pv = p + head;
  if (blockIdx.x == 0) {  // scalars around the aligned body
    const int64_t done = head + (nvec << 2);
    const int64_t e = threadIdx.x < head ? threadIdx.x : done + (threadIdx.x - head);
    if (threadIdx.x < head + (n - done)) take(p[e], e);
  }
  const int64_t per = (int64_t)LF_THREADS * LF_UNROLL;
  for (int64_t v0 = (int64_t)blockIdx.x * per; v0 < nvec; v0 += (int64_t)gridDim.x * per) {
    float4 x[LF_UNROLL];
    if (v0 + per <= nvec) {
#pragma unroll
      for (int u = 0; u < LF_UNROLL; ++u)
        x[u] = __ldcs(reinterpret_cast<const float4*>(pv + ((v0 + u * LF_THREADS + threadIdx.x) << 2)));
#pragma unroll
      for (int u = 0; u < LF_UNROLL; ++u) {
        const bool any = !(fl<LG>(x[u].x) >= thr_x) | !(fl<LG>(x[u].y) >= thr_x) | !(fl<LG>(x[u].z) >= thr_x) |
                         !(fl<LG>(x[u].w) >= thr_x);
        if (any) {
          const int64_t e = head + ((v0 + u * LF_THREADS + threadIdx.x) << 2);
          take(x[u].x, e);
          take(x[u].y, e + 1);
          take(x[u].z, e + 2);
          take(x[u].w, e + 3);
        }
      }
    } else {
      for (int u = 0; u < LF_UNROLL; ++u) {
        const int64_t v = v0 + u * LF_THREADS + threadIdx.x;
        if (v < nvec) {
          const float4 y = ld_stream4(pv + (v << 2));
          const int64_t e = head + (v << 2);
          take(y.x, e);
          take(y.y, e + 1);
          take(y.z, e + 2);
          take(y.w, e + 3);
        }
      }
    }
  }
}

template <int CAPT, bool AL, bool LG>
int launch_rows_t(const RowArgs& a, cudaStream_t s) {
  using SM = RowSmem<CAPT, AL>;
  static int occ_of[64] = {};  // per device: function attributes and occupancy belong to the device
  int dev = 0;
  FS_CUDA(cudaGetDevice(&dev));
  const int slot = dev >= 0 && dev < 64 ? dev : 0;
  int occ = occ_of[slot];
  if (occ == 0 || slot != dev) {
    FS_CUDA(cudaFuncSetAttribute(kselect_row_kernel<CAPT, AL, LG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::total));
    FS_CUDA(cudaFuncSetAttribute(kselect_row_kernel<CAPT, AL, LG>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 cudaSharedmemCarveoutMaxShared));
    int o = 0;
    FS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kselect_row_kernel<CAPT, AL, LG>, RTHREADS, SM::total));
    occ = o > 0 ? o : 1;
    occ_of[slot] = occ;
  }
  int64_t grid = (int64_t)sm_count() * occ;
  if (grid > a.n_rows) grid = a.n_rows;
  kselect_row_kernel<CAPT, AL, LG><<<(unsigned)grid, RTHREADS, SM::total, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
}

template <bool LG>
int launch_rows_l(const RowArgs& a, cudaStream_t s) {
  if (a.map) return launch_rows_t<4096, false, LG>(a, s);  // one CTA per long row: room for a wide window
  if (a.k <= 256) return launch_rows_t<1024, false, LG>(a, s);
  // two held stages: every row must span at least two (head and tail scalars are at most 6 elements)
  const bool two = a.n >= 2 * (int64_t)RowCfg<2048, true>::SEG;
  return two ? launch_rows_t<2048, true, LG>(a, s) : launch_rows_t<2048, false, LG>(a, s);
}

int launch_rows(const RowArgs& a, cudaStream_t s) {
  if (a.n_rows == 0) return FS_OK;
  return a.largest ? launch_rows_l<true>(a, s) : launch_rows_l<false>(a, s);
}

}  // namespace

// ---- interface to kselect.cu ----------------------------------------------------------------
constexpr int64_t kLongRowMin = 4 * (int64_t)LS_S;  // rows at least this long may take the A4 path

// survivors the long-row bound is expected to let through, with head-room; the list capacity per row
int64_t kselect_long_cap(int64_t n, int k) {
  const double c0 = (double)k * LS_S / (double)n;
  const double r = 0.5 * (4.0 + sqrt(16.0 + 4.0 * c0));
  const double expect = (r * r + 4.0) * 1.125 * (double)n / LS_S;
  int64_t cap = (int64_t)(2.0 * expect) + 8192;
  return (cap + 3) / 4 * 4;
}

bool kselect_use_long(int64_t n_rows, int64_t n, int k) {
  return k >= 2 && n >= kLongRowMin && n_rows > 0 && n_rows * 2 <= sm_count();
}

size_t kselect_rows_ws_bytes(int64_t n_rows, int64_t n, int k) {
  size_t b = 256;  // work counter
  if (kselect_use_long(n_rows, n, k)) {
    const int64_t cap = kselect_long_cap(n, k);
    b += align_up((size_t)n_rows * sizeof(float), 256) + 2 * align_up((size_t)n_rows * sizeof(unsigned int), 256) +
         align_up((size_t)n_rows * cap * sizeof(float), 256) + align_up((size_t)n_rows * cap * sizeof(uint32_t), 256);
  }
  return b;
}

// k >= 2.  ws: kselect_rows_ws_bytes.
int kselect_rows_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                        int32_t* out_idx, void* ws, cudaStream_t s, bool largest) {
  char* w = static_cast<char*>(ws);
  RowArgs a;
  a.vals = rows;
  a.n_rows = n_rows;
  a.n = n;
  a.ld = ld;
  a.k = k;
  a.len = nullptr;
  a.len_nan = nullptr;
  a.len_cap = 0;
  a.map = nullptr;
  a.orig = rows;
  a.n_orig = n;
  a.orig_ld = ld;
  a.out_val = out_val;
  a.out_idx = out_idx;
  a.work = reinterpret_cast<unsigned int*>(w);
  a.largest = largest ? 1 : 0;
  if (!kselect_use_long(n_rows, n, k)) {
    FS_CUDA(cudaMemsetAsync(w, 0, 256, s));
    return launch_rows(a, s);
  }
  const int64_t cap = kselect_long_cap(n, k);
  size_t o = 256;
  float* thr = reinterpret_cast<float*>(w + o);
  o += align_up((size_t)n_rows * sizeof(float), 256);
  unsigned int* count = reinterpret_cast<unsigned int*>(w + o);
  o += align_up((size_t)n_rows * sizeof(unsigned int), 256);
  unsigned int* nan_count = reinterpret_cast<unsigned int*>(w + o);
  o += align_up((size_t)n_rows * sizeof(unsigned int), 256);
  float* cval = reinterpret_cast<float*>(w + o);
  o += align_up((size_t)n_rows * cap * sizeof(float), 256);
  uint32_t* cidx = reinterpret_cast<uint32_t*>(w + o);
  FS_CUDA(cudaMemsetAsync(w, 0, 256 + align_up((size_t)n_rows * sizeof(float), 256) +
                                    2 * align_up((size_t)n_rows * sizeof(unsigned int), 256), s));
  auto* sample = largest ? kselect_sample_kernel<true> : kselect_sample_kernel<false>;
  FS_CUDA(cudaFuncSetAttribute(sample, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSampleSmem));  // per device
  sample<<<(unsigned)n_rows, 1024, kSampleSmem, s>>>(rows, n, ld, k, thr);
  FS_LAUNCHED();
  int64_t gx = (int64_t)sm_count() * 8 / n_rows;
  const int64_t maxg = ceil_div(n / 4, (int64_t)LF_THREADS * LF_UNROLL);
  if (gx > maxg) gx = maxg;
  if (gx < 1) gx = 1;
  auto* filter = largest ? kselect_filter_kernel<true> : kselect_filter_kernel<false>;
  filter<<<dim3((unsigned)gx, (unsigned)n_rows), LF_THREADS, 0, s>>>(rows, n, ld, thr, cval, cidx, count, nan_count, cap);
  FS_LAUNCHED();
  a.vals = cval;
  a.ld = cap;
  a.n = cap;
  a.len = count;
  a.len_nan = nan_count;
  a.len_cap = cap;
  a.map = cidx;
  return launch_rows(a, s);
}

}  // namespace fs
