// kselect_row.cu -- fs_kselect for k >= 2: one CTA per row, counting selection.
//
// The contract is the paper's (WarpSelect P:L210-248): the k smallest (value, index) keys of
// every row, ascending, ties by lower index, bit-exact.  The mechanism is cut for B200, where a row of
// 16 384 floats has a budget of a few thousand issue slots per SM at 60 % of the HBM rate:
//
//   A1  a producer warp streams the 16-byte aligned body of the row through a ring of 8 KB stages with
//       cp.async.bulk (TMA bulk copy, mbarrier full / empty pairs); the ring runs ahead into the next
//       rows, which the producer draws from an atomic counter.  Eight consumer warps read a stage with
//       128-bit shared-memory loads and apply the first-level filter: ONE float compare per
//       element against a bound.
//   bound: not the running k-th (P:L232 restores it after every overflow) but a SAMPLED one: the first
//       stage of the row is a sample of S = 2 048 elements; a counting search over it (interpolation with
//       a bisection safeguard, all 256 threads, one block barrier per probe) finds a value that c sample
//       elements pass, with c - 3 sqrt(c) >= k S / n, so that >= k elements of the row pass with ~3 sigma
//       confidence and ~k + 3.3 sqrt(k n / S) are expected to (1 333 for k = 1 024, n = 16 384).
//   A2/A3  the survivors (warp-aggregated append to a dense shared-memory array) are ordered by COUNTING,
//       not by merge networks (Alg. 1-3): a monotone linear map sends the values between the sample
//       minimum and the bound to 2 048 buckets; one shared-memory atomic per survivor gives the bucket
//       histogram and the survivor's slot in its bucket, one block-wide exclusive scan gives the bucket
//       starts and the bucket that holds rank k, a scatter groups the keys by bucket, and every key of a
//       bucket at or under that one counts the keys of ITS bucket that are smaller (buckets hold ~0.7
//       keys on average): rank = bucket start + that count, exact whatever the distribution, ties on the
//       full 64-bit (value, index) key.  Keys of rank < k go straight to their place in the output.
//       Skewed buckets (heavy ties) switch to a block-wide bitonic sort of the kept keys.
//   exactness: if the sampled bound lets fewer than k elements through, or more than the 2 048 slots
//       (a sample that does not represent the row: sorted rows), the row is done again by the paper's own
//       scheme -- chunks of the row merged into a running top-k with the exact k-th key as the bound --
//       using the same counting step as the restore operation.  Slow, rare, exact.
//   A4  long rows (few rows, n >= 2^17): a 32 768-element strided sample gives a 4-sigma bound
//       (kselect_sample_kernel), the whole row is streamed once by every SM with that bound and the
//       few survivors (~70 k of 2^27) are appended to a per-row list (kselect_filter_kernel), which this
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
constexpr int RTHREADS = RT + 32;    // + producer warp
constexpr int SEG = 2048;            // floats per ring stage (8 KB)
constexpr int CAP = 2048;            // candidate slots per row
constexpr int NBK = 2048;            // buckets of the counting step
constexpr int RANK_MAX_BUCKET = 32;  // larger buckets among the kept ones -> bitonic sort instead
#ifndef FS_KROW_STAGES
#define FS_KROW_STAGES 3
#endif
constexpr int NSTAGE = FS_KROW_STAGES;

struct RowArgs {
  const float* vals;      // [n_rows][ld] values to select from
  int64_t n_rows, n, ld;
  int k;
  const unsigned int* len;  // per-row length (long rows: survivors of the filter pass) or NULL: n
  int64_t len_cap;          // rows with len[row] > len_cap or < min(k, n_orig) take the exact slow path on orig
  const uint32_t* map;      // [n_rows][ld] index of vals[row][i] in the original row, or NULL: i
  const float* orig;        // original rows (ties of +-0 / NaN re-read their bits here; slow path of mapped rows)
  int64_t n_orig, orig_ld;
  float* out_val;           // [n_rows][k]
  int32_t* out_idx;
  unsigned int* work;       // row counter of the persistent CTAs (zero before the launch)
};

struct StageDesc {
  int64_t row;   // -1: no more rows
  int seg;       // stage number inside the row
  int cnt;       // floats in the stage (multiple of 4)
  int last;      // last stage of the row
  int fallback;  // mapped row whose list is unusable: slow path on the original row
};

struct RowShared {
  uint64_t full[NSTAGE], empty[NSTAGE];
  StageDesc desc[NSTAGE];
  int red[2][RW];
  unsigned int redu[2][RW];
  int cnt, ovf;              // candidates appended, overflow flag
  int kb, kept, maxc;        // counting step: boundary bucket, keys in buckets <= kb, largest such bucket
  unsigned long long thr_key;  // slow path: exact k-th key so far
  int wsum[RW];
};

constexpr size_t kRingBytes = (size_t)NSTAGE * SEG * sizeof(float);
constexpr size_t kCandBytes = (size_t)CAP * sizeof(uint64_t);
constexpr size_t kHistBytes = (size_t)(NBK + 8) * sizeof(uint32_t);
constexpr size_t kBsBytes = (size_t)CAP * sizeof(uint32_t);
constexpr size_t kRowSmem = kRingBytes + 2 * kCandBytes + kHistBytes + kBsBytes + sizeof(RowShared) + 128;

__device__ __forceinline__ void cbar() { asm volatile("bar.sync 1, %0;" ::"n"(RT) : "memory"); }

// bucket of a key under the monotone map value -> [0, NBK): non-decreasing in the key for any lo, scale >= 0
__device__ __forceinline__ int bucket_of(uint64_t key, float lo, float scale) {
  const uint32_t o = (uint32_t)(key >> 32);
  if (o == 0xFFFFFFFFu) return NBK - 1;  // NaN sorts last
  const float t = (ord_f32(o) - lo) * scale;
  int b = __float2int_rz(t);  // saturating; NaN -> 0
  b = b < 0 ? 0 : b;
  return b > NBK - 1 ? NBK - 1 : b;
}

struct RowCtx {
  const RowArgs* a;
  float* ring;
  uint64_t* cand;
  uint64_t* sorted;
  uint32_t* hist;
  uint32_t* bs;
  RowShared* s;
  int tid, warp, lane;
};

__device__ __forceinline__ void emit_out(const RowCtx& c, int64_t row, int r, uint64_t key) {
  const RowArgs& a = *c.a;
  const uint32_t idx = key_idx(key), o = (uint32_t)(key >> 32);
  // the value is rebuilt from the order image except for the two images that are not injective
  // (+-0 and NaN), which are re-read from the row (original bits, A3)
  const float v = (o == 0x80000000u || o == 0xFFFFFFFFu) ? a.orig[row * a.orig_ld + idx] : ord_f32(o);
  a.out_val[row * a.k + r] = v;
  a.out_idx[row * a.k + r] = (int32_t)idx;
}

// Block-wide bitonic sort of sorted[0..n2) (n2 a power of two <= CAP), ascending.
__device__ void block_bitonic(const RowCtx& c, int n2) {
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
// publishes the want-th smallest in s->thr_key.  lo / hi: value range of the map (have_range), else
// taken from the candidates.  All consumer threads; ends with a block barrier.
template <bool RESTORE>
__device__ void count_select(const RowCtx& c, int64_t row, int m, int want, bool have_range, float lo, float hi) {
  RowShared* s = c.s;
  const int tid = c.tid, lane = c.lane, warp = c.warp;
  // zero the histogram (NBK + 8 words)
  {
    uint4* h4 = reinterpret_cast<uint4*>(c.hist);
    h4[tid] = make_uint4(0, 0, 0, 0);
    h4[tid + RT] = make_uint4(0, 0, 0, 0);
    if (tid < 2) h4[2 * RT + tid] = make_uint4(0, 0, 0, 0);
    if (tid == 0) {
      s->kb = NBK - 1;
      s->kept = m;
      s->maxc = 0;
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
  } else {
    cbar();
  }
  const float span = hi - lo;
  const float scale = (span > 0.f && span < 3.0e38f) ? (float)NBK / span : 0.f;
  // 1. histogram: one shared-memory atomic per key gives the bucket count and the key's slot
  for (int i = tid; i < m; i += RT) {
    const int b = bucket_of(c.cand[i], lo, scale);
    const unsigned int slot = atomicAdd(&c.hist[b], 1u);
    c.bs[i] = (uint32_t)b | (slot << 12);
  }
  cbar();
  // 2. exclusive scan of the 2 048 counts (8 per thread), boundary bucket, largest kept bucket
  {
    uint4* h4 = reinterpret_cast<uint4*>(c.hist);
    const uint4 p = h4[2 * tid], q = h4[2 * tid + 1];
    const unsigned int cn[8] = {p.x, p.y, p.z, p.w, q.x, q.y, q.z, q.w};
    unsigned int ex[8], run = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
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
    for (int j = 0; j < 8; ++j) {
      ex[j] += base;
      if ((int)ex[j] < want) {
        mxc = cn[j] > mxc ? cn[j] : mxc;
        if ((int)(ex[j] + cn[j]) >= want) {  // rank want-1 lives here
          s->kb = tid * 8 + j;
          s->kept = (int)(ex[j] + cn[j]);
        }
      }
    }
    h4[2 * tid] = make_uint4(ex[0], ex[1], ex[2], ex[3]);
    h4[2 * tid + 1] = make_uint4(ex[4], ex[5], ex[6], ex[7]);
    if (tid == RT - 1) c.hist[NBK] = base + run;  // = m: end of the last bucket
    mxc = __reduce_max_sync(kFull, mxc);
    if (lane == 0 && mxc > 0) atomicMax(&s->maxc, (int)mxc);
  }
  cbar();
  // 3. scatter the keys of the buckets up to the boundary one, grouped by bucket
  const int kb = s->kb, kept = s->kept;
  for (int i = tid; i < m; i += RT) {
    const uint32_t e = c.bs[i];
    const int b = (int)(e & 0xFFFu);
    if (b <= kb) c.sorted[c.hist[b] + (e >> 12)] = c.cand[i];
  }
  cbar();
  // 4. rank inside the bucket (or sort everything kept when some bucket is crowded) and emit
  if (s->maxc <= RANK_MAX_BUCKET) {
    for (int p = tid; p < kept; p += RT) {
      const uint64_t key = c.sorted[p];
      const int b = bucket_of(key, lo, scale);
      const int s0 = (int)c.hist[b], e0 = (int)c.hist[b + 1];
      int r = s0;
      for (int j = s0; j < e0; ++j) r += c.sorted[j] < key ? 1 : 0;
      if (r < want) {
        if (RESTORE) {
          c.cand[r] = key;
          if (r == want - 1) s->thr_key = key;
        } else {
          emit_out(c, row, r, key);
        }
      }
    }
  } else {
    int n2 = 2;
    while (n2 < kept) n2 <<= 1;
    for (int p = kept + tid; p < n2; p += RT) c.sorted[p] = kSentinelKey;
    cbar();
    block_bitonic(c, n2);
    for (int p = tid; p < want; p += RT) {
      const uint64_t key = c.sorted[p];
      if (RESTORE) {
        c.cand[p] = key;
        if (p == want - 1) s->thr_key = key;
      } else {
        emit_out(c, row, p, key);
      }
    }
  }
  if (!RESTORE) {
    const RowArgs& a = *c.a;
    for (int r = want + tid; r < a.k; r += RT) {  // fewer than k elements: (+inf, -1) padding
      a.out_val[row * a.k + r] = __uint_as_float(0x7F800000u);
      a.out_idx[row * a.k + r] = -1;
    }
  }
  cbar();
}

// Exact selection of one row by the paper's scheme: chunks of the row are merged into a
// running top-k whose k-th key is the bound for what follows; the merge is count_select<RESTORE>.
__device__ void slow_row(const RowCtx& c, int64_t row, const float* src, int64_t len, const uint32_t* map) {
  RowShared* s = c.s;
  const RowArgs& a = *c.a;
  const int k = a.k;
  const int want_all = (int64_t)k < len ? k : (int)len;
  if (c.tid == 0) {
    s->cnt = 0;
    s->thr_key = kSentinelKey;
  }
  cbar();
  const int64_t chunk = CAP - k > 256 ? CAP - k : 256;  // k <= 1 024 < CAP
  if (len == 0) {
    count_select<false>(c, row, 0, 0, false, 0.f, 0.f);
    return;
  }
  for (int64_t e0 = 0; e0 < len; e0 += chunk) {
    const int64_t e1 = e0 + chunk < len ? e0 + chunk : len;
    const unsigned long long thr = s->thr_key;
    for (int64_t e = e0 + c.tid; e < e1; e += RT) {
      const uint64_t key = make_key(src[e], map ? map[e] : (uint32_t)e);
      if (key < thr) c.cand[atomicAdd(&s->cnt, 1)] = key;
    }
    cbar();
    const int m = s->cnt;
    if (e1 >= len) {
      count_select<false>(c, row, m, m < want_all ? m : want_all, false, 0.f, 0.f);
    } else if (m > k) {
      count_select<true>(c, row, m, k, false, 0.f, 0.f);
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

__global__ void __launch_bounds__(RTHREADS) kselect_row_kernel(const RowArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  RowCtx c;
  c.a = &a;
  c.ring = reinterpret_cast<float*>(smem_raw);
  c.cand = reinterpret_cast<uint64_t*>(smem_raw + kRingBytes);
  c.sorted = reinterpret_cast<uint64_t*>(smem_raw + kRingBytes + kCandBytes);
  c.hist = reinterpret_cast<uint32_t*>(smem_raw + kRingBytes + 2 * kCandBytes);
  c.bs = reinterpret_cast<uint32_t*>(smem_raw + kRingBytes + 2 * kCandBytes + kHistBytes);
  c.s = reinterpret_cast<RowShared*>(smem_raw + kRingBytes + 2 * kCandBytes + kHistBytes + kBsBytes);
  c.tid = threadIdx.x;
  c.warp = threadIdx.x >> 5;
  c.lane = threadIdx.x & 31;
  RowShared* s = c.s;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < NSTAGE; ++i) {
      mbar_init(&s->full[i], 1);
      mbar_init(&s->empty[i], RW);
    }
    fence_mbar_init();
  }
  __syncthreads();

  if (c.warp == RW) {
    // ---------------- producer: rows -> ring stages ----------------
    if (c.lane != 0) return;
    uint32_t stage = 0;
    int64_t row = blockIdx.x;
    auto acquire = [&]() {
      const int slot = (int)(stage % NSTAGE);
      mbar_wait(&s->empty[slot], ((stage / NSTAGE) & 1u) ^ 1u);
      return slot;
    };
    while (row < a.n_rows) {
      int64_t len = a.n;
      int fallback = 0;
      if (a.len) {
        const int64_t l = (int64_t)a.len[row];
        const int64_t need = (int64_t)a.k < a.n_orig ? a.k : a.n_orig;
        if (l > a.len_cap || l < need) {
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
        d.seg = (int)seg;
        d.cnt = cnt;
        d.last = seg == nseg - 1;
        d.fallback = fallback;
        if (cnt > 0) {
          mbar_expect_tx(&s->full[slot], (uint32_t)cnt * 4u);
          bulk_load(c.ring + (size_t)slot * SEG, p + head + seg * SEG, (uint32_t)cnt * 4u, &s->full[slot]);
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

  // ---------------- consumers ----------------
  const int tid = c.tid, lane = c.lane, warp = c.warp;
  const int k = a.k;
  uint32_t stage = 0;
  float thr_x = 0.f;     // an element enters iff !(v >= thr_x)
  float map_lo = 0.f, map_hi = 0.f;
  bool sampled = false;
  int64_t len = 0, head = 0;
  const float* p = nullptr;
  const uint32_t* mp = nullptr;
  for (;;) {
    const int slot = (int)(stage % NSTAGE);
    mbar_wait(&s->full[slot], (stage / NSTAGE) & 1u);
    const StageDesc d = s->desc[slot];
    if (d.row < 0) break;
    const int64_t row = d.row;
    const float* st = c.ring + (size_t)slot * SEG;
    if (d.seg == 0) {
      // ---- row begin: state, sampled bound ----
      len = a.len ? (d.fallback ? 0 : (int64_t)a.len[row]) : a.n;
      p = a.vals + row * a.ld;
      mp = a.map ? a.map + row * a.ld : nullptr;
      head = (4 - (int64_t)(((uintptr_t)p >> 2) & 3)) & 3;
      if (head > len) head = len;
      if (tid == 0) {
        s->cnt = 0;
        s->ovf = 0;
      }
      const int S = d.cnt >= 2048 ? 2048 : 1024;
      const float rho = sample_target(3.f, k, S, len);
      const int rho_lo = (int)rho + 1, rho_hi = rho_lo + (rho_lo >> 3) + 2;
      sampled = d.cnt >= 1024 && rho_hi < S / 2 && len > CAP;
      thr_x = __uint_as_float(0x7FFFFFFFu);  // NaN: everything passes
      if (sampled) {
        float4 x0 = reinterpret_cast<const float4*>(st)[tid];
        float4 x1 = make_float4(x0.x, x0.x, x0.x, x0.x);
        const bool two = S == 2048;
        if (two) x1 = reinterpret_cast<const float4*>(st)[tid + RT];
        float mn = fminf(fminf(fminf(x0.x, x0.y), fminf(x0.z, x0.w)), fminf(fminf(x1.x, x1.y), fminf(x1.z, x1.w)));
        float mx = fmaxf(fmaxf(fmaxf(x0.x, x0.y), fmaxf(x0.z, x0.w)), fmaxf(fmaxf(x1.x, x1.y), fmaxf(x1.z, x1.w)));
        // fminf / fmaxf drop NaN operands; a NaN anywhere in the sample is seen by the count below
        const bool has_nan = (x0.x != x0.x) | (x0.y != x0.y) | (x0.z != x0.z) | (x0.w != x0.w) | (x1.x != x1.x) |
                             (x1.y != x1.y) | (x1.z != x1.z) | (x1.w != x1.w);
        uint32_t omn = __reduce_min_sync(kFull, f32_ord(mn)), omx = __reduce_max_sync(kFull, f32_ord(mx));
        const unsigned nanw = __ballot_sync(kFull, has_nan);
        if (lane == 0) {
          s->redu[0][warp] = omn;
          s->redu[1][warp] = nanw ? 0xFFFFFFFFu : omx;
        }
        cbar();
#pragma unroll
        for (int w = 0; w < RW; ++w) {
          omn = s->redu[0][w] < omn ? s->redu[0][w] : omn;
          omx = s->redu[1][w] > omx ? s->redu[1][w] : omx;
        }
        // bracket [lo, hi] in the order image with counts clo < rho_lo, chi > rho_hi; probes interpolate
        // linearly in the value domain (3 of 4 steps) or bisect the order image (every 4th: termination)
        uint32_t lo = omn > 0u ? omn - 1u : 0u, hi = omx, pick = 0xFF800000u;
        if (hi > 0xFF800000u) hi = 0xFF800000u;  // NaN in the sample: the +inf image is the widest bound
        int clo = 0, chi = S;
        const float target = 0.5f * (float)(rho_lo + rho_hi);
        const int per = two ? 2 : 1;
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
          int cme = (x0.x <= tf) + (x0.y <= tf) + (x0.z <= tf) + (x0.w <= tf);
          if (two) cme += (x1.x <= tf) + (x1.y <= tf) + (x1.z <= tf) + (x1.w <= tf);
          cme = __reduce_add_sync(kFull, cme);
          if (lane == 0) s->red[it & 1][warp] = cme;
          cbar();
          int cw = 0;
#pragma unroll
          for (int w = 0; w < RW; ++w) cw += s->red[it & 1][w];
          (void)per;
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
        if (pick == 0xFF800000u && hi < 0xFF800000u && hi > lo) pick = hi;  // window never hit: hi passes >= rho_lo
        // inclusive bound `pick`: everything with order image <= pick passes
        thr_x = pick >= 0xFF800000u ? __uint_as_float(0x7FFFFFFFu) : ord_f32(pick + 1u);
        map_lo = ord_f32(omn);
        map_hi = ord_f32(pick);
        if (pick >= 0xFF800000u) sampled = false;  // no usable bound: behaves as an unsampled row
      }
      cbar();  // cnt / ovf reset visible; sample registers dead
      // head and tail scalars around the aligned body (plain loads)
      {
        const int64_t body = ((len - head) >> 2) << 2;
        const int64_t ntail = len - head - body;
        if (tid < head + ntail) {
          const int64_t e = tid < head ? tid : head + body + (tid - head);
          const float v = p[e];
          if (!(v >= thr_x)) {
            const int pos = atomicAdd(&s->cnt, 1);
            if (pos < CAP)
              c.cand[pos] = make_key(v, mp ? mp[e] : (uint32_t)e);
            else
              s->ovf = 1;
          }
        }
      }
    }
    // ---- A1: first-level filter over this stage ----
    if (d.cnt > 0 && !s->ovf) {
      const int nvec = d.cnt >> 2;
      const uint32_t ib = (uint32_t)(head + (int64_t)d.seg * SEG);
      uint32_t mask = 0u;
      if (nvec == SEG / 4) {
        const float4 x0 = reinterpret_cast<const float4*>(st)[tid];
        const float4 x1 = reinterpret_cast<const float4*>(st)[tid + RT];
        // the sign of (bound - v) is funnel-shifted into the mask (v equal to the bound passes the float
        // test only if it is below thr_x = next above the inclusive bound; NaN bounds pass everything)
        mask = (!(x0.x >= thr_x) ? 1u : 0u) | (!(x0.y >= thr_x) ? 2u : 0u) | (!(x0.z >= thr_x) ? 4u : 0u) |
               (!(x0.w >= thr_x) ? 8u : 0u) | (!(x1.x >= thr_x) ? 16u : 0u) | (!(x1.y >= thr_x) ? 32u : 0u) |
               (!(x1.z >= thr_x) ? 64u : 0u) | (!(x1.w >= thr_x) ? 128u : 0u);
      } else {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int f = u * RT + tid;
          if (f < nvec) {
            const float4 x = reinterpret_cast<const float4*>(st)[f];
            mask |= ((!(x.x >= thr_x) ? 1u : 0u) | (!(x.y >= thr_x) ? 2u : 0u) | (!(x.z >= thr_x) ? 4u : 0u) |
                     (!(x.w >= thr_x) ? 8u : 0u))
                    << (4 * u);
          }
        }
      }
      const int cm = __popc(mask);
      int incl = cm;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += v;
      }
      const int total = __shfl_sync(kFull, incl, 31);
      if (total > 0) {
        int base = 0;
        if (lane == 31) base = atomicAdd(&s->cnt, total);
        base = __shfl_sync(kFull, base, 31);
        if (base + total > CAP) {
          if (lane == 0) s->ovf = 1;
        } else {
          int pos = base + incl - cm;
          while (mask) {
            const int b2 = __ffs(mask) - 1;
            mask &= mask - 1u;
            const int off = ((b2 >> 2) * RT + tid) * 4 + (b2 & 3);
            const uint32_t e = ib + (uint32_t)off;
            c.cand[pos++] = make_key(st[off], mp ? mp[e] : e);
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&s->empty[slot]);
    ++stage;
    if (d.last) {
      // ---- row end: counting step, or the exact slow path ----
      cbar();
      const int m = s->cnt;
      const int want = (int64_t)k < len ? k : (int)len;
      if (d.fallback) {
        slow_row(c, row, a.orig + row * a.orig_ld, a.n_orig, nullptr);
      } else if (s->ovf || m < want) {
        slow_row(c, row, p, len, mp);
      } else {
        count_select<false>(c, row, m, want, sampled, map_lo, map_hi);
      }
    }
  }
}

// ---------------------------------------------------------------------------
// A4: long rows.  Step 1: bound from a strided sample of 32 768 elements.
// ---------------------------------------------------------------------------
constexpr int LS_PIECES = 32, LS_PIECE = 1024, LS_S = LS_PIECES * LS_PIECE;  // 32 sample values per thread stay in registers

__global__ void __launch_bounds__(1024) kselect_sample_kernel(const float* __restrict__ rows, int64_t n, int64_t ld,
                                                               int k, float* __restrict__ thr_out) {
  __shared__ int red[2][32];
  __shared__ unsigned int redu[2][32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float* p = rows + (int64_t)blockIdx.x * ld;
  const int64_t stride = n / LS_PIECES;  // >= LS_PIECE: pieces do not overlap
  float x[LS_PIECES];
#pragma unroll
  for (int j = 0; j < LS_PIECES; ++j) x[j] = p[j * stride + tid];
  float mn = x[0], mx = x[0];
  bool has_nan = false;
#pragma unroll
  for (int j = 0; j < LS_PIECES; ++j) {
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
    for (int j = 0; j < LS_PIECES; ++j) cme += x[j] <= tf;
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

__global__ void __launch_bounds__(LF_THREADS) kselect_filter_kernel(const float* __restrict__ rows, int64_t n, int64_t ld,
                                                                     const float* __restrict__ thr,
                                                                     float* __restrict__ cval, uint32_t* __restrict__ cidx,
                                                                     unsigned int* __restrict__ count, int64_t cap) {
  const int64_t row = blockIdx.y;
  const float* p = rows + row * ld;
  const float thr_x = thr[row];
  float* cv = cval + row * cap;
  uint32_t* ci = cidx + row * cap;
  auto take = [&](float v, int64_t e) {
    if (!(v >= thr_x)) {
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
      for (int u = 0; u < LF_UNROLL; ++u) x[u] = ld_stream4(pv + ((v0 + u * LF_THREADS + threadIdx.x) << 2));
#pragma unroll
      for (int u = 0; u < LF_UNROLL; ++u) {
        const bool any = !(x[u].x >= thr_x) | !(x[u].y >= thr_x) | !(x[u].z >= thr_x) | !(x[u].w >= thr_x);
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

int row_occupancy() {
  static int occ = 0;
  if (occ == 0) {
    if (cudaFuncSetAttribute(kselect_row_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowSmem) != cudaSuccess)
      return 0;
    cudaFuncSetAttribute(kselect_row_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    int o = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kselect_row_kernel, RTHREADS, kRowSmem) != cudaSuccess) return 0;
    occ = o > 0 ? o : 1;
  }
  return occ;
}

int launch_rows(const RowArgs& a, cudaStream_t s) {
  if (a.n_rows == 0) return FS_OK;
  const int occ = row_occupancy();
  if (occ == 0) return set_error(FS_ECUDA, "fs_kselect: cannot configure kselect_row_kernel");
  int64_t grid = (int64_t)sm_count() * occ;
  if (grid > a.n_rows) grid = a.n_rows;
  kselect_row_kernel<<<(unsigned)grid, RTHREADS, kRowSmem, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
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
    b += align_up((size_t)n_rows * sizeof(float), 256) + align_up((size_t)n_rows * sizeof(unsigned int), 256) +
         align_up((size_t)n_rows * cap * sizeof(float), 256) + align_up((size_t)n_rows * cap * sizeof(uint32_t), 256);
  }
  return b;
}

// k >= 2.  ws: kselect_rows_ws_bytes.
int kselect_rows_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                        int32_t* out_idx, void* ws, cudaStream_t s) {
  char* w = static_cast<char*>(ws);
  RowArgs a;
  a.vals = rows;
  a.n_rows = n_rows;
  a.n = n;
  a.ld = ld;
  a.k = k;
  a.len = nullptr;
  a.len_cap = 0;
  a.map = nullptr;
  a.orig = rows;
  a.n_orig = n;
  a.orig_ld = ld;
  a.out_val = out_val;
  a.out_idx = out_idx;
  a.work = reinterpret_cast<unsigned int*>(w);
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
  float* cval = reinterpret_cast<float*>(w + o);
  o += align_up((size_t)n_rows * cap * sizeof(float), 256);
  uint32_t* cidx = reinterpret_cast<uint32_t*>(w + o);
  FS_CUDA(cudaMemsetAsync(w, 0, 256 + align_up((size_t)n_rows * sizeof(float), 256) +
                                    align_up((size_t)n_rows * sizeof(unsigned int), 256), s));
  kselect_sample_kernel<<<(unsigned)n_rows, 1024, 0, s>>>(rows, n, ld, k, thr);
  FS_LAUNCHED();
  int64_t gx = (int64_t)sm_count() * 8 / n_rows;
  const int64_t maxg = ceil_div(n / 4, (int64_t)LF_THREADS * LF_UNROLL);
  if (gx > maxg) gx = maxg;
  if (gx < 1) gx = 1;
  kselect_filter_kernel<<<dim3((unsigned)gx, (unsigned)n_rows), LF_THREADS, 0, s>>>(rows, n, ld, thr, cval, cidx, count, cap);
  FS_LAUNCHED();
  a.vals = cval;
  a.ld = cap;
  a.n = cap;
  a.len = count;
  a.len_cap = cap;
  a.map = cidx;
  return launch_rows(a, s);
}

}  // namespace fs
