// kselect.cu -- fs_kselect: batched k-selection.
//
//   A1 stream + first-level filter   kselect_stream_kernel main loop
//   A2 restore invariants            tsel_flush in tselect.cuh
//   A3 output                        final sort + gather of the original bits
//   A4 long rows                     rows are cut into P chunks; every chunk
//                                    keeps its k smallest keys, the largest of the
//                                    chunks' j-th smallest keys (j = ceil(k/(P-1)))
//                                    bounds the row's k-th key from above, only keys
//                                    under that bound are gathered and selected again
//   A5 k = 1                         kselect_k1_kernel: min/argmin reduction
//
// One warp owns one work item (a row, or a chunk of a row).  Warps are persistent:
// warp w takes items w, w + W, ...  The 16-byte aligned body of each item reaches
// the warp through a private ring of 2 KB segments in shared memory filled by
// cp.async.bulk (the TMA bulk-copy engine) and tracked by mbarriers, so several
// segments per warp are in flight whatever the register budget, and the ring runs
// ahead across item boundaries (the next row is already arriving while the current
// one is being selected).  "Lane j reads a_{32i+j}" becomes: lane j reads
// elements 4j..4j+3 of each 128-element group with one 128-bit shared-memory load.
#include <cstdlib>
#include <mutex>

#include "common.cuh"
#include "select.cuh"
#include "tselect.cuh"

namespace fs {

struct KSelArgs {
  const float* vals;  // [n_rows][ld]
  int64_t n_rows, n, ld;
  int P;              // chunks per row
  int64_t chunk;      // elements per chunk (multiple of 4)
  int k;
  float* out_val;     // P == 1: [n_rows][k]
  int32_t* out_idx;
  uint64_t* out_keys;  // P > 1: [n_rows][P][k] keys, sentinel padded (sorted unless jth == 1)
  uint64_t* heads;     // P > 1: [n_rows][P-1][jth] the jth smallest keys of every chunk but the last
  int jth;             // ceil(k / (P - 1))
  unsigned int* work;  // item counter of the persistent warps (zero before the launch)
};

// ---- mbarrier / bulk-copy PTX --------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// global -> shared bulk copy (16-byte aligned, size a multiple of 16), completion on bar
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}

// the same on 32-bit shared-memory addresses computed once per warp
__device__ __forceinline__ void mbar_expect_tx_a(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s_a(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}

#ifndef FS_KSEG
#define FS_KSEG 512
#endif
#ifndef FS_KSTAGES
#define FS_KSTAGES 2
#endif
constexpr int kSeg = FS_KSEG;    // floats per ring segment (2 KB)
constexpr int kStages = FS_KSTAGES;   // ring depth per warp
static_assert(kSeg >= 512 && kSeg % 512 == 0, "the sampled bound reads the first 1024 elements as two ring segments");
static_assert(kStages >= 2, "the sample spans two segments");
constexpr int kSample = 1024;

struct ItemDesc {
  const float* p;   // first element of the item
  int64_t len;      // elements
  int64_t row;
  int c;            // chunk number
  uint32_t base;    // index of p[0] in the row
  int head;         // scalars before the aligned body
  int64_t nvec;     // float4 in the body
  int nseg;         // ring segments of the body
};

__device__ __forceinline__ ItemDesc decode_item(const KSelArgs& a, int64_t item) {
  ItemDesc d;
  d.row = item / a.P;
  d.c = (int)(item - d.row * a.P);
  const int64_t start = (int64_t)d.c * a.chunk;
  int64_t len = a.n - start;
  if (len > a.chunk) len = a.chunk;
  if (len < 0) len = 0;
  d.len = len;
  d.p = a.vals + d.row * a.ld + start;
  d.base = (uint32_t)start;
  int64_t head = (4 - (int)(((uintptr_t)d.p >> 2) & 3)) & 3;
  if (head > len) head = len;
  d.head = (int)head;
  d.nvec = (len - head) >> 2;
  d.nseg = (int)((d.nvec + (kSeg / 4 - 1)) / (kSeg / 4));
  return d;
}

// Per-warp ring: the producer side runs ahead of the consumer, at most into the
// item after the one being consumed.  Items are handed out dynamically (one atomic
// per item), so a late or slow warp never holds a fixed share of the work.
struct Ring {
  float* data;     // [kStages][kSeg]
  uint64_t* bar;   // [kStages]
  uint32_t data_a, bar_a;  // the same as shared-memory addresses
  uint32_t issued, consumed;
  int64_t c_item;  // item being consumed
  int64_t n_item;  // the item after it (-1: not drawn yet)
  int64_t p_item;  // item the producer is issuing (c_item or n_item)
  const float* p_ptr;  // next segment of p_item
  int p_left;          // float4 of p_item not yet issued
};

__device__ __forceinline__ int64_t draw_item(const KSelArgs& a, int64_t n_warps, int lane) {
  unsigned int t = 0;
  if (lane == 0) t = atomicAdd(a.work, 1u);
  t = __shfl_sync(kFull, t, 0);
  return (int64_t)t + n_warps;
}

__device__ __forceinline__ void ring_point(const KSelArgs& a, Ring& r, int64_t n_items) {
  r.p_left = 0;
  if (r.p_item < n_items) {
    const ItemDesc d = decode_item(a, r.p_item);
    r.p_ptr = d.p + d.head;
    r.p_left = (int)d.nvec;
  }
}

// Issue bulk copies until the ring is full or the producer may not advance.
// All lanes keep the cursor (uniform); lane 0 issues.
__device__ __forceinline__ void ring_fill(const KSelArgs& a, Ring& r, int64_t n_items, int64_t n_warps,
                                          int lane) {
  while (r.issued - r.consumed < (uint32_t)kStages) {
    if (r.p_left > 0) {
      const int slot = (int)(r.issued % kStages);
      const int n4 = r.p_left < kSeg / 4 ? r.p_left : kSeg / 4;
      if (lane == 0) {
        mbar_expect_tx_a(r.bar_a + slot * 8, (uint32_t)n4 * 16u);
        bulk_g2s_a(r.data_a + slot * (kSeg * 4), r.p_ptr, (uint32_t)n4 * 16u, r.bar_a + slot * 8);
      }
      ++r.issued;
      r.p_ptr += kSeg;
      r.p_left -= n4;
    } else if (r.p_item == r.c_item && r.c_item < n_items) {
      r.n_item = draw_item(a, n_warps, lane);
      r.p_item = r.n_item;
      ring_point(a, r, n_items);
    } else {
      break;
    }
  }
}

// ---------------------------------------------------------------------------
// General k: persistent warps, one item at a time, threshold-filtered selection.
// ---------------------------------------------------------------------------
template <int NQ>
struct StreamSmem {
  static constexpr int WARPS = TSelCfg<NQ>::WARPS;
  static constexpr int LCAP = TSelCfg<NQ>::LCAP;
  static constexpr size_t ring_bytes = (size_t)kStages * kSeg * sizeof(float);
  static constexpr size_t queue_bytes = (size_t)32 * LCAP * sizeof(uint64_t);
  static constexpr size_t scratch_bytes = sel_scratch_bytes<TSelCfg<NQ>::RB>();
  static constexpr size_t per_warp = ring_bytes + queue_bytes + scratch_bytes;
  static constexpr size_t total = per_warp * WARPS + (size_t)WARPS * kStages * sizeof(uint64_t);
};

// Writes the k winners of one item/row, sorted: values + indices (final) or keys.
template <int NQ>
__device__ __forceinline__ void write_sorted(const uint64_t* buf, int k, int lane, const float* g,
                                             float* ov, int32_t* oi) {
  // the value is rebuilt from the key's order image, except for the two images that are
  // not injective (+-0 and NaN), which are re-read from the row (original bits, A3)
  for (int i = lane; i < k; i += 32) {
    const uint64_t key = buf[swz<NQ>(i)];
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

template <int NQ>
__global__ void __launch_bounds__(TSelCfg<NQ>::WARPS * 32) kselect_stream_kernel(const KSelArgs a) {
  using SM = StreamSmem<NQ>;
  constexpr int WARPS = SM::WARPS;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  unsigned char* mine = smem_raw + (size_t)warp * SM::per_warp;
  Ring ring;
  ring.data = reinterpret_cast<float*>(mine);
  uint64_t* qbuf = reinterpret_cast<uint64_t*>(mine + SM::ring_bytes);
  uint32_t* scratch = reinterpret_cast<uint32_t*>(mine + SM::ring_bytes + SM::queue_bytes);
  ring.bar = reinterpret_cast<uint64_t*>(smem_raw + SM::per_warp * WARPS) + warp * kStages;
  ring.data_a = smem_u32(ring.data);
  ring.bar_a = smem_u32(ring.bar);
  if (lane == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) mbar_init(ring.bar + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();

  const int64_t n_items = a.n_rows * a.P;
  const int64_t n_warps = (int64_t)gridDim.x * WARPS;
  ring.issued = ring.consumed = 0;
  ring.c_item = (int64_t)blockIdx.x * WARPS + warp;
  ring.n_item = -1;
  ring.p_item = ring.c_item;
  ring_point(a, ring, n_items);
  ring_fill(a, ring, n_items, n_warps, lane);

  TSel<NQ> q;
  q.init(qbuf, scratch, lane, a.k);

  while (ring.c_item < n_items) {
    const int64_t item = ring.c_item;
    const ItemDesc d = decode_item(a, item);
    const uint32_t vbase = d.base + (uint32_t)d.head;
    const int64_t want = a.k < d.len ? a.k : d.len;
    q.reset();
    if (d.head) q.push(lane < d.head, lane < d.head ? d.p[lane] : 0.f, d.base + lane);

    // sampled bound: counting bisection in the order image over the first kSample
    // elements of the body (two ring segments): find o with rho_lo <= #(v <= o) <= rho_hi
    const float rho = sample_target(a.k, kSample, d.len);
    const int rho_lo = (int)rho + 1, rho_hi = rho_lo + (rho_lo >> 3) + 2;
    const bool sampled = d.nvec >= kSample / 4 && rho_hi < kSample / 2;
    if (sampled) {
      const int s0 = (int)(ring.consumed % kStages), s1 = (int)((ring.consumed + 1) % kStages);
      mbar_wait(ring.bar + s0, (ring.consumed / kStages) & 1u);
      mbar_wait(ring.bar + s1, ((ring.consumed + 1) / kStages) & 1u);
      float4 x[8];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        x[u] = reinterpret_cast<const float4*>(ring.data + s0 * kSeg)[u * 32 + lane];
        x[4 + u] = reinterpret_cast<const float4*>(ring.data + s1 * kSeg)[u * 32 + lane];
      }
      // bracket [lo, hi] in the order image with counts (clo < rho_lo, chi > rho_hi);
      // probes interpolate linearly in the value domain (3 of 4 steps) or bisect the
      // order image (every 4th step: guarantees termination)
      float mn = x[0].x, mx = x[0].x;
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        mn = fminf(fminf(mn, x[u].x), fminf(fminf(x[u].y, x[u].z), x[u].w));
        mx = fmaxf(fmaxf(mx, x[u].x), fmaxf(fmaxf(x[u].y, x[u].z), x[u].w));
      }
#pragma unroll
      for (int sft = 16; sft >= 1; sft >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(kFull, mn, sft));
        mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, sft));
      }
      uint32_t lo = f32_ord(mn), hi = f32_ord(mx), pick = 0xFF800000u;
      lo = lo > 0u ? lo - 1u : 0u;
      if (hi > 0xFF800000u) hi = 0xFF800000u;  // NaN in the sample: +inf image is the widest bound
      int clo = 0, chi = kSample;
      const float target = 0.5f * (float)(rho_lo + rho_hi);
      if (!(mn == mn) || !(mx == mx) || hi <= lo) hi = lo;  // degenerate: keep pick = +inf
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
#pragma unroll
        for (int u = 0; u < 8; ++u)
          cme += (x[u].x <= tf) + (x[u].y <= tf) + (x[u].z <= tf) + (x[u].w <= tf);
        const int cw = __reduce_add_sync(kFull, cme);
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
      q.set_sampled_bound(pick);
    }

    // A1: stream the body segment by segment
    const int nseg = d.nseg;
#pragma unroll 1
    for (int seg = 0; seg < nseg; ++seg) {
      const int slot = (int)(ring.consumed % kStages);
      mbar_wait_a(ring.bar_a + slot * 8, (ring.consumed / kStages) & 1u);
      const int left = (int)d.nvec - seg * (kSeg / 4);
      const float* sf = ring.data + slot * kSeg + lane * 4;
      const uint32_t ib = vbase + (uint32_t)seg * kSeg + (uint32_t)lane * 4u;
      // first-level filter: one compare per element, results in a 16-bit mask
      const float thr = q.thr_x;
      uint32_t mask = 0u;
      if (left >= kSeg / 4) {
        // the sign of (bound - v) is funnel-shifted into the mask: one subtract and one shift per
        // element (v equal to the bound and NaN pass as well: the restore step tests keys exactly)
        uint32_t rj[4];  // four independent chains (one per 128-bit load)
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const float4 x = *reinterpret_cast<const float4*>(sf + u * 128);
          rj[u] = __float_as_uint(thr - x.x) >> 31;
          rj[u] = __funnelshift_l(__float_as_uint(thr - x.y), rj[u], 1);
          rj[u] = __funnelshift_l(__float_as_uint(thr - x.z), rj[u], 1);
          rj[u] = __funnelshift_l(__float_as_uint(thr - x.w), rj[u], 1);
        }
        const uint32_t rej = (rj[0] << 12) | (rj[1] << 8) | (rj[2] << 4) | rj[3];
        mask = __brev(~rej) >> 16;  // element e = 4u + t back at bit e
      } else {
#pragma unroll 1
        for (int u = 0; u < 4; ++u) {
          if (u * 32 + lane < left) {
            const float4 x = *reinterpret_cast<const float4*>(sf + u * 128);
            mask |= ((!(x.x >= thr) ? 1u : 0u) | (!(x.y >= thr) ? 2u : 0u) | (!(x.z >= thr) ? 4u : 0u) |
                     (!(x.w >= thr) ? 8u : 0u))
                    << (4 * u);
          }
        }
      }
      // accepted elements (few) move from the ring slot to the lane queue
      if (__any_sync(kFull, q.cnt + __popc(mask) > TSel<NQ>::LCAP)) q.flush(true);
      while (mask) {
        const int b2 = __ffs(mask) - 1;
        mask &= mask - 1u;
        const int off = (b2 >> 2) * 128 + (b2 & 3);
        q.push_raw(sf[off], ib + (uint32_t)off);
      }
      __syncwarp();  // every lane is done with the slot before it is refilled
      ++ring.consumed;
      ring_fill(a, ring, n_items, n_warps, lane);
    }
    {  // scalar tail
      const int64_t done = d.head + (d.nvec << 2);
      if (done < d.len) {
        if (q.crowded(1)) q.flush(true);
        const bool ok = done + lane < d.len;
        q.push(ok, ok ? d.p[done + lane] : 0.f, d.base + (uint32_t)(done + lane));
      }
    }
    q.flush(true);
    if (sampled && !q.exact && q.total < want) {
      // the sampled bound let fewer than k elements through (~3 sigma): scan again with
      // the paper's adaptive bound only (exact in every case; plain loads)
      q.reset();
#pragma unroll 1
      for (int64_t e0 = 0; e0 < d.len; e0 += 128) {
        float v[4];
        bool ok[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int64_t e = e0 + u * 32 + lane;
          ok[u] = e < d.len;
          v[u] = ok[u] ? d.p[e] : 0.f;
        }
        if (q.crowded(4)) q.flush(true);
#pragma unroll
        for (int u = 0; u < 4; ++u) q.push(ok[u], v[u], d.base + (uint32_t)(e0 + u * 32 + lane));
      }
      q.flush(true);
    }

    // A3 / A4 output.  Chunked rows (P > 1) write keys: the sorted winners, whose
    // first `heads` entries also go to the row's head list for the bound of step 2.
    if (a.P > 1 && a.jth == 1) {
      // many chunks: the head is the chunk's smallest key, the winners stay unsorted
      uint64_t* ok = a.out_keys + item * a.k;
      uint64_t mn = kSentinelKey;
      for (int i = lane; i < a.k; i += 32) {
        const uint64_t key = i < q.total ? q.buf[i] : kSentinelKey;
        ok[i] = key;
        mn = umin64(mn, key);
      }
#pragma unroll
      for (int sft = 16; sft >= 1; sft >>= 1) mn = umin64(mn, shfl_xor64(mn, sft));
      if (lane == 0 && d.c != a.P - 1) a.heads[d.row * (a.P - 1) + d.c] = mn;
    } else {
      sort_block_inl<NQ>(q.buf, q.total);
      if (a.P == 1) {
        write_sorted<NQ>(q.buf, a.k, lane, a.vals + d.row * a.ld, a.out_val + d.row * a.k,
                         a.out_idx + d.row * a.k);
      } else {
        uint64_t* ok = a.out_keys + item * a.k;
        for (int i = lane; i < a.k; i += 32) ok[i] = q.buf[swz<NQ>(i)];
        if (d.c != a.P - 1) {
          uint64_t* hd = a.heads + (d.row * (a.P - 1) + d.c) * a.jth;
          for (int i = lane; i < a.jth; i += 32) hd[i] = q.buf[swz<NQ>(i)];
        }
      }
    }
    __syncwarp();

    // next item
    if (ring.n_item < 0) ring.n_item = draw_item(a, n_warps, lane);
    ring.c_item = ring.n_item;
    ring.n_item = -1;
    if (ring.p_item != ring.c_item) {
      ring.p_item = ring.c_item;
      ring_point(a, ring, n_items);
    }
    ring_fill(a, ring, n_items, n_warps, lane);
  }
}

// ---------------------------------------------------------------------------
// k = 1: min / argmin reduction on packed keys, one warp per (row, chunk).
// ---------------------------------------------------------------------------
__device__ __forceinline__ float4 ld_stream4(const float* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w)
               : "l"(p));
  return r;
}

template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) kselect_k1_kernel(const KSelArgs a) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t item = (int64_t)blockIdx.x * WARPS + warp;
  if (item >= a.n_rows * a.P) return;
  const ItemDesc d = decode_item(a, item);
  const float* p = d.p;
  uint64_t best = kSentinelKey;
  if (lane < d.head) best = umin64(best, make_key(p[lane], d.base + lane));
  const float* pv = p + d.head;
  const int64_t nvec = d.nvec;
  const uint32_t vbase = d.base + (uint32_t)d.head;
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
  const int64_t done = d.head + (nvec << 2);
  if (done + lane < d.len) take(p[done + lane], d.base + (uint32_t)(done + lane));
#pragma unroll
  for (int s = 16; s >= 1; s >>= 1) best = umin64(best, shfl_xor64(best, s));
  if (lane == 0) {
    if (a.P > 1) {
      a.out_keys[item] = best;
      if (d.c != a.P - 1) a.heads[d.row * (a.P - 1) + d.c] = best;
    } else if (best == kSentinelKey) {
      a.out_val[item] = __uint_as_float(0x7F800000u);
      a.out_idx[item] = -1;
    } else {
      const uint32_t idx = key_idx(best);
      a.out_val[item] = a.vals[d.row * a.ld + idx];
      a.out_idx[item] = (int32_t)idx;
    }
  }
}

// ---------------------------------------------------------------------------
// A4, steps 2-4.  Step 2: the row's bound = the k-th smallest of the chunks' head
// keys (every chunk but the last contributes its jth smallest, (P-1)*jth >= k of
// them: real elements of the row, so their k-th smallest is >= the row's k-th
// smallest).  Step 3: gather the chunk winners under the bound.  Step 4: select.
// Steps 2 and 4 are the same kernel: one warp per row over a list of keys.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
    kselect_prune_kernel(const uint64_t* __restrict__ keys, int64_t n_lists, int P, int k,
                         const unsigned long long* __restrict__ bound, uint64_t* __restrict__ cand,
                         unsigned int* __restrict__ count) {
  // a warp takes 256 consecutive keys of one list
  const int lane = threadIdx.x & 31;
  const int parts = (k + 255) / 256;
  const int64_t w = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int64_t list = w / parts;
  if (list >= n_lists) return;
  const int i_begin = (int)(w - list * parts) * 256;
  const int i_end = i_begin + 256 < k ? i_begin + 256 : k;
  const int64_t row = list / P;
  const uint64_t B = bound[row];
  uint64_t* out = cand + row * ((int64_t)P * k);
  for (int i0 = i_begin; i0 < i_end; i0 += 32) {
    const int i = i0 + lane;
    uint64_t key = kSentinelKey;
    if (i < i_end) key = keys[list * k + i];
    const bool keep = key != kSentinelKey && key <= B;
    const unsigned b = __ballot_sync(kFull, keep);
    if (b == 0u) continue;
    unsigned int pos = 0;
    if (lane == 0) pos = atomicAdd(count + row, (unsigned int)__popc(b));
    pos = __shfl_sync(kFull, pos, 0);
    if (keep) out[pos + __popc(b & ((1u << lane) - 1u))] = key;
  }
}

template <int NQ>
__global__ void __launch_bounds__(128)
    kselect_keys_kernel(const uint64_t* __restrict__ src, const unsigned int* __restrict__ count,
                        int64_t n_fixed, int64_t n_rows, int64_t cap, int k,
                        const float* __restrict__ rows, int64_t ld, float* __restrict__ out_val,
                        int32_t* __restrict__ out_idx, unsigned long long* __restrict__ bound_out) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int LCAP = TSelCfg<NQ>::LCAP;
  constexpr size_t per_warp = (size_t)32 * LCAP * sizeof(uint64_t) + sel_scratch_bytes<TSelCfg<NQ>::RB>();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 4 + warp;
  if (row >= n_rows) return;
  unsigned char* mine = smem_raw + (size_t)warp * per_warp;
  TSel<NQ> q;
  q.init(reinterpret_cast<uint64_t*>(mine),
         reinterpret_cast<uint32_t*>(mine + (size_t)32 * LCAP * sizeof(uint64_t)), lane, k);
  const uint64_t* c = src + row * cap;
  const int64_t n = count ? (int64_t)count[row] : n_fixed;
#pragma unroll 1
  for (int64_t e0 = 0; e0 < n; e0 += 128) {
    uint64_t key[4];
    bool ok[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t e = e0 + u * 32 + lane;
      ok[u] = e < n;
      key[u] = ok[u] ? c[e] : kSentinelKey;
    }
    if (q.crowded(4)) q.flush(false);
#pragma unroll
    for (int u = 0; u < 4; ++u) q.push(ok[u] && key[u] != kSentinelKey, key_val(key[u]), key_idx(key[u]));
  }
  q.flush(false);
  if (bound_out) {
    if (lane == 0) bound_out[row] = q.total >= k ? q.thr_key : kSentinelKey;
    return;
  }
  sort_block<NQ>(q.buf, q.total);
  write_sorted<NQ>(q.buf, k, lane, rows + row * ld, out_val + row * k, out_idx + row * k);
}

// ---------------------------------------------------------------------------
// Host side: plan (A4) and launches.
// ---------------------------------------------------------------------------
namespace {

constexpr int kWarpsPerCtaK1 = 4;
// Planning estimate of the resident warps per SM of a queue class (shared memory
// per warp decides it); the grid itself uses the real occupancy.
template <int NQ>
constexpr int resident_est() {
  return (int)((227 * 1024) / (StreamSmem<NQ>::total + 1024));
}
int resident_warps_per_sm(int k) {
  if (k == 1) return 16;
  if (k <= 32) return resident_est<1>();
  if (k <= 64) return resident_est<2>();
  if (k <= 128) return resident_est<4>();
  if (k <= 256) return resident_est<8>();
  if (k <= 512) return resident_est<16>();
  return resident_est<32>();
}

struct Plan {
  int P;          // chunks per row
  int64_t chunk;  // elements per chunk (multiple of 4)
  int jth;        // head keys per chunk: ceil(k / (P - 1))
  size_t off_work, off_keys, off_heads, off_cand, off_bound, off_count, bytes;  // workspace layout
};

// Rows are cut into chunks only when there are too few rows to occupy the GPU, and
// never below max(4096, 8k) elements per chunk (below that the k outputs per chunk
// dominate).  One chunk per resident warp.
Plan make_plan(int64_t n_rows, int64_t n, int k) {
  Plan p;
  const int64_t resident = (int64_t)sm_count() * resident_warps_per_sm(k);
  const int64_t min_chunk = k * 8 > 4096 ? (int64_t)k * 8 : 4096;
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
  p.jth = P > 1 ? (int)ceil_div(k, P - 1) : 1;
  size_t o = 0;
  p.off_work = o;
  o += 256;
  p.off_bound = o;
  if (P > 1) o += align_up((size_t)n_rows * sizeof(unsigned long long), 256);
  p.off_count = o;
  if (P > 1) o += align_up((size_t)n_rows * sizeof(unsigned int), 256);
  p.off_keys = o;
  if (P > 1) o += align_up((size_t)n_rows * P * k * sizeof(uint64_t), 256);
  p.off_heads = o;
  if (P > 1) o += align_up((size_t)n_rows * (P - 1) * p.jth * sizeof(uint64_t), 256);
  p.off_cand = o;
  if (P > 1) o += align_up((size_t)n_rows * P * k * sizeof(uint64_t), 256);
  p.bytes = o;
  return p;
}

template <int NQ>
int launch_stream(const KSelArgs& a, cudaStream_t s) {
  using SM = StreamSmem<NQ>;
  const int64_t items = a.n_rows * a.P;
  if (items == 0) return FS_OK;
  static int ctas_per_sm = 0;
  if (ctas_per_sm == 0) {
    FS_CUDA(cudaFuncSetAttribute(kselect_stream_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)SM::total));
    FS_CUDA(cudaFuncSetAttribute(kselect_stream_kernel<NQ>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 cudaSharedmemCarveoutMaxShared));
    int occ = 0;
    FS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kselect_stream_kernel<NQ>, SM::WARPS * 32,
                                                          SM::total));
    ctas_per_sm = occ > 0 ? occ : 1;
  }
  int64_t grid = ceil_div(items, SM::WARPS);
  const int64_t cap = (int64_t)sm_count() * ctas_per_sm;
  if (grid > cap) grid = cap;
  kselect_stream_kernel<NQ><<<(unsigned)grid, SM::WARPS * 32, SM::total, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
}

struct KeysArgs {
  const uint64_t* src;
  const unsigned int* count;  // per-row length, or NULL: n_fixed
  int64_t n_fixed, n_rows, cap;
  int k;
  const float* rows;
  int64_t ld;
  float* out_val;
  int32_t* out_idx;
  unsigned long long* bound_out;  // not NULL: write only the k-th smallest key
};

template <int NQ>
int launch_keys(const KeysArgs& g, cudaStream_t s) {
  const size_t smem = 4 * ((size_t)32 * TSelCfg<NQ>::LCAP * sizeof(uint64_t) + sel_scratch_bytes<TSelCfg<NQ>::RB>());
  static bool attr_done = false;
  if (!attr_done) {
    FS_CUDA(cudaFuncSetAttribute(kselect_keys_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)smem));
    attr_done = true;
  }
  kselect_keys_kernel<NQ><<<(unsigned)ceil_div(g.n_rows, 4), 128, smem, s>>>(
      g.src, g.count, g.n_fixed, g.n_rows, g.cap, g.k, g.rows, g.ld, g.out_val, g.out_idx, g.bound_out);
  FS_LAUNCHED();
  return FS_OK;
}

#define FS_KCLASS_DISPATCH(k, CALL)          \
  do {                                       \
    if ((k) <= 32) return CALL(1);           \
    if ((k) <= 64) return CALL(2);           \
    if ((k) <= 128) return CALL(4);          \
    if ((k) <= 256) return CALL(8);          \
    if ((k) <= 512) return CALL(16);         \
    return CALL(32);                         \
  } while (0)

int launch_level1(const KSelArgs& a, cudaStream_t s) {
  if (a.k == 1) {
    const int64_t items = a.n_rows * a.P;
    if (items == 0) return FS_OK;
    const int64_t grid = ceil_div(items, kWarpsPerCtaK1);
    if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "too many rows for one launch");
    kselect_k1_kernel<kWarpsPerCtaK1><<<(unsigned)grid, kWarpsPerCtaK1 * 32, 0, s>>>(a);
    FS_LAUNCHED();
    return FS_OK;
  }
#define FS_CALL(NQ) launch_stream<NQ>(a, s)
  FS_KCLASS_DISPATCH(a.k, FS_CALL);
#undef FS_CALL
}

int launch_keys_any(const KeysArgs& g, cudaStream_t s) {
#define FS_CALL(NQ) launch_keys<NQ>(g, s)
  FS_KCLASS_DISPATCH(g.k, FS_CALL);
#undef FS_CALL
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
                        int32_t* out_idx, void* ws, cudaStream_t s);
static bool use_old_path() {
  static int v = -1;
  if (v < 0) {
    const char* e = getenv("FS_KSELECT");
    v = (e && e[0] == 'o') ? 1 : 0;
  }
  return v == 1;
}

// Selection over device rows; also used by the flat and IVFPQ drivers.
size_t kselect_ws_bytes(int64_t n_rows, int64_t n, int k) {
  const size_t a = make_plan(n_rows, n, k).bytes, b = k >= 2 ? kselect_rows_ws_bytes(n_rows, n, k) : 0;
  return a > b ? a : b;
}

int kselect_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                   int32_t* out_idx, void* ws, cudaStream_t s) {
  if (k >= 2 && !use_old_path()) return kselect_rows_device(rows, n_rows, n, ld, k, out_val, out_idx, ws, s);
  const Plan p = make_plan(n_rows, n, k);
  char* w = static_cast<char*>(ws);
  KSelArgs a;
  a.vals = rows;
  a.n_rows = n_rows;
  a.n = n;
  a.ld = ld;
  a.P = p.P;
  a.chunk = p.chunk;
  a.k = k;
  a.out_val = out_val;
  a.out_idx = out_idx;
  a.out_keys = nullptr;
  a.heads = nullptr;
  a.jth = p.jth;
  a.work = reinterpret_cast<unsigned int*>(w + p.off_work);
  // work counter, and for chunked rows bound + count (adjacent): one memset
  FS_CUDA(cudaMemsetAsync(w, 0, p.off_keys, s));
  if (p.P == 1) return launch_level1(a, s);
  a.out_keys = reinterpret_cast<uint64_t*>(w + p.off_keys);
  a.heads = reinterpret_cast<uint64_t*>(w + p.off_heads);
  unsigned long long* bound = reinterpret_cast<unsigned long long*>(w + p.off_bound);
  unsigned int* count = reinterpret_cast<unsigned int*>(w + p.off_count);
  uint64_t* cand = reinterpret_cast<uint64_t*>(w + p.off_cand);
  int rc = launch_level1(a, s);  // step 1: per-chunk winners
  if (rc != FS_OK) return rc;
  KeysArgs g;
  g.src = a.heads;  // step 2: bound = k-th smallest head key
  g.count = nullptr;
  g.n_fixed = (int64_t)(p.P - 1) * p.jth;
  g.n_rows = n_rows;
  g.cap = g.n_fixed;
  g.k = k;
  g.rows = rows;
  g.ld = ld;
  g.out_val = nullptr;
  g.out_idx = nullptr;
  g.bound_out = bound;
  if ((rc = launch_keys_any(g, s)) != FS_OK) return rc;
  const int64_t n_lists = n_rows * p.P;  // step 3: gather under the bound
  const int64_t warps = n_lists * ((k + 255) / 256);
  kselect_prune_kernel<<<(unsigned)ceil_div(warps, 8), 256, 0, s>>>(a.out_keys, n_lists, p.P, k, bound, cand,
                                                                    count);
  FS_LAUNCHED();
  g.src = cand;  // step 4: select among the gathered keys
  g.count = count;
  g.cap = (int64_t)p.P * k;
  g.out_val = out_val;
  g.out_idx = out_idx;
  g.bound_out = nullptr;
  return launch_keys_any(g, s);
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
    rc = fs::kselect_device(d_rows + r0 * ld, nr, n, ld, k, d_val + r0 * k, d_idx + r0 * k, base + o_ws, st.s_run);
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
