// flat_tc.cu -- tensor-core engine of fs_flat_l2_knn:
// the -2<x,y> contraction on tcgen05 tensor cores with the accumulator
// in TMEM, operands staged by TMA, and the "+||y||^2 then k-select" step run
// by the epilogue warps straight from TMEM: the nq x nb matrix never reaches HBM.
//
// Precision (reading F-5): every fp32 operand is split as x = hi + lo with
// hi = x truncated to TF32 (10 explicit mantissa bits) and lo = (x - hi) truncated to
// TF32; the tile accumulates hi*hi + lo*hi + hi*lo in fp32 ("3xTF32", ~2^-21 relative).
// The hi plane is the operand itself (the MMA ignores the 13 low mantissa bits); a pre-pass
// computes the squared norms (B1) and checks whether any lo is non-zero; only then is the lo
// plane written, and if lo == 0 everywhere (e.g. small-integer data such as cfg3) the kernel
// issues the hi*hi products only, which is then exact -- a checked dispatch, never a guess.
//
// Kernel shape: persistent CTAs (one per SM), 320 threads:
//   warp 8      TMA producer   query tile (128 rows, resident per work item) and a ring
//                              of database stages (256 rows x 32 columns x fp32 = 32 KB)
//   warp 9      MMA issuer     tcgen05.mma kind::tf32, M=128 N=256 K=8, two 256-column
//                              accumulators in TMEM (ping-pong with the epilogue)
//   warps 0-7   epilogue       two warpgroups, each on half of the tile's columns; thread = TMEM lane = query row: tcgen05.ld, d' = ||y||^2 -
//                              2 acc, compare with the row's bound; the rare survivors go
//                              to a per-row candidate buffer, merged into the row's queue
//                              by the whole warp (warp_flush of select.cuh)
// Work item = (database split s, query tile): items are ordered split-major, so CTAs that
// run at the same time read the same part of the database (L2 reuse), and a query's
// bound found in earlier splits (gbound) prunes the later ones.
#include <cuda.h>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "flat.cuh"
#include "sm100.cuh"
#include "tselect.cuh"

namespace fs {

namespace {

constexpr int BM = 128;                      // query rows per tile (MMA M)
constexpr int BN = 256;                      // database rows per tile (MMA N)
constexpr int BK = 32;                       // fp32 columns per stage = 128 bytes (swizzle span)
constexpr int A_KB_BYTES = BM * BK * 4;      // 16 KB
constexpr int B_STAGE_BYTES = BN * BK * 4;   // 32 KB
constexpr int MAX_STAGES = 4;
constexpr int CLUSTER = 2;                    // CTAs per cluster: same database tiles, different query tiles;
                                              // each loads 1/CLUSTER of a database stage and multicasts it
constexpr int YN_RING = 2;                    // ||y||^2 tiles (1 KB each) in flight ahead of the epilogue
constexpr int EPI_GROUPS = 2;                 // epilogue warpgroups; group g takes columns [g*128, g*128+128) of a tile
constexpr int TC_THREADS = 64 + EPI_GROUPS * 128;
// Warp roles.  The two single-thread roles take the highest warp ids (the sub-partition
// schedulers favour higher warp ids; a starved MMA issuer would idle the tensor pipe).
constexpr int TMA_WARP = EPI_GROUPS * 4, MMA_WARP = EPI_GROUPS * 4 + 1;
constexpr int EPI_RB = 4;                     // radix digit width of the epilogue selection (1 KB of counters per warp)
constexpr int STAGE_KEYS = 256;               // row buffers up to this size are selected in shared memory
constexpr int SCRATCH_BYTES = EPI_GROUPS * 4 * ((1 << EPI_RB) * 64 + STAGE_KEYS * 8);  // 8 warps x (1 KB + 2 KB)
#ifndef FS_TC_REFRESH
#define FS_TC_REFRESH 8  // tiles between two looks at the published bounds (power of two)
#endif
#ifndef FS_TC_EAGER
#define FS_TC_EAGER 48
#endif
#ifndef FS_TC_EAGER_Q
#define FS_TC_EAGER_Q 3
#endif
constexpr int EAGER_EXTRA = FS_TC_EAGER;       // idle-time restore of rows holding >= k + max(this, k * FS_TC_EAGER_Q / 4) keys
                                              // (sweep in profiles/r01_flat.md)
constexpr int KREG = 12;                      // k <= KREG: the row's queue is a sorted array of the thread's own, kept in the
                                              // warp's selection scratch (3 KB = 12 keys per lane, [slot][lane]: conflict-free)
constexpr int HB_LEVELS = 3;                  // hierarchical bound: levels 1..3 (2, 4, 8 queues)
constexpr int HB_SLOTS = 2 + 4 + 8;
constexpr int SMEM_LIMIT = 227 * 1024;

struct TcArgs {
  int64_t nq, nb;
  int d, KB, k, kclass, K;
  int S, qtiles;
  int qgroups;                 // ceil(qtiles / CLUSTER): work item = (split, group of CLUSTER query tiles)
  int cap;                     // keys per row buffer: K + 128
  int smem_bytes;              // dynamic shared memory of the launch
  int64_t chunk;               // database rows per split (multiple of BN)
  int64_t chunk0;              // rows of split 0 (= chunk; a smaller first split was measured and lost: the splits of
                               // the first wave run concurrently and cannot use its bound)
  const float* ynorm;          // [>= nb rounded up to BN]
  uint64_t* Wg;                // [nq][S * EPI_GROUPS][K]
  unsigned int* gbound;        // [nq] order image of the best known k-th distance
  unsigned int* hbound;        // [nq][HB_SLOTS] level l (1..HB_LEVELS) holds the ceil(k / 2^l)-th smallest
                               // distances of 2^l different finished partial queues (+inf image: empty)
  unsigned int* hclaim;        // [nq][HB_LEVELS] slots handed out per level
  uint64_t* cbuf;              // [gridDim.x][EPI_GROUPS][BM][cap]: winners so far, then new candidates
  const unsigned int* lo_flag; // != 0: lo planes are not all zero (3xTF32)
  const unsigned int* nq_dev;  // != NULL: the number of queries, on the device (<= nq; re-run of the failed queries)
  int lazy_final;              // != 0: the queues start from a sampled bound; a queue is not restored at the end of its
                               // item just to publish its k-th distance (only if it holds more than K keys)
  float* dout;                 // != NULL: no selection, d'(q, j) = ||y_j||^2 - 2 <x_q, y_j> is written to
  int64_t dld;                 //          dout[q * dld + j] (dld % 4 == 0); the launch passes k = 1
};

// ---------------------------------------------------------------------------
// B1 + operand split.  The hi plane is the caller's array itself: tcgen05.mma kind::tf32 reads the
// upper 19 bits of every fp32 operand and ignores the 13 low mantissa bits, i.e. it multiplies
// hi = x truncated to TF32 (checked on B200: bit-identical results with an explicitly truncated copy).
// norm_flag_kernel: squared norms (one warp per vector) and whether any lo = (x - hi) truncated is
// non-zero; lo_plane_kernel writes the lo plane, and only when the flag is set (small-integer data such as
// cfg3 never pay for it: one read of the database for the norms instead of a read and two writes).
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
    norm_flag_kernel(const float* __restrict__ x, int64_t n, int d, float* __restrict__ norm,
                     unsigned int* __restrict__ flag) {
  const int lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (row >= n) return;
  const float* p = x + row * d;
  float s = 0.f;
  bool any = false;
  for (int c = lane; c < d; c += 32) {
    const float v = p[c];
    s = fmaf(v, v, s);
    const float h = __uint_as_float(__float_as_uint(v) & 0xFFFFE000u);
    any |= (__float_as_uint(v - h) & 0xFFFFE000u) != 0u && (v - h) != 0.f;
  }
#pragma unroll
  for (int m = 16; m >= 1; m >>= 1) s += __shfl_xor_sync(kFull, s, m);
  if (lane == 0) norm[row] = s;
  if (__any_sync(kFull, any) && lane == 0) atomicOr(flag, 1u);
}

__global__ void __launch_bounds__(256)
    lo_plane_kernel(const float* __restrict__ x, int64_t n_elems, float* __restrict__ lo,
                    const unsigned int* __restrict__ flag) {
  if (*flag == 0u) return;  // every lo is zero: the kernel issues hi * hi only and never reads the plane
  for (int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4; i < n_elems; i += (int64_t)gridDim.x * blockDim.x * 4) {
    float4 v;  // n_elems = rows * d, d % 4 == 0; x itself may be misaligned (lo is ours: aligned)
    if ((reinterpret_cast<uintptr_t>(x) & 15u) == 0)
      v = *reinterpret_cast<const float4*>(x + i);
    else
      v = make_float4(x[i], x[i + 1], x[i + 2], x[i + 3]);
    float4 l;
    l.x = __uint_as_float(__float_as_uint(v.x - __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u)) & 0xFFFFE000u);
    l.y = __uint_as_float(__float_as_uint(v.y - __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u)) & 0xFFFFE000u);
    l.z = __uint_as_float(__float_as_uint(v.z - __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u)) & 0xFFFFE000u);
    l.w = __uint_as_float(__float_as_uint(v.w - __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u)) & 0xFFFFE000u);
    *reinterpret_cast<float4*>(lo + i) = l;
  }
}

// Explicitly truncated copy (operands that are not 16-byte aligned cannot be read by TMA in place).
__global__ void __launch_bounds__(256) hi_plane_kernel(const float* __restrict__ x, int64_t n_elems, float* __restrict__ hi) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_elems; i += (int64_t)gridDim.x * blockDim.x)
    hi[i] = __uint_as_float(__float_as_uint(x[i]) & 0xFFFFE000u);
}

// The sample: every stride-th row of the database (and of its lo plane in 3xTF32 mode) with its ||y||^2,
// copied to a compact array -- one warp per row.
__global__ void __launch_bounds__(256) gather_sample_kernel(const float* __restrict__ hi, const float* __restrict__ lo,
                                                            const float* __restrict__ ynorm, int64_t stride, int64_t n, int d,
                                                            const unsigned int* __restrict__ lo_flag, float* __restrict__ shi,
                                                            float* __restrict__ slo, float* __restrict__ syn) {
  const int64_t i = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (i >= n) return;
  const int lane = threadIdx.x & 31;
  const int64_t r = i * stride;
  const bool split = *lo_flag != 0u;
  for (int j = lane; j < d; j += 32) {
    shi[i * d + j] = hi[r * d + j];
    if (split) slo[i * d + j] = lo[r * d + j];
  }
  if (lane == 0) syn[i] = ynorm[r];
}

// Rows of the queries whose sampled bound failed, gathered for the re-run: one warp per failed query.
__global__ void __launch_bounds__(256) gather_failed_kernel(const float* __restrict__ hi, const float* __restrict__ lo, int d,
                                                            const unsigned int* __restrict__ fail_cnt,
                                                            const int* __restrict__ fail_q, const unsigned int* __restrict__ lo_flag,
                                                            float* __restrict__ ghi, float* __restrict__ glo) {
  const int64_t i = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (i >= (int64_t)*fail_cnt) return;
  const int lane = threadIdx.x & 31;
  const int64_t q = fail_q[i];
  const bool split = *lo_flag != 0u;
  for (int j = lane; j < d; j += 32) {
    ghi[i * d + j] = hi[q * d + j];
    if (split) glo[i * d + j] = lo[q * d + j];
  }
}

// ---------------------------------------------------------------------------
// B2 + B3: the tile kernel.
// ---------------------------------------------------------------------------
struct Pipe {
  int stage;
  uint32_t phase;
  __device__ __forceinline__ void advance(int nstage) {
    if (++stage == nstage) {
      stage = 0;
      phase ^= 1u;
    }
  }
};

__global__ void __launch_bounds__(TC_THREADS, 1)
    flat_tc_kernel(const __grid_constant__ CUtensorMap map_a_hi, const __grid_constant__ CUtensorMap map_a_lo,
                   const __grid_constant__ CUtensorMap map_b_hi, const __grid_constant__ CUtensorMap map_b_lo,
                   const TcArgs a) {
  extern __shared__ unsigned char smem_dyn[];
  // operand tiles need 1024-byte alignment (128-byte swizzle atoms of 8 rows)
  unsigned char* smem = smem_dyn + ((1024u - (sm100::smem_addr(smem_dyn) & 1023u)) & 1023u);
  const bool split = *a.lo_flag != 0u;
  const int KB = a.KB;
  // carve: barriers | selection scratch | A hi (| A lo) | ring of B stages (as many as fit, <= 4)
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
  uint64_t* full = bars;                    // [MAX_STAGES]
  uint64_t* empty = bars + MAX_STAGES;      // [MAX_STAGES]
  uint64_t* tfull = bars + 2 * MAX_STAGES;  // [2]
  uint64_t* tempty = tfull + 2;             // [2]
  uint64_t* a_full = tempty + 2;
  uint64_t* a_empty = a_full + 1;
  uint64_t* yfull = a_empty + 1;            // [YN_RING]
  uint64_t* yempty = yfull + YN_RING;       // [YN_RING]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(yempty + YN_RING);
  float* s_yn = reinterpret_cast<float*>(smem + 1024);  // [YN_RING][BN]
  unsigned char* scratch_all = smem + 1024 + YN_RING * BN * 4;
  unsigned char* sA_hi = scratch_all + SCRATCH_BYTES;
  unsigned char* sA_lo = sA_hi + (size_t)KB * A_KB_BYTES;
  unsigned char* sB = sA_lo + (split ? (size_t)KB * A_KB_BYTES : 0);
  int nstage = (int)((smem_dyn + a.smem_bytes - sB) / B_STAGE_BYTES);
  if (nstage > MAX_STAGES) nstage = MAX_STAGES;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int i = 0; i < MAX_STAGES; ++i) {
      sm100::mbar_init(full + i, 1);
      sm100::mbar_init(empty + i, CLUSTER);  // the MMA warps of all CTAs of the cluster release a stage
    }
    for (int i = 0; i < 2; ++i) {
      sm100::mbar_init(tfull + i, 1);
      sm100::mbar_init(tempty + i, 4 * EPI_GROUPS);
    }
    sm100::mbar_init(a_full, 1);
    sm100::mbar_init(a_empty, 1);
    for (int i = 0; i < YN_RING; ++i) {
      sm100::mbar_init(yfull + i, 1);
      sm100::mbar_init(yempty + i, 4 * EPI_GROUPS);
    }
    sm100::fence_mbar_init();
    sm100::tma_prefetch_desc(&map_a_hi);
    sm100::tma_prefetch_desc(&map_a_lo);
    sm100::tma_prefetch_desc(&map_b_hi);
    sm100::tma_prefetch_desc(&map_b_lo);
  }
  if (warp == MMA_WARP) sm100::tmem_alloc(tmem_slot, 512);
  sm100::tc_fence_before();
  __syncthreads();
  if (CLUSTER > 1) sm100::cluster_sync_all();  // peers' barriers are initialised before anything lands on them
  sm100::tc_fence_after();
  const uint32_t crank = CLUSTER > 1 ? sm100::cluster_ctarank() : 0u;
  const int64_t cluster_id = blockIdx.x / CLUSTER, n_clusters = gridDim.x / CLUSTER;
  constexpr uint16_t kAllCtas = (uint16_t)((1u << CLUSTER) - 1u);
  const uint32_t tmem_base = *tmem_slot;
  int64_t nq = a.nq;
  if (a.nq_dev) nq = (int64_t)*a.nq_dev < nq ? (int64_t)*a.nq_dev : nq;
  const int64_t qgroups = a.nq_dev ? (nq + (int64_t)BM * CLUSTER - 1) / ((int64_t)BM * CLUSTER) : a.qgroups;
  const int64_t n_items = (int64_t)a.S * qgroups;

  if (warp == TMA_WARP) {
    // ===== TMA producer =====
    if (lane == 0) {
      Pipe pp{0, 0u};
      int it = 0;
      uint32_t ptile = 0;
      for (int64_t item = cluster_id; item < n_items; item += n_clusters, ++it) {
        const int s = (int)(item / qgroups), qt = (int)(item - (int64_t)s * qgroups) * CLUSTER + (int)crank;
        const int64_t b_begin = s == 0 ? 0 : a.chunk0 + (int64_t)(s - 1) * a.chunk;
        const int64_t b_len = s == 0 ? a.chunk0 : a.chunk;
        const int64_t b_end = b_begin + b_len < a.nb ? b_begin + b_len : a.nb;
        const int ntiles = (int)((b_end - b_begin + BN - 1) / BN);
        if (it > 0) sm100::mbar_wait(a_empty, (uint32_t)(it - 1) & 1u);  // previous item's MMAs are done with A
        sm100::mbar_expect_tx(a_full, (uint32_t)(KB * A_KB_BYTES * (split ? 2 : 1)));
        for (int kb = 0; kb < KB; ++kb) {
          sm100::tma_load_2d(sA_hi + kb * A_KB_BYTES, &map_a_hi, kb * BK, qt * BM, a_full);
          if (split) sm100::tma_load_2d(sA_lo + kb * A_KB_BYTES, &map_a_lo, kb * BK, qt * BM, a_full);
        }
        for (int t = 0; t < ntiles; ++t, ++ptile) {
          const int row0 = (int)(b_begin + (int64_t)t * BN);
          {  // the tile's ||y||^2 values for the epilogue
            const uint32_t ys = ptile % YN_RING;
            sm100::mbar_wait(yempty + ys, ((ptile / YN_RING) & 1u) ^ 1u);
            sm100::mbar_expect_tx(yfull + ys, BN * 4);
            sm100::bulk_load(s_yn + ys * BN, a.ynorm + row0, BN * 4, yfull + ys);
          }
          for (int kb = 0; kb < KB; ++kb) {
            for (int pl = 0; pl < (split ? 2 : 1); ++pl) {
              sm100::mbar_wait(empty + pp.stage, pp.phase ^ 1u);  // free in every CTA of the cluster
              sm100::mbar_expect_tx(full + pp.stage, (uint32_t)B_STAGE_BYTES);
              if (CLUSTER > 1) {  // this CTA's share of the rows, delivered to all CTAs
                constexpr int rows = BN / CLUSTER;
                sm100::tma_load_2d_mc(sB + (size_t)pp.stage * B_STAGE_BYTES + (size_t)crank * rows * BK * 4,
                                      pl ? &map_b_lo : &map_b_hi, kb * BK, row0 + (int)crank * rows, full + pp.stage,
                                      kAllCtas);
              } else {
                sm100::tma_load_2d(sB + (size_t)pp.stage * B_STAGE_BYTES, pl ? &map_b_lo : &map_b_hi, kb * BK, row0,
                                   full + pp.stage);
              }
              pp.advance(nstage);
            }
          }
        }
      }
    }
  } else if (warp == MMA_WARP) {
    // ===== MMA issuer =====
    if (lane == 0) {
      constexpr uint32_t idesc = sm100::make_idesc_tf32(BM, BN);
      Pipe pc{0, 0u};
      uint32_t tile_count = 0;
      int it = 0;
      for (int64_t item = cluster_id; item < n_items; item += n_clusters, ++it) {
        const int s = (int)(item / qgroups);
        const int64_t b_begin = s == 0 ? 0 : a.chunk0 + (int64_t)(s - 1) * a.chunk;
        const int64_t b_len = s == 0 ? a.chunk0 : a.chunk;
        const int64_t b_end = b_begin + b_len < a.nb ? b_begin + b_len : a.nb;
        const int ntiles = (int)((b_end - b_begin + BN - 1) / BN);
        sm100::mbar_wait(a_full, (uint32_t)it & 1u);
        sm100::tc_fence_after();
        for (int t = 0; t < ntiles; ++t, ++tile_count) {
          const uint32_t as = tile_count & 1u;
          sm100::mbar_wait(tempty + as, ((tile_count >> 1) & 1u) ^ 1u);  // epilogue drained this accumulator
          sm100::tc_fence_after();
          const uint32_t d_tmem = tmem_base + as * BN;
          for (int kb = 0; kb < KB; ++kb) {
            const uint64_t da_hi = sm100::make_kmajor_sw128_desc(sm100::smem_addr(sA_hi + kb * A_KB_BYTES));
            const uint64_t da_lo = sm100::make_kmajor_sw128_desc(sm100::smem_addr(sA_lo + kb * A_KB_BYTES));
            // stage with the hi plane of the database: hi*hi (+ lo*hi)
            sm100::mbar_wait(full + pc.stage, pc.phase);
            sm100::tc_fence_after();
            uint64_t db = sm100::make_kmajor_sw128_desc(sm100::smem_addr(sB + (size_t)pc.stage * B_STAGE_BYTES));
#pragma unroll
            for (int ks = 0; ks < BK / 8; ++ks)  // K = 8 per MMA = 32 bytes = 2 descriptor units
              sm100::mma_tf32_ss(d_tmem, da_hi + 2 * ks, db + 2 * ks, idesc, (kb | ks) != 0 ? 1u : 0u);
            if (split) {
#pragma unroll
              for (int ks = 0; ks < BK / 8; ++ks) sm100::mma_tf32_ss(d_tmem, da_lo + 2 * ks, db + 2 * ks, idesc, 1u);
            }
            if (CLUSTER > 1) sm100::mma_commit_mc(empty + pc.stage, kAllCtas); else sm100::mma_commit(empty + pc.stage);
            pc.advance(nstage);
            if (split) {  // stage with the lo plane: hi*lo
              sm100::mbar_wait(full + pc.stage, pc.phase);
              sm100::tc_fence_after();
              db = sm100::make_kmajor_sw128_desc(sm100::smem_addr(sB + (size_t)pc.stage * B_STAGE_BYTES));
#pragma unroll
              for (int ks = 0; ks < BK / 8; ++ks) sm100::mma_tf32_ss(d_tmem, da_hi + 2 * ks, db + 2 * ks, idesc, 1u);
              if (CLUSTER > 1) sm100::mma_commit_mc(empty + pc.stage, kAllCtas); else sm100::mma_commit(empty + pc.stage);
              pc.advance(nstage);
            }
          }
          sm100::mma_commit(tfull + as);
        }
        sm100::mma_commit(a_empty);
      }
    }
  } else {
    // ===== epilogue: B3 =====
    const int quarter = warp & 3;  // TMEM lanes 32*quarter .. +31 belong to this warp
    const int eg = warp >> 2;  // epilogue group: its own columns, candidate buffers and partial queues
    const int K = a.K, k = a.k, cap = a.cap;
    const int SQ = a.S * EPI_GROUPS;  // partial queues per query
    const bool rq = k <= KREG;        // thread-private sorted queue: exact bound after every insertion, no restore steps
    uint32_t* scratch = reinterpret_cast<uint32_t*>(scratch_all + (size_t)warp * (sel_scratch_bytes<EPI_RB>() + STAGE_KEYS * 8));
    uint64_t* stage = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(scratch) + sel_scratch_bytes<EPI_RB>());
    uint64_t* cb_warp = a.cbuf + (((size_t)blockIdx.x * EPI_GROUPS + eg) * BM + quarter * 32) * cap;
    uint64_t* cb = cb_warp + (size_t)lane * cap;
    uint32_t tile_count = 0;
    for (int64_t item = cluster_id; item < n_items; item += n_clusters) {
      const int s = (int)(item / qgroups), qt = (int)(item - (int64_t)s * qgroups) * CLUSTER + (int)crank;
      const int64_t b_begin = s == 0 ? 0 : a.chunk0 + (int64_t)(s - 1) * a.chunk;
      const int64_t b_len = s == 0 ? a.chunk0 : a.chunk;
      const int64_t b_end = b_begin + b_len < a.nb ? b_begin + b_len : a.nb;
      const int ntiles = (int)((b_end - b_begin + BN - 1) / BN);
      const int64_t q_warp = (int64_t)qt * BM + quarter * 32;
      const int64_t q = q_warp + lane;
      const bool valid = q < nq;
      // start from the best bound other splits have published (inclusive)
      uint32_t gb = valid ? a.gbound[q] : 0u;
      if (valid && k >= 8) {
        // 2^l disjoint partial queues whose ceil(k / 2^l)-th smallest distances are all <= m hold
        // >= k elements <= m together: m bounds the query's k-th distance (tighter than any
        // single queue's own k-th once several splits have finished)
        const unsigned int* hb = a.hbound + q * HB_SLOTS;
        int o = 0;
#pragma unroll
        for (int l = 1; l <= HB_LEVELS; ++l) {
          unsigned int mx = 0u;
          for (int t = 0; t < (1 << l); ++t) mx = max(mx, hb[o + t]);
          gb = min(gb, mx);
          o += 1 << l;
        }
      }
      if (gb > 0xFF800000u) gb = 0xFF800000u;  // no bound yet: +inf
      uint64_t thr0 = valid ? (((uint64_t)gb << 32) | 0xFFFFFFFFull) : 0ull;
      uint64_t thr_key = thr0;
      float thr_val = valid ? ord_f32((uint32_t)(thr0 >> 32)) : __uint_as_float(0xFF800000u);
      int cnt = 0;  // keys in this row's buffer: the winners so far, then new candidates
      uint64_t* Rq = reinterpret_cast<uint64_t*>(scratch) + lane;  // rq: the row's cnt <= k smallest keys, ascending, stride 32
      __syncwarp();

      // Restore step for the rows that ask for it: the whole warp selects the k
      // smallest of the row's buffer by radix counting (tselect.cuh), in place.
      auto flush_rows = [&](bool need, bool final) {
        unsigned todo = __ballot_sync(kFull, need);
        while (todo) {
          const int r = __ffs(todo) - 1;
          todo &= todo - 1u;
          const int m = __shfl_sync(kFull, cnt, r);
          if (m < k) continue;
          uint64_t* gbuf = cb_warp + (size_t)r * cap;
          __syncwarp();
          // small buffers are selected in shared memory (one coalesced read instead of a
          // chain of dependent global round trips), the winners go back to the row buffer
          const bool staged = m <= STAGE_KEYS;
          uint64_t* buf = staged ? stage : gbuf;
          uint64_t kor = 0ull, kand = ~0ull;
          for (int i = lane; i < m; i += 32) {
            const uint64_t key = gbuf[i];
            if (staged) stage[i] = key;
            kor |= key;
            kand &= key;
          }
          __syncwarp();
          const uint32_t olo = __reduce_or_sync(kFull, (uint32_t)kor), ohi = __reduce_or_sync(kFull, (uint32_t)(kor >> 32));
          const uint32_t alo = __reduce_and_sync(kFull, (uint32_t)kand), ahi = __reduce_and_sync(kFull, (uint32_t)(kand >> 32));
          const uint64_t diff = (((uint64_t)ohi << 32) | olo) & ~(((uint64_t)ahi << 32) | alo);
          const uint64_t kth = radix_select_kth<EPI_RB>(buf, m, k, diff, scratch);
          if (final && staged && k >= 8) {
            // publish this queue's ceil(k / 2^l)-th smallest distances (first come, first served)
            int o = 0;
#pragma unroll 1
            for (int l = 1; l <= HB_LEVELS; ++l) {
              const int rank = (k + (1 << l) - 1) >> l;
              const uint64_t kv = radix_select_kth<EPI_RB>(buf, m, rank, diff, scratch);
              if (lane == 0) {
                const unsigned int slot = atomicAdd(a.hclaim + (q_warp + r) * HB_LEVELS + (l - 1), 1u);
                if (slot < (1u << l)) a.hbound[(q_warp + r) * HB_SLOTS + o + slot] = (unsigned int)(kv >> 32);
              }
              o += 1 << l;
            }
            __syncwarp();
          }
          int w = 0;
          for (int i0 = 0; i0 < m; i0 += 32) {  // keep the keys <= kth: exactly k (keys are distinct)
            const int i = i0 + lane;
            uint64_t key = 0;
            bool keep = false;
            if (i < m) {
              key = buf[i];
              keep = key <= kth;
            }
            const unsigned b = __ballot_sync(kFull, keep);
            if (keep) gbuf[w + __popc(b & ((1u << lane) - 1u))] = key;
            w += __popc(b);
          }
          __syncwarp();
          if (lane == r) {
            thr_key = kth < thr0 ? kth : thr0;
            thr_val = key_val(thr_key);
            cnt = k;
            // this queue's k-th distance bounds the query's: splits running now may use it at once
            if (kth < thr0) atomicMin(a.gbound + q, (unsigned int)(kth >> 32));
          }
        }
      };

      for (int t = 0; t < ntiles; ++t, ++tile_count) {
        const uint32_t as = tile_count & 1u;
        if (k > 1 && (t & (FS_TC_REFRESH - 1)) == (FS_TC_REFRESH - 1) && valid) {
          // adopt what the other splits of this query have published since the item began
          const uint32_t g2 = *reinterpret_cast<volatile unsigned int*>(a.gbound + q);
          const uint64_t t2 = ((uint64_t)g2 << 32) | 0xFFFFFFFFull;
          if (t2 < thr0) {
            thr0 = t2;
            if (t2 < thr_key) {
              thr_key = t2;
              thr_val = ord_f32(g2);
            }
          }
        }
        const int64_t col0 = b_begin + (int64_t)t * BN;
        const int ncols = (int)(b_end - col0 < BN ? b_end - col0 : BN);
        // The accumulator is not ready (the other epilogue group or the peer CTA holds the pipeline
        // back): restore the rows that already hold more than k keys now instead of spinning -- it
        // tightens their bounds early and takes restore work off the path of later tiles.
        if (k > 1 && a.dout == nullptr && !__all_sync(kFull, sm100::mbar_test(tfull + as, (tile_count >> 1) & 1u)))
          flush_rows(cnt >= k + (EAGER_EXTRA > (k * FS_TC_EAGER_Q >> 2) ? EAGER_EXTRA : (k * FS_TC_EAGER_Q >> 2)), false);
        sm100::mbar_wait(tfull + as, (tile_count >> 1) & 1u);
        sm100::tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + as * BN;
        // this group's 128 columns in four blocks of 32; ||y||^2 comes from the shared-memory
        // tile the producer staged (the TMEM load is not pipelined: its destination
        // registers must not be touched before tcgen05.wait::ld)
        constexpr int BW = 64;  // columns per TMEM load
        constexpr int NBLK = BN / BW / EPI_GROUPS;
        const int cg0 = eg * NBLK;  // first block of this group
        uint32_t v[BW];
        const uint32_t ys = tile_count % YN_RING;
        sm100::mbar_wait(yfull + ys, (tile_count / YN_RING) & 1u);
        const float4* ynp = reinterpret_cast<const float4*>(s_yn + ys * BN + cg0 * BW);
#pragma unroll 1
        for (int i = 0; i < NBLK; ++i) {
          flush_rows(cnt > cap - BW, false);
          sm100::tmem_ld64(taddr + (cg0 + i) * BW, v);
          sm100::tmem_ld_wait();
          const uint32_t cbase = (uint32_t)col0 + (cg0 + i) * BW;
          const int climit = ncols - (cg0 + i) * BW;  // columns of this block that exist
          // first-level filter: d' = ||y||^2 - 2 acc, then the sign of thr - d' is
          // shifted into a mask: FFMA + FADD + funnel shift per element (element j -> bit
          // 31 - j, 1 = reject)
          uint32_t rej[2] = {0u, 0u};
#pragma unroll
          for (int j = 0; j < BW; ++j) {
            const float4 y4 = ynp[i * (BW / 4) + j / 4];
            const float y = j % 4 == 0 ? y4.x : j % 4 == 1 ? y4.y : j % 4 == 2 ? y4.z : y4.w;
            const float dp = fmaf(-2.f, __uint_as_float(v[j]), y);
            v[j] = __float_as_uint(dp);
            rej[j >> 5] = __funnelshift_l(__float_as_uint(thr_val - dp), rej[j >> 5], 1);
          }
          if (a.dout != nullptr) {  // distance-matrix mode: the block goes to global memory as it is
            if (valid) {
              float* o = a.dout + q * a.dld + cbase;
              if (climit >= BW) {
#pragma unroll
                for (int j = 0; j < BW; j += 4)
                  *reinterpret_cast<uint4*>(o + j) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
              } else {
#pragma unroll
                for (int j = 0; j < BW; ++j)
                  if (j < climit) o[j] = __uint_as_float(v[j]);
              }
            }
            continue;
          }
          uint32_t mk[2];
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int cl = climit - 32 * h;
            mk[h] = __brev(~rej[h]);
            if (cl < 32) mk[h] &= cl > 0 ? (0xFFFFFFFFu >> (32 - cl)) : 0u;
          }
          auto take = [&](float dp, uint32_t col) {  // exact key test, append to the row's buffer
            const uint64_t key = make_key(dp, col);
            if (key < thr_key) {
              if (rq) {  // sorted insertion (a full queue drops its last key); the bound is the k-th key at once
                int e = cnt < k ? cnt : k - 1;
                while (e > 0) {
                  const uint64_t pk = Rq[(e - 1) * 32];
                  if (pk < key) break;
                  Rq[e * 32] = pk;
                  --e;
                }
                Rq[e * 32] = key;
                if (cnt < k) ++cnt;
                if (cnt == k) {
                  const uint64_t t = Rq[(k - 1) * 32];
                  if (t < thr_key) {
                    thr_key = t;
                    thr_val = key_val(t);
                  }
                }
              } else {
                cb[cnt++] = key;
              }
            }
          };
          // survivors (rare once the row has a bound): each lane walks its own mask; the
          // register pick is a select tree, so the lanes of an iteration stay converged
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            uint32_t m2 = mk[h];
            while (m2) {
              const int j = __ffs(m2) - 1;
              m2 &= m2 - 1u;
              uint32_t t16[16], t8[8], t4[4], t2[2];
#pragma unroll
              for (int e = 0; e < 16; ++e) t16[e] = (j & 16) ? v[32 * h + 16 + e] : v[32 * h + e];
#pragma unroll
              for (int e = 0; e < 8; ++e) t8[e] = (j & 8) ? t16[8 + e] : t16[e];
#pragma unroll
              for (int e = 0; e < 4; ++e) t4[e] = (j & 4) ? t8[4 + e] : t8[e];
#pragma unroll
              for (int e = 0; e < 2; ++e) t2[e] = (j & 2) ? t4[2 + e] : t4[e];
              const uint32_t pv = (j & 1) ? t2[1] : t2[0];
              take(__uint_as_float(pv), cbase + 32 * h + j);
            }
          }
        }
        // accumulator drained
        sm100::tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          sm100::mbar_arrive(tempty + as);
          sm100::mbar_arrive(yempty + ys);
        }
      }
      if (a.dout != nullptr) continue;  // nothing was selected
      // establishes the split's k-th distance (published below); a single split has nobody to publish to and
      // B4 takes up to K keys per queue as they are
      if (rq) {  // the thread's queue becomes the row's buffer
        for (int e = 0; e < cnt; ++e) cb[e] = Rq[e * 32];
      } else {
        // With a sampled bound every queue already starts tight and holds ~c nb / (ns 2 S) keys at the end, about k
        // for k just above KREG: restoring half the rows of every warp (a radix selection plus three more for the
        // hierarchical bounds, row after row) to publish bounds nobody needs cost 0.3 ms of a 1.3 ms search
        // (nb = 65 536, k = 13 .. 16: slower than k = 64).  B4 takes up to K keys per queue as they are.
        flush_rows((a.S > 1 && !a.lazy_final) ? cnt >= k : cnt > K, true);
      }
      __syncwarp();
      // the row's partial queue for B4 (unordered, sentinel padded), and this split's k-th
      // distance (when a restore step has established it) as a bound for the splits to come
      for (int r = 0; r < 32; ++r) {
        if (q_warp + r >= nq) break;
        const int m = __shfl_sync(kFull, cnt, r);
        const uint64_t* buf = cb_warp + (size_t)r * cap;
        uint64_t* W = a.Wg + ((q_warp + r) * SQ + s * EPI_GROUPS + eg) * K;
        for (int i = lane; i < K; i += 32) W[i] = i < m ? buf[i] : kSentinelKey;
      }
      if (valid && cnt >= k && thr_key < thr0) atomicMin(a.gbound + q, (unsigned int)(thr_key >> 32));
      __syncwarp();
    }
  }
  // teardown (no CTA may exit while a peer can still write into it or arrive on its barriers)
  sm100::tc_fence_before();
  __syncthreads();
  if (CLUSTER > 1) sm100::cluster_sync_all();
  if (warp == MMA_WARP) {
    sm100::tc_fence_after();
    sm100::tmem_dealloc(tmem_base, 512);
  }
}

}  // namespace

// ---------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
    cudaGetLastError();
  }
  return fn;
}

// 2-D fp32 row-major [rows][d] tensor, box = box_rows x 32 columns, 128-byte swizzle,
// out-of-range rows read as zeros.
int make_map(CUtensorMap* m, const float* base, int64_t rows, int d, int box_rows) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return set_error(FS_ECUDA, "cuTensorMapEncodeTiled is not available");
  const cuuint64_t dims[2] = {(cuuint64_t)d, (cuuint64_t)(rows > 0 ? rows : 1)};
  const cuuint64_t strides[1] = {(cuuint64_t)d * sizeof(float)};
  const cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_error(FS_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return FS_OK;
}

}  // namespace

bool flat_tc_supported(int d) {
  static int forced_off = -1;
  if (forced_off < 0) {
    const char* e = getenv("FS_FLAT_ENGINE");
    forced_off = (e && strcmp(e, "ffma") == 0) ? 1 : 0;
  }
  // d need not be a multiple of the 32-column stage: the tensor maps are built on the real d, TMA fills the
  // columns of the last stage that lie beyond it with zeros, and zeros add nothing to <x, y>.  Rows must be
  // 16-byte multiples for TMA (d % 4 == 0).
  return !forced_off && d % 4 == 0 && d >= BK && d <= 128;
}

// Every extra split is one more partial queue per query (more survivors in the epilogue,
// more keys in B4): weigh it against the wave quantisation of the MMA work.
static double split_penalty(int kclass) { return kclass == 0 ? 0.002 : 0.004; }

// ---------------------------------------------------------------------------
// Sampled bound (k >= 8, nb >= 8 192).  Every partial queue of a query pays ~k ln(n / k) candidates when
// it starts without a bound, and a query has 2 S of them.  Instead a strided sample of
// ns <= min(8 192, nb / 32) rows is searched first for the query's c-th smallest distance, which
// then bounds every queue from its first tile on.  c is the smallest rank with
// P(Poisson(k ns / nb) >= c) <= 1e-7: the bound is below the true k-th distance only if c or more of the
// sample rows are among the query's k - 1 nearest.  Then fewer than k rows of the whole database pass,
// B4 sees fewer than k keys, and the query is searched again without a sampled bound (same kernel, the
// failed queries gathered, their number read on the device): exact in every case, ~c nb / ns candidates
// per query instead of ~2 S k ln(nb / (2 S k)).  FS_FLAT_SAMPLE=off disables it; =fail makes c = 1 (most
// queries fail: the tests run the re-run path with it).
// ---------------------------------------------------------------------------
static int sample_mode() {
  static int mode = -1;
  if (mode < 0) {
    const char* e = getenv("FS_FLAT_SAMPLE");
    mode = (e && strcmp(e, "off") == 0) ? 0 : (e && strcmp(e, "fail") == 0) ? 2 : 1;
  }
  return mode;
}

static int poisson_tail_rank(double lambda, double eps) {
  double term = exp(-lambda), cdf = term;  // P(X <= 0)
  int c = 1;
  while (1.0 - cdf > eps && c < 8192) {    // P(X >= c) = 1 - P(X <= c - 1)
    term *= lambda / (double)c;
    cdf += term;
    ++c;
  }
  return c;
}

static FlatTcPlan flat_tc_plan_base(int64_t nq, int64_t nb, int d, int k, bool sample_pass = false);

FlatTcPlan flat_tc_plan(int64_t nq, int64_t nb, int d, int k) {
  FlatTcPlan p = flat_tc_plan_base(nq, nb, d, k);
  p.ns = p.sstride = 0;
  p.c = 0;
  p.off_fail = p.off_failq = p.off_qfhi = p.off_qflo = p.off_sub = 0;
  // k < 8: the thread-private queues (k <= KREG) keep exact bounds from the start; nothing to gain
  if (k < 8 || sample_mode() == 0 || nb < 8192) return p;
  // Sample size: the pass costs ns / nb of the main one and the main pass sees ~c nb / ns candidates per
  // query.  ns is taken so that c <= KREG (expected hits k ns / nb <= ~1.5): the sample pass then runs on
  // the thread-private queues itself, and the candidates stay within ~10 k per query.
  int64_t ns = (int64_t)(1.5 * (double)nb / (double)k);
  if (ns > nb / 32) ns = nb / 32;
  if (ns > 8192) ns = 8192;
  ns = ns / BN * BN;
  int c = 0;
  for (; ns >= BN; ns -= BN) {
    c = sample_mode() == 2 ? 1 : poisson_tail_rank((double)k * (double)ns / (double)nb, 1e-7);
    if (c <= KREG) break;
  }
  if (ns < BN) return p;
  const int64_t stride = nb / ns;
  p.ns = ns;
  p.sstride = stride;
  p.c = c;
  size_t o = p.bytes;
  auto take = [&](size_t bytes) {
    const size_t at = o;
    o += align_up(bytes, 256);
    return at;
  };
  p.off_fail = take(256);
  p.off_failq = take((size_t)(nq + 1) * sizeof(int));
  p.off_qfhi = take((size_t)nq * d * sizeof(float));
  p.off_qflo = take((size_t)nq * d * sizeof(float));
  p.off_sub = take(flat_tc_plan_base(nq, ns, d, c, true).bytes);
  p.bytes = o;
  return p;
}

static FlatTcPlan flat_tc_plan_base(int64_t nq, int64_t nb, int d, int k, bool sample_pass) {
  FlatTcPlan p;
  p.kclass = k_class(k);
  p.K = 32 << p.kclass;
  p.qtiles = (int)ceil_div(nq, BM);
  const int64_t nt = ceil_div(nb > 0 ? nb : 1, BN);
  const int64_t sms = sm_count();
  const int64_t qgroups = ceil_div(p.qtiles, CLUSTER), ncl = sms / CLUSTER;
  p.qgroups = (int)qgroups;
  // database splits: fill whole waves of CTAs with as few partial queues as possible
  int64_t best_S = 1;
  double best = -1.0;
  const int64_t max_S = nt < 64 ? nt : 64;
  for (int64_t S = 1; S <= max_S; ++S) {
    const int64_t per = ceil_div(nt, S);
    const int64_t realS = ceil_div(nt, per);
    const int64_t items = realS * qgroups;
    const int64_t g = items < ncl ? items : ncl;
    const double eff = (double)items / (double)(ceil_div(items, g) * g) * ((double)g / (double)ncl);
    // the sample pass is short: its items' fixed costs (query tile load, pipeline fill, final restore) outweigh a
    // half-empty wave, so it takes as few items as possible
    const double score = eff - (sample_pass ? 0.05 : split_penalty(p.kclass)) * (double)realS;
    if (score > best) {
      best = score;
      best_S = realS;
    }
  }
  const int64_t per = ceil_div(nt, best_S);
  p.chunk = per * BN;
  p.chunk0 = p.chunk;
  p.S = (int)ceil_div(nb > 0 ? nb : 1, p.chunk);
  const int64_t items = (int64_t)p.S * qgroups;
  p.grid = (int)(items < ncl ? items : ncl) * CLUSTER;
  p.KB = (d + BK - 1) / BK;  // the last stage may be partial (zero-filled by TMA)
  p.cap = p.K + 128;  // the restore step runs when fewer than 64 more keys would fit
  // the kernel carves the ring at run time (the lo plane of the query tile is only
  // resident in 3xTF32 mode); worst case = with the lo plane
  const int fixed = 1024 /*alignment*/ + 1024 /*barriers*/ + YN_RING * BN * 4 + SCRATCH_BYTES + 2 * p.KB * A_KB_BYTES;
  int st = (SMEM_LIMIT - fixed) / B_STAGE_BYTES;
  p.nstage = st > MAX_STAGES ? MAX_STAGES : st;
  p.smem = SMEM_LIMIT;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    const size_t at = o;
    o += align_up(bytes, 256);
    return at;
  };
  p.off_ynorm = take((size_t)(nb + 2 * BN) * sizeof(float));
  p.off_xnorm = take((size_t)(nq + 1) * sizeof(float));
  p.off_flag = take(256);
  p.off_gbound = take((size_t)(nq + 1) * sizeof(unsigned int));
  p.off_hbound = take((size_t)(nq + 1) * HB_SLOTS * sizeof(unsigned int));
  p.off_hclaim = take((size_t)(nq + 1) * HB_LEVELS * sizeof(unsigned int));
  p.off_W = take((size_t)nq * p.S * EPI_GROUPS * p.K * sizeof(uint64_t));
  p.off_cbuf = take((size_t)sms * EPI_GROUPS * BM * p.cap * sizeof(uint64_t));
  p.off_qhi = take((size_t)nq * d * sizeof(float));
  p.off_qlo = take((size_t)nq * d * sizeof(float));
  p.off_bhi = take((size_t)nb * d * sizeof(float));
  p.off_blo = take((size_t)nb * d * sizeof(float));
  p.bytes = o;
  return p;
}

// ---------------------------------------------------------------------------
// Prepared database: the database's share of the pre-pass (norms, lo flag, lo plane) is query-independent
// -- 0.45 ms of every cfg3 call.  fs_flat_prepare does it once into a block of the caller's.
// The lo plane is always written (zeros for TF32-representable data): whether it is read is decided per call
// by the database's flag OR the queries'.
// ---------------------------------------------------------------------------
static size_t prep_ynorm_bytes(int64_t nb) { return align_up((size_t)(nb + 2 * BN) * sizeof(float), 256); }

size_t flat_prep_bytes(int64_t nb, int d) {
  size_t b = 256 + prep_ynorm_bytes(nb);
  if (flat_tc_supported(d)) b += align_up((size_t)nb * d * sizeof(float), 256);
  return b;
}

FlatPrep flat_prep_view(const void* prep, int64_t nb, int d) {
  const char* w = static_cast<const char*>(prep);
  FlatPrep v;
  v.ynorm = reinterpret_cast<const float*>(w + 256);
  const bool tc = flat_tc_supported(d);
  v.flag = tc ? reinterpret_cast<const unsigned int*>(w) : nullptr;
  v.blo = tc ? reinterpret_cast<const float*>(w + 256 + prep_ynorm_bytes(nb)) : nullptr;
  return v;
}

int flat_prepare_device(const float* xb, int64_t nb, int d, void* prep, cudaStream_t s) {
  char* w = static_cast<char*>(prep);
  float* ynorm = reinterpret_cast<float*>(w + 256);
  FS_CUDA(cudaMemsetAsync(w, 0, 256, s));
  if (nb == 0) return FS_OK;
  if (!flat_tc_supported(d)) return launch_row_norms(xb, nb, d, ynorm, s);
  unsigned int* flag = reinterpret_cast<unsigned int*>(w);
  float* blo = reinterpret_cast<float*>(w + 256 + prep_ynorm_bytes(nb));
  FS_CUDA(cudaMemsetAsync(w + 4, 0x01, 4, s));  // word 1: a non-zero word for the unconditional lo-plane pass
  norm_flag_kernel<<<(unsigned)ceil_div(nb, 8), 256, 0, s>>>(xb, nb, d, ynorm, flag);
  FS_LAUNCHED();
  const int64_t nbe = nb * d;
  const int sms = sm_count();
  lo_plane_kernel<<<(unsigned)(ceil_div(nbe, 1024) < sms * 8 ? ceil_div(nbe, 1024) : sms * 8), 256, 0, s>>>(xb, nbe, blo, flag + 1);
  FS_LAUNCHED();
  return FS_OK;
}

int flat_knn_tc_device(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k, float* out_dist,
                       int64_t* out_ids, void* ws, cudaStream_t s, float* dout, int64_t dld, const FlatPrep* prep) {
  if (dout != nullptr) k = 1;  // distance-matrix mode: the plan of the cheapest queue class
  // a database that TMA cannot read in place needs its truncated copy made per call: the prepared block has none
  if (prep != nullptr && (prep->flag == nullptr || (reinterpret_cast<uintptr_t>(xb) & 15u) != 0)) prep = nullptr;
  const FlatTcPlan p = flat_tc_plan(nq, nb, d, k);
  if (p.nstage < 2) return set_error(FS_EUNSUPPORTED, "flat tensor-core engine: d = %d leaves no room for the stage ring", d);
  char* w = static_cast<char*>(ws);
  const float* ynorm = prep ? prep->ynorm : reinterpret_cast<float*>(w + p.off_ynorm);
  float* xnorm = reinterpret_cast<float*>(w + p.off_xnorm);
  unsigned int* flag = reinterpret_cast<unsigned int*>(w + p.off_flag);
  unsigned int* gbound = reinterpret_cast<unsigned int*>(w + p.off_gbound);
  float* qhi = reinterpret_cast<float*>(w + p.off_qhi);
  float* qlo = reinterpret_cast<float*>(w + p.off_qlo);
  float* bhi = reinterpret_cast<float*>(w + p.off_bhi);
  const float* blo = prep ? prep->blo : reinterpret_cast<float*>(w + p.off_blo);
  FS_CUDA(cudaMemsetAsync(flag, 0, 256, s));
  if (prep) FS_CUDA(cudaMemcpyAsync(flag, prep->flag, sizeof(unsigned int), cudaMemcpyDeviceToDevice, s));  // the queries OR theirs in
  // +inf image and above: no bound (gbound and hbound are adjacent); no slot handed out yet
  FS_CUDA(cudaMemsetAsync(gbound, 0xFF, p.off_hclaim - p.off_gbound, s));
  FS_CUDA(cudaMemsetAsync(w + p.off_hclaim, 0, (size_t)(nq + 1) * HB_LEVELS * sizeof(unsigned int), s));
  if (!prep) {
    norm_flag_kernel<<<(unsigned)ceil_div(nb, 8), 256, 0, s>>>(xb, nb, d, reinterpret_cast<float*>(w + p.off_ynorm), flag);
    FS_LAUNCHED();
  }
  norm_flag_kernel<<<(unsigned)ceil_div(nq, 8), 256, 0, s>>>(xq, nq, d, xnorm, flag);
  FS_LAUNCHED();
  const int64_t nbe = nb * d, nqe = nq * d;
  const int sms = sm_count();
  // lo planes only if some lo is non-zero (decided on the device: the kernels return at once otherwise)
  if (!prep) {
    lo_plane_kernel<<<(unsigned)(ceil_div(nbe, 1024) < sms * 8 ? ceil_div(nbe, 1024) : sms * 8), 256, 0, s>>>(
        xb, nbe, reinterpret_cast<float*>(w + p.off_blo), flag);
    FS_LAUNCHED();
  }
  lo_plane_kernel<<<(unsigned)(ceil_div(nqe, 1024) < sms * 8 ? ceil_div(nqe, 1024) : sms * 8), 256, 0, s>>>(xq, nqe, qlo, flag);
  FS_LAUNCHED();
  // hi planes: the operands themselves (the MMA ignores the 13 low mantissa bits) unless they are misaligned for TMA
  static int force_planes = -1;  // FS_TC_PLANES=1: explicit truncated copies (A/B check of the truncation claim)
  if (force_planes < 0) {
    const char* e = getenv("FS_TC_PLANES");
    force_planes = (e && e[0] == '1') ? 1 : 0;
  }
  const float* a_hi = xq;
  const float* b_hi = xb;
  if (force_planes || (reinterpret_cast<uintptr_t>(xq) & 15u) != 0) {
    hi_plane_kernel<<<(unsigned)(ceil_div(nqe, 256) < sms * 8 ? ceil_div(nqe, 256) : sms * 8), 256, 0, s>>>(xq, nqe, qhi);
    FS_LAUNCHED();
    a_hi = qhi;
  }
  if (force_planes || (reinterpret_cast<uintptr_t>(xb) & 15u) != 0) {
    hi_plane_kernel<<<(unsigned)(ceil_div(nbe, 256) < sms * 8 ? ceil_div(nbe, 256) : sms * 8), 256, 0, s>>>(xb, nbe, bhi);
    FS_LAUNCHED();
    b_hi = bhi;
  }

  CUtensorMap ma_hi, ma_lo, mb_hi, mb_lo;
  int rc;
  if ((rc = make_map(&ma_hi, a_hi, nq, d, BM)) != FS_OK || (rc = make_map(&ma_lo, qlo, nq, d, BM)) != FS_OK ||
      (rc = make_map(&mb_hi, b_hi, nb, d, BN / CLUSTER)) != FS_OK ||
      (rc = make_map(&mb_lo, blo, nb, d, BN / CLUSTER)) != FS_OK)
    return rc;
  FS_CUDA(cudaFuncSetAttribute(flat_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem));  // per device
  // one launch of the tile kernel: plan pl over a database of n rows seen through (m_bhi, m_blo), queries
  // through (m_ahi, m_alo), workspace region wr laid out by pl
  auto run_tiles = [&](const FlatTcPlan& pl, char* wr, int64_t n, int kk, const float* yn, const CUtensorMap& m_ahi,
                       const CUtensorMap& m_alo, const CUtensorMap& m_bhi, const CUtensorMap& m_blo,
                       const unsigned int* nq_dev, unsigned int* gb) -> int {
    TcArgs a;
    a.nq = nq;
    a.nb = n;
    a.d = d;
    a.KB = pl.KB;
    a.k = kk;
    a.kclass = pl.kclass;
    a.K = pl.K;
    a.S = pl.S;
    a.qtiles = pl.qtiles;
    a.qgroups = pl.qgroups;
    a.cap = pl.cap;
    a.smem_bytes = (int)pl.smem;
    a.chunk = pl.chunk;
    a.chunk0 = pl.chunk0;
    a.ynorm = yn;
    a.Wg = reinterpret_cast<uint64_t*>(wr + pl.off_W);
    a.gbound = gb;
    a.hbound = reinterpret_cast<unsigned int*>(wr + pl.off_hbound);
    a.hclaim = reinterpret_cast<unsigned int*>(wr + pl.off_hclaim);
    a.cbuf = reinterpret_cast<uint64_t*>(wr + pl.off_cbuf);
    a.lo_flag = flag;
    a.lazy_final = (p.ns > 0 && dout == nullptr && &pl == &p && nq_dev == nullptr) ? 1 : 0;  // main pass over a sampled bound
    a.nq_dev = nq_dev;
    a.dout = dout;
    a.dld = dld;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)pl.grid);
    cfg.blockDim = dim3(TC_THREADS);
    cfg.dynamicSmemBytes = pl.smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CLUSTER;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    FS_CUDA(cudaLaunchKernelEx(&cfg, flat_tc_kernel, m_ahi, m_alo, m_bhi, m_blo, a));
    FS_LAUNCHED();
    return FS_OK;
  };
  const bool sampled = p.ns > 0 && dout == nullptr;
  if (sampled) {
    // the sample pass: the c-th smallest d' over every sstride-th row becomes gbound[q]
    const FlatTcPlan sub = flat_tc_plan_base(nq, p.ns, d, p.c, true);
    char* w2 = w + p.off_sub;
    float* yn_s = reinterpret_cast<float*>(w2 + sub.off_ynorm);
    unsigned int* gb_s = reinterpret_cast<unsigned int*>(w2 + sub.off_gbound);
    float* s_hi = reinterpret_cast<float*>(w2 + sub.off_bhi);
    float* s_lo = reinterpret_cast<float*>(w2 + sub.off_blo);
    gather_sample_kernel<<<(unsigned)ceil_div(p.ns, 8), 256, 0, s>>>(b_hi, blo, ynorm, p.sstride, p.ns, d, flag, s_hi, s_lo, yn_s);
    FS_LAUNCHED();
    FS_CUDA(cudaMemsetAsync(gb_s, 0xFF, sub.off_hclaim - sub.off_gbound, s));
    FS_CUDA(cudaMemsetAsync(w2 + sub.off_hclaim, 0, (size_t)(nq + 1) * HB_LEVELS * sizeof(unsigned int), s));
    CUtensorMap ms_hi, ms_lo;
    if ((rc = make_map(&ms_hi, s_hi, p.ns, d, BN / CLUSTER)) != FS_OK ||
        (rc = make_map(&ms_lo, s_lo, p.ns, d, BN / CLUSTER)) != FS_OK)
      return rc;
    if ((rc = run_tiles(sub, w2, p.ns, p.c, yn_s, ma_hi, ma_lo, ms_hi, ms_lo, nullptr, gb_s)) != FS_OK) return rc;
    FinishExtra ex;
    ex.packed = true;
    ex.bound_out = gbound;
    if ((rc = launch_flat_finish(reinterpret_cast<uint64_t*>(w2 + sub.off_W), nq, sub.S * EPI_GROUPS, p.c, nullptr, nullptr,
                                 nullptr, s, &ex)) != FS_OK)
      return rc;
  }
  if ((rc = run_tiles(p, w, nb, k, ynorm, ma_hi, ma_lo, mb_hi, mb_lo, nullptr, gbound)) != FS_OK) return rc;
  if (dout != nullptr) return FS_OK;
  uint64_t* Wg = reinterpret_cast<uint64_t*>(w + p.off_W);
  FinishExtra ex0;
  ex0.packed = true;
  if (!sampled) return launch_flat_finish(Wg, nq, p.S * EPI_GROUPS, k, xnorm, out_dist, out_ids, s, &ex0);
  // B4 with the check of the sampled bound, then the failed queries once more without one
  unsigned int* fail_cnt = reinterpret_cast<unsigned int*>(w + p.off_fail);
  int* fail_q = reinterpret_cast<int*>(w + p.off_failq);
  float* qf_hi = reinterpret_cast<float*>(w + p.off_qfhi);
  float* qf_lo = reinterpret_cast<float*>(w + p.off_qflo);
  FS_CUDA(cudaMemsetAsync(fail_cnt, 0, 256, s));
  FinishExtra ex;
  ex.packed = true;
  ex.fail_cnt = fail_cnt;
  ex.fail_q = fail_q;
  ex.need = (int)((int64_t)k < nb ? k : nb);
  if ((rc = launch_flat_finish(Wg, nq, p.S * EPI_GROUPS, k, xnorm, out_dist, out_ids, s, &ex)) != FS_OK) return rc;
  gather_failed_kernel<<<(unsigned)ceil_div(nq, 8), 256, 0, s>>>(a_hi, qlo, d, fail_cnt, fail_q, flag, qf_hi, qf_lo);
  FS_LAUNCHED();
  FS_CUDA(cudaMemsetAsync(gbound, 0xFF, p.off_hclaim - p.off_gbound, s));
  FS_CUDA(cudaMemsetAsync(w + p.off_hclaim, 0, (size_t)(nq + 1) * HB_LEVELS * sizeof(unsigned int), s));
  CUtensorMap mf_hi, mf_lo;
  if ((rc = make_map(&mf_hi, qf_hi, nq, d, BM)) != FS_OK || (rc = make_map(&mf_lo, qf_lo, nq, d, BM)) != FS_OK) return rc;
  if ((rc = run_tiles(p, w, nb, k, ynorm, mf_hi, mf_lo, mb_hi, mb_lo, fail_cnt, gbound)) != FS_OK) return rc;
  FinishExtra ex2;
  ex2.packed = true;
  ex2.nq_dev = fail_cnt;
  ex2.qmap = fail_q;
  return launch_flat_finish(Wg, nq, p.S * EPI_GROUPS, k, xnorm, out_dist, out_ids, s, &ex2);
}

}  // namespace fs
