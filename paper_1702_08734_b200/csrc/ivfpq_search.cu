// ivfpq_search.cu -- fs_ivfpq_search: Alg. 4, SURVEY 8a rows C1-C5.
//
//   C1 coarse quantizer  L_IVF = tau-argmin_c ||x - c||^2 (Eq. 5): the exact-search engine over
//                        the centroids with k = nprobe (P:L308 takes term 2 of Eq. 11 from here, "a
//                        by-product of the first-level quantizer"; this scan recomputes it, see C2)
//   C2 lookup tables     Eq. 11 pushed one step further than the paper's table layout:
//                        ||x - q1(y) - q2(y)||^2 = ||x - q1||^2            term 2: per (query, list), recomputed by the
//                                                                          scan in the direct form sum (x - c)^2
//                                                                          (C1's Eq. 2 value loses ~1e-5 relative
//                                                                          to cancellation; 96 flops per list)
//                                               + ||q2||^2 + 2 <q1, q2>    term 1: per STORED VECTOR, computed when
//                                                                          it is added (ivfpq.cu, fs_ivfpq::s1)
//                                               - 2 <x, q2>                term 3: sum_m T_m[code_m],
//                        T_m[c] = -2 <x^m, B[m][c]>: ONE table per QUERY (ivfpq_qtable_kernel), independent
//                        of the list, so no table is built per (query, list) pair at all (the paper
//                        stores term 1 per (list, code), 1 GB at 65 536 lists, and still combines a
//                        table per pair; here term 1 costs 4 bytes per vector and the scan
//                        adds it to the sum of look-ups).  M = 8 / 16.  Other M: tables from scratch
//                        (Eq. 10) in shared memory per pair, ivfpq_scan_kernel.
//   C3 list scan         dist = term 2 + term 1 + sum_m T_m[code_m] over the list's codes, streamed from
//                        HBM (Alg. 4).  The table is FIXED-POINT and stored as lut[c][b],
//                        b = 0..31: word (c, b) lives in shared-memory bank b and holds T_{b mod M}[c]
//                        (32 / M replicas); lane l adds its sub-quantizers in the order m = (s ^ l) mod M,
//                        so every look-up is one wavefront at bank l ^ s; the codes are stored in that
//                        order per list position (ivfpq.cu), so the scan does no byte shuffling.  Integer
//                        sums are exact and order-independent: identical codes give identical distances
//                        (reading C-6), and integer-valued data stay exact.
//   C4 pass-1 selection  fused: every warp k-selects the distances it produces in a register queue; a
//                        CTA covers a GROUP of G probed lists of one query, so one partial list of k
//                        leaves the SM per group (the paper writes all distances out first, P:L319-321,
//                        and found the fused form <= 15 % faster on Maxwell)
//   C5 pass-2 + ids      the groups' partial lists are selected again to k; int64 ids are fetched for
//                        the winners only
#include <cstdlib>
#include <algorithm>
#include <cstring>

#include "flat.cuh"
#include "ivfpq.cuh"
#include "ivfpq_scan.cuh"
#include "select.cuh"

namespace fs {

// kselect.cu
size_t kselect_ws_bytes(int64_t n_rows, int64_t n, int k);
int kselect_device(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                   int32_t* out_idx, void* ws, cudaStream_t s, bool largest);

namespace {
constexpr int SCAN_WARPS = 8;
constexpr int SCAN_THREADS = SCAN_WARPS * 32;

// ---------------------------------------------------------------------------
// Any M: tables from scratch per (query, list) pair (Eq. 10), float, natural byte order.
// Shared memory: T[M][256] | r[d] | per-warp batches | merge area [SCAN_WARPS][K]
// ---------------------------------------------------------------------------
template <int NQ>
__global__ void __launch_bounds__(SCAN_THREADS) ivfpq_scan_kernel(const ScanArgs a) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  float* T = reinterpret_cast<float*>(scan_smem);
  float* r = T + a.M * 256;
  uint64_t* bufs = reinterpret_cast<uint64_t*>(r + ((a.d + 3) & ~3));
  uint64_t* merge = bufs + SCAN_WARPS * warp_select_smem_keys<NB>();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t q = blockIdx.x / a.ngroups;
  const int g = (int)(blockIdx.x - q * a.ngroups);
  const int p_begin = g * a.G;
  const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;
  const int M = a.M, dsub = a.dsub, d = a.d;

  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  unsigned long long bytes = 0;
  // the CTA's K-th distance is <= every warp's K-th: the smallest one published bounds all warps
  __shared__ uint32_t cta_bound;
  if (tid == 0) cta_bound = 0x7F800000u;

  for (int p = p_begin; p < p_end; ++p) {
    const int64_t L = a.probe_ids[q * a.nprobe + p];
    if (a.out_probed && tid == 0) a.out_probed[q * a.nprobe + p] = (int32_t)L;
    if (L < 0) continue;  // fewer than nprobe centroids: cannot happen (nprobe <= nlist)
    const int64_t lb = a.offsets[L], le = a.offsets[L + 1];
    const int64_t len = le - lb;
    if (len == 0) continue;  // empty lists are probed and contribute nothing
    __syncthreads();         // previous list's table is no longer read
    const uint8_t* cl = a.codes + lb * M;
    // C2: residual and tables
    for (int j = tid; j < d; j += SCAN_THREADS) r[j] = a.xq[q * d + j] - a.coarse[L * d + j];
    __syncthreads();
    for (int e = tid; e < M * 256; e += SCAN_THREADS) {
      const int m = e >> 8;
      const float* b = a.pq + (int64_t)e * dsub;
      const float* rm = r + m * dsub;
      float acc = 0.f;
      for (int j = 0; j < dsub; ++j) {
        const float t = rm[j] - b[j];
        acc = fmaf(t, t, acc);
      }
      T[e] = acc;
    }
    __syncthreads();
    // C3 + C4: scan and select
    bytes += (unsigned long long)len * M;
    // 32-bit indices inside a piece of at most 2^30 vectors (one piece unless a list is enormous)
    for (int64_t c0 = 0; c0 < len; c0 += (int64_t)1 << 30) {
      const int n = (int)((len - c0) < ((int64_t)1 << 30) ? (len - c0) : ((int64_t)1 << 30));
      const uint8_t* cc = cl + c0 * M;
      const uint32_t pos0 = (uint32_t)(lb + c0);
      for (int v0 = 0; v0 < n; v0 += SCAN_THREADS) {
        const int v = v0 + tid;
        const bool ok = v < n;
        float dist = 0.f;
        if (ok) {
          const uint8_t* cv = cc + (size_t)(uint32_t)v * M;
          if ((M & 3) == 0) {
            const uint32_t* cw = reinterpret_cast<const uint32_t*>(cv);
            for (int w = 0; w < (M >> 2); ++w) {
              const uint32_t c = cw[w];
              const float* Tw = T + (w << 10);
              dist += Tw[c & 255u];
              dist += Tw[256 + ((c >> 8) & 255u)];
              dist += Tw[512 + ((c >> 16) & 255u)];
              dist += Tw[768 + (c >> 24)];
            }
          } else {
            for (int m = 0; m < M; ++m) dist += T[(m << 8) + cv[m]];
          }
        }
        const float bound = fminf(sel.thr_val, __uint_as_float(*reinterpret_cast<volatile uint32_t*>(&cta_bound)));
        const bool cand = ok && !(dist > bound);
        if (__any_sync(kFull, cand)) {  // the exact key is only built when some lane may have a winner
          const uint64_t key = make_key(dist, pos0 + (uint32_t)v);
          const uint64_t thr_before = sel.thr;
          sel.push(cand && sel.wants(key), key);
          if (sel.thr != thr_before && lane == 0) atomicMin(&cta_bound, __float_as_uint(sel.thr_val));
        }
      }
    }
  }
  sel.finish();
  if (tid == 0 && bytes) atomicAdd(a.scanned, bytes);

  // merge the warps' queues: warp 0 selects again over SCAN_WARPS * K keys
  __syncthreads();
#pragma unroll
  for (int rr = 0; rr < NQ; ++rr) merge[warp * K + rr * 32 + lane] = sel.W[rr];
  __syncthreads();
  if (warp == 0) {
    sel.reset();
    for (int e0 = 0; e0 < SCAN_WARPS * K; e0 += 32) {
      const uint64_t key = merge[e0 + lane];
      sel.push(key < sel.thr, key);
    }
    sel.finish();
    uint64_t* W = a.Wg + (int64_t)blockIdx.x * K;
#pragma unroll
    for (int rr = 0; rr < NQ; ++rr) W[rr * 32 + lane] = sel.W[rr];
  }
}

__global__ void pq_bmax_kernel(const float* __restrict__ pq, float* __restrict__ bmax, int dsub) {
  const int m = blockIdx.x, lane = threadIdx.x;  // one warp per sub-quantizer
  float mx = 0.f;
  for (int c = lane; c < 256; c += 32) {
    float n = 0.f;
    for (int j = 0; j < dsub; ++j) {
      const float v = pq[((int64_t)m * 256 + c) * dsub + j];
      n = fmaf(v, v, n);
    }
    mx = fmaxf(mx, n);
  }
  for (int sft = 16; sft >= 1; sft >>= 1) mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, sft));
  if (lane == 0) bmax[m] = sqrtf(mx);
}


// ---------------------------------------------------------------------------
// M = 8 / 16.  Per query: the term-3 table T_m[c] = -2 <x^m, B[m][c]> in fixed point, ||x||^2, and
// the constants that turn an integer sum of look-ups back into a distance.
//   |T_m[c]| <= 2 ||x^m|| max_c ||B[m][c]|| =: b_m, so T_m[c] + b_m >= 0; one power-of-two scale per
//   query makes every entry (T_m[c] + b_m) * scale an integer < 2^27 (b_m rounded up to a multiple of
//   1 / scale first, so that integer-valued inputs stay exact); the sum of a vector's M entries minus
//   isum = sum_m b_m * scale, times 1 / scale, is term 3.
// Tq[q] is written in the LANE ORDER of the scan kernel's table build: element (c / REP) * 32 +
// (c % REP) * M + m, REP = 32 / M, so that a warp reads 32 consecutive words and its stores of the
// replicated table are conflict-free.
// ---------------------------------------------------------------------------
constexpr int QT_QPB = 8;  // queries per block of ivfpq_qtable_kernel

struct QMeta {
  float inv_scale;  // 2^-se
  uint32_t isum;    // sum_m b_m * 2^se (exact integer)
  float xnorm;      // ||x||^2 (added to C1's distances when they come without it)
  float pad;
};

template <int M>
__global__ void __launch_bounds__(256) ivfpq_qtable_kernel(const float* __restrict__ xq, const float* __restrict__ pq,
                                                           const float* __restrict__ bmax, int d, int dsub,
                                                           uint32_t* __restrict__ Tq, QMeta* __restrict__ meta,
                                                           int64_t nq, int qpb) {
  constexpr int REP = 32 / M;
  __shared__ float x[2048];
  __shared__ float bm[M];
  __shared__ float xn_s;
  // the table is staged in shared memory (word o at o + o / 32: the stores of a warp -- 32 entries c of one m,
  // 16 words apart -- fall in 32 different banks) and leaves in whole 128-byte lines; a block takes qpb queries
  // one after the other, so that the codebook (M x 256 x dsub floats) is read from L2 once per block
  __shared__ uint32_t stg[256 * M + 8 * M];
  const int tid = threadIdx.x, lane = tid & 31;
  for (int qi = 0; qi < qpb; ++qi) {
  const int64_t q = (int64_t)blockIdx.x * qpb + qi;
  if (q >= nq) break;
  for (int j = tid; j < d; j += 256) x[j] = xq[q * d + j];
  __syncthreads();
  if (tid < 32) {  // warp 0: ||x^m|| for m = lane (< M), ||x||^2
    float n = 0.f;
    if (lane < M)
      for (int j = 0; j < dsub; ++j) n = fmaf(x[lane * dsub + j], x[lane * dsub + j], n);
    if (lane < M) bm[lane] = 2.f * sqrtf(n) * bmax[lane] * 1.0001f;
    float xn = 0.f;  // dimension order, as the flat engine's norms
    if (lane == 0) {
      for (int j = 0; j < d; ++j) xn = fmaf(x[j], x[j], xn);
      xn_s = xn;
    }
  }
  __syncthreads();
  float u = 0.f;
#pragma unroll
  for (int m = 0; m < M; ++m) u = fmaxf(u, bm[m]);
  int ex = 0;
  if (u > 0.f && u < 3.0e38f) frexpf(2.f * u, &ex);  // entries < 2 b_m <= 2 u < 2^ex
  int se = 27 - ex;
  se = se > 100 ? 100 : (se < -100 ? -100 : se);
  const float scale = __uint_as_float((uint32_t)(127 + se) << 23);
  uint32_t bi[M], isum = 0;
#pragma unroll
  for (int m = 0; m < M; ++m) {
    bi[m] = (uint32_t)ceilf(bm[m] * scale);  // b_m rounded up to a multiple of 1 / scale
    isum += bi[m];
  }
  // thread c builds entry c of every table
  const int c = tid;
  for (int m = 0; m < M; ++m) {
    const float* b = pq + ((int64_t)m * 256 + c) * dsub;
    float acc = 0.f;
    for (int j = 0; j < dsub; ++j) acc = fmaf(x[m * dsub + j], b[j], acc);
    const float t = -2.f * acc * scale + (float)bi[m];  // exact for integer-valued inputs
    const int o = (c / REP) * 32 + (c % REP) * M + m;
    stg[o + (o >> 5)] = __float2uint_rn(fmaxf(t, 0.f));
  }
  if (tid == 0) {
    QMeta mt;
    mt.inv_scale = __uint_as_float((uint32_t)(127 - se) << 23);
    mt.isum = isum;
    mt.xnorm = xn_s;
    mt.pad = 0.f;
    meta[q] = mt;
  }
  __syncthreads();
  for (int o = tid; o < 256 * M; o += 256) Tq[q * (256 * M) + o] = stg[o + (o >> 5)];
  __syncthreads();  // the next query overwrites x, bm and the staged table
  }
}

// acc += lut[byte s of w][bank lane ^ s] for s = 0 .. M-1; A = table + 4 * lane (table 128-byte aligned).
// The code words are in the list's stored order: byte s holds sub-quantizer (s ^ lane) mod M.
template <int s, int M>
__device__ __forceinline__ void xor_gather(const uint32_t* w, uint32_t A, uint32_t& acc) {
  if constexpr (s < M) {
    const uint32_t c = __byte_perm(w[s >> 2], 0u, 0x4440u + (s & 3));  // byte s, zero-extended
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((A ^ (4u * s)) + c * 128u));
    acc += v;
    xor_gather<s + 1, M>(w, A, acc);
  }
}

// The same for VPL vectors at once (independent chains).  As[s] = A ^ 4 s is kept in registers; the
// address is one IMAD and the sum one IMAD too (FMA pipe), so that the ALU pipe -- the busiest one of
// this kernel, 67 % in the first version -- only extracts the byte.
template <int s, int M, int VPL>
__device__ __forceinline__ void xor_gather_n(const uint32_t (&w)[VPL][M / 4], const uint32_t (&As)[M], uint32_t (&acc)[VPL]) {
  if constexpr (s < M) {
    uint32_t ad[VPL], v[VPL];
#pragma unroll
    for (int u = 0; u < VPL; ++u) {
      const uint32_t c = __byte_perm(w[u][s >> 2], 0u, 0x4440u + (s & 3));  // byte s, zero-extended
      asm("mad.lo.u32 %0, %1, 128, %2;" : "=r"(ad[u]) : "r"(c), "r"(As[s]));
    }
#pragma unroll
    for (int u = 0; u < VPL; ++u) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[u]) : "r"(ad[u]));
#pragma unroll
    for (int u = 0; u < VPL; ++u) asm("mad.lo.u32 %0, %1, 1, %0;" : "+r"(acc[u]) : "r"(v[u]));
    xor_gather_n<s + 1, M, VPL>(w, As, acc);
  }
}

// The scan of M = 8 / 16 indexes.  Persistent CTAs of 8 warps draw (query, list group) items from a
// counter; per item the query's table is copied from Tq into the replicated shared-memory layout (16
// loads and 16 x REP stores per thread), then the warps stream the group's lists: one 8 / 16-byte code
// load and one 4-byte term-1 load per vector, M look-ups, one FMA, the selection.
// Shared memory: lut[256][32] (the merge area aliases it) | select batches.
#ifndef FS_QS_CTAS
#define FS_QS_CTAS 4
#endif
constexpr int QS_CTAS = FS_QS_CTAS;  // CTAs per SM (K <= 128): 4 x 8 warps, 64 registers

template <int NQ>
constexpr int qs_ctas() { return NQ <= 4 ? QS_CTAS : (NQ <= 8 ? 2 : 1); }  // the register queue grows with K = 32 NQ
constexpr int QS_MAXG = 128;  // lists per work item (their bounds, term 2 and pass prefix sit in shared memory)

template <int NQ>
constexpr size_t qs_smem_bytes(int d) {
  return (size_t)256 * 32 * 4 + (size_t)SCAN_WARPS * warp_select_smem_keys<2>() * 8 + (size_t)2 * SCAN_WARPS * 32 * NQ * 8 +
         (size_t)QS_MAXG * 16 + 0 * (size_t)d;
}

template <int NQ, int M>
__global__ void __launch_bounds__(SCAN_THREADS, qs_ctas<NQ>())
    ivfpq_scan_q_kernel(const ScanArgs a, const uint32_t* __restrict__ Tq, const QMeta* __restrict__ meta,
                        unsigned int* __restrict__ work, int64_t n_items) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int VPL = M == 8 ? 4 : 2;  // vectors per lane and pass
  constexpr int PV = 32 * VPL;         // vectors per pass
  // Shared memory: lut[256][32] | select batches | merge areas [2][SCAN_WARPS][K] (warp 0 merges one item's
  // queues while the warps park the next item's in the other) | per list: begin, length, term 2, first pass
  uint32_t* lut = reinterpret_cast<uint32_t*>(scan_smem);
  uint64_t* bufs = reinterpret_cast<uint64_t*>(lut + 256 * 32);
  uint64_t* merge = bufs + SCAN_WARPS * warp_select_smem_keys<NB>();
  uint32_t* l_begin = reinterpret_cast<uint32_t*>(merge + 2 * SCAN_WARPS * K);  // CSR position of the list's first vector
  int* l_len = reinterpret_cast<int*>(l_begin + QS_MAXG);
  float* l_t2 = reinterpret_cast<float*>(l_len + QS_MAXG);
  int* l_pass = reinterpret_cast<int*>(l_t2 + QS_MAXG);  // passes (of PV vectors) before this list
  __shared__ uint32_t cta_bound;
  __shared__ float cta_sub[SCAN_WARPS];  // each warp's ceil(k / 8)-th smallest distance
  __shared__ int cta_item, cta_pass, cta_npass;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  unsigned long long bytes = 0;
  const int my_m = lane % M, cofs = lane / M;
  const uint32_t lane_base = (uint32_t)__cvta_generic_to_shared(lut) + ((uint32_t)lane << 2);  // step s reads bank lane ^ s
  uint32_t As[M];
#pragma unroll
  for (int i = 0; i < M; ++i) As[i] = lane_base ^ (4u * i);
  const int d = a.d;
  int64_t prev_item = -1;  // warp 0: the item whose queues wait in the merge area
  int round = 0;           // items this CTA has scanned: parity picks the merge area

  while (true) {
    __syncthreads();  // A: every warp has scanned its share of the previous item and parked its queue
    if (tid == 0) {
      cta_item = (int)atomicAdd(work, 1u);
      cta_bound = 0x7F800000u;
      cta_pass = 0;
    }
    if (tid < SCAN_WARPS) cta_sub[tid] = __uint_as_float(0x7F800000u);
    __syncthreads();
    const int64_t item = cta_item;
    const bool live = item < n_items;
    int nl = 0;
    int64_t q = 0;
    int p_begin = 0;
    QMeta mt = {};
    if (live) {
      q = item / a.ngroups;
      const int g = (int)(item - q * a.ngroups);
      p_begin = g * a.G;
      const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;
      nl = p_end - p_begin;
      mt = meta[q];
      // C2: the query's table into the replicated, bank-aligned layout
      const uint32_t* tq = Tq + q * (256 * M);
#pragma unroll 4
      for (int i = warp; i < 256 / REP; i += SCAN_WARPS) {
        const uint32_t v = __ldg(tq + i * 32 + lane);
        const int c = i * REP + cofs;
#pragma unroll
        for (int rep = 0; rep < REP; ++rep) lut[c * 32 + my_m + ((rep + cofs) % REP) * M] = v;
      }
      // the lists of the item: bounds and term 2, ||x - c_L||^2 in the direct form (C1's value went through
      // the Eq. 2 expansion, whose cancellation error is absolute, ~1e-7 (||x||^2 + ||c||^2), and would be the
      // largest one in the distance of a close vector); one warp per list, fixed summation order
      const float* xq = a.xq + q * d;
      for (int j = warp; j < nl; j += SCAN_WARPS) {
        const int64_t L = a.probe_ids[q * a.nprobe + p_begin + j];
        int64_t lb = 0, le = 0;
        float t2 = 0.f;
        if (L >= 0) {
          lb = a.offsets[L];
          le = a.offsets[L + 1];
          for (int i = lane; i < d; i += 32) {
            const float df = xq[i] - a.coarse[L * d + i];
            t2 = fmaf(df, df, t2);
          }
        }
#pragma unroll
        for (int sft = 16; sft >= 1; sft >>= 1) t2 += __shfl_xor_sync(kFull, t2, sft);
        if (lane == 0) {
          l_begin[j] = (uint32_t)lb;
          l_len[j] = (int)(le - lb);
          l_t2[j] = t2;
          if (a.out_probed) a.out_probed[q * a.nprobe + p_begin + j] = (int32_t)L;
        }
      }
    }
    __syncthreads();  // B: table and list records are in place
    if (warp == 0) {
      if (live) {  // exclusive prefix of the lists' pass counts (nl <= QS_MAXG = 4 x 32)
        int run = 0;
        unsigned long long by = 0;
        for (int j0 = 0; j0 < nl; j0 += 32) {
          const int j = j0 + lane;
          const int n = j < nl ? (l_len[j] + PV - 1) / PV : 0;
          if (j < nl) by += (unsigned long long)l_len[j] * M;
          int incl = n;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += v;
          }
          if (j < nl) l_pass[j] = run + incl - n;
          run += __shfl_sync(kFull, incl, 31);
        }
#pragma unroll
        for (int sft = 16; sft >= 1; sft >>= 1) by += __shfl_xor_sync(kFull, by, sft);
        if (lane == 0) {
          cta_npass = run;
          bytes += by;
        }
      }
    }
    __syncthreads();  // C: pass prefix
    if (warp == 0 && prev_item >= 0) {
      // C4, second half: the previous item's eight queues -> one (the other warps are already scanning)
      // (every parked queue is sorted: a tree of bitonic merges, not 8 K pushes through a selection queue)
      const uint64_t* area = merge + ((round - 1) & 1) * (SCAN_WARPS * K);
      uint64_t* W = a.Wg + prev_item * K;
      if constexpr (M == 8) {
        // M = 8: the keys go through a selection queue instead.  Same result; measured per instantiation on a
        // 10^8-vector M = 8 index, k = 100: scan stage 3.95 / 12.5 ms at nprobe 32 / 128 against 4.10 / 13.3 with
        // the merge tree (the 64-register kernel is allocated differently around it), while M = 16 gains from
        // the tree (1.95 against 2.07 ms at nprobe 16).
        WarpSelect<NQ, NB> ms;
        ms.init(bufs, lane);  // warp 0's own batch area is idle between its items
        for (int e0 = 0; e0 < SCAN_WARPS * K; e0 += 32) {
          const uint64_t key = area[e0 + lane];
          ms.push(key < ms.thr, key);
        }
        ms.finish();
#pragma unroll
        for (int rr = 0; rr < NQ; ++rr) W[rr * 32 + lane] = ms.W[rr];
      } else {
        uint64_t Wm[NQ];
#pragma unroll
        for (int rr = 0; rr < NQ; ++rr) Wm[rr] = area[rr * 32 + lane];
#pragma unroll 1
        for (int w8 = 1; w8 < SCAN_WARPS; ++w8) merge_sorted_queue<NQ>(Wm, area + w8 * K, lane);
#pragma unroll
        for (int rr = 0; rr < NQ; ++rr) W[rr * 32 + lane] = Wm[rr];
      }
      __syncwarp();
    }
    if (!live) break;
    prev_item = item;
    sel.reset();
    sel.set_k(a.k, SCAN_WARPS);
    // C3 + C4.  Warps draw passes of PV = 32 VPL consecutive vectors (VPL per lane: independent look-up
    // chains, and the loop, cursor and selection overhead is paid once for all of them) from a counter, so
    // that the lists of the item are shared evenly whatever their lengths; the list of a pass is found by
    // walking the prefix array forward (passes are handed out in increasing order).
    const int npass = cta_npass;
    const uint32_t pass_sa = (uint32_t)__cvta_generic_to_shared(&cta_pass);
    auto draw = [&]() {
      int t = 0;  // lane 0 draws (predicated, no branch)
      asm volatile("{\n\t.reg .pred p;\n\tsetp.eq.u32 p, %2, 0;\n\t@p atom.shared.add.u32 %0, [%1], 1;\n\t}"
                   : "+r"(t)
                   : "r"(pass_sa), "r"(lane)
                   : "memory");
      return __shfl_sync(kFull, t, 0);
    };
    int lj = 0;                                      // cursor: list of the last pass this warp took
    int nxt_start = nl > 1 ? l_pass[1] : 0x7fffffff;  // first pass of the list after it
    int t = draw();
    while (t < npass) {
      while (t >= nxt_start) {
        ++lj;
        nxt_start = lj + 1 < nl ? l_pass[lj + 1] : 0x7fffffff;
      }
      const int len = l_len[lj];
      const uint32_t pos0 = l_begin[lj];
      const float bias = l_t2[lj];
      const int v = (t - l_pass[lj]) * PV + lane;
      const uint8_t* cv = a.codes + ((size_t)pos0 + (uint32_t)v) * M;
      const float* sv = a.s1 + pos0 + v;
      uint32_t w[VPL][MW];
      float s1v[VPL];
      if (v + PV - 32 < len) {  // full pass
#pragma unroll
        for (int u = 0; u < VPL; ++u) {
          load_code<MW>(cv + u * 32 * M, w[u]);
          s1v[u] = __ldcs(sv + u * 32);
        }
      } else {
#pragma unroll
        for (int u = 0; u < VPL; ++u) {
#pragma unroll
          for (int i = 0; i < MW; ++i) w[u][i] = 0u;
          s1v[u] = 0.f;
          if (v + u * 32 < len) {
            load_code<MW>(cv + u * 32 * M, w[u]);
            s1v[u] = __ldcs(sv + u * 32);
          }
        }
      }
      const int tn = draw();  // the next pass is drawn while the loads are in flight
      uint32_t acc[VPL];
#pragma unroll
      for (int u = 0; u < VPL; ++u) acc[u] = 0u;
      xor_gather_n<0, M, VPL>(w, As, acc);
      const float bound = fminf(sel.thr_val, __uint_as_float(*reinterpret_cast<volatile uint32_t*>(&cta_bound)));
      float dist[VPL];
      bool any = false;
#pragma unroll
      for (int u = 0; u < VPL; ++u) {
        // term 3 = (acc - isum) / scale, an exact integer step for integer-valued data
        dist[u] = fmaf((float)(int32_t)(acc[u] - mt.isum), mt.inv_scale, bias + s1v[u]);
        if (!(v + u * 32 < len)) dist[u] = __uint_as_float(0x7F800000u);  // past the end: never a candidate
        any |= !(dist[u] > bound) && v + u * 32 < len;
      }
      if (__any_sync(kFull, any)) {
        const uint64_t thr_before = sel.thr;
#pragma unroll
        for (int u = 0; u < VPL; ++u) {
          const uint64_t key = make_key(dist[u], pos0 + (uint32_t)(v + u * 32));
          sel.push(v + u * 32 < len && !(dist[u] > bound) && sel.wants(key), key);
        }
        if (sel.thr != thr_before && lane == 0) {
          // two bounds of the item's k-th distance: this warp's own k-th, and the largest of the eight
          // warps' ceil(k / 8)-th distances (their queues cover disjoint passes of the same stream)
          cta_sub[warp] = sel.sub_val;
          float mx = sel.sub_val;
#pragma unroll
          for (int w8 = 0; w8 < SCAN_WARPS; ++w8) mx = fmaxf(mx, *reinterpret_cast<volatile float*>(&cta_sub[w8]));
          atomicMin(&cta_bound, __float_as_uint(fminf(mx, sel.thr_val)));
        }
      }
      t = tn;
    }
    sel.finish();
    // park the queue; the next round's barrier A orders it before warp 0's merge
#pragma unroll
    for (int rr = 0; rr < NQ; ++rr) merge[(round & 1) * (SCAN_WARPS * K) + warp * K + rr * 32 + lane] = sel.W[rr];
    ++round;
  }
  if (tid == 0 && bytes) atomicAdd(a.scanned, bytes);
}

// C1 for a coarse quantizer of modest size and nprobe >= 16: the fused engine's selection runs
// almost entirely on its unbounded first tiles there (profiles/r01_ivfpq.md: 0.95 / 1.2 / 2.7 ms at
// nlist = 8 192, 1.9 / 2.8 / 10.8 ms at 65 536 for nprobe 16 / 64 / 256, against 0.3 / 0.7 ms for
// k = 1).  The paper's own two-step form is cheaper: the tensor-core engine writes the
// distance matrix (no selection), fs_kselect's kernels take nprobe per row.  FS_IVFPQ_C1=fused|matrix
// forces one (A/B runs).
bool c1_matrix(int64_t nq, int64_t nlist, int nprobe, int d) {
  static int forced = -1;
  if (forced < 0) {
    const char* e = getenv("FS_IVFPQ_C1");
    forced = !e ? 0 : strcmp(e, "fused") == 0 ? 1 : strcmp(e, "matrix") == 0 ? 2 : 0;
  }
  if (!flat_tc_supported(d) || nq < 1 || nprobe > nlist || nlist >= ((int64_t)1 << 31)) return false;
  if (forced == 1) return false;
  if (forced == 2) return true;
  if (nprobe < 16 || nq < 256) return false;
  // With a sampled bound (flat_tc.cu: k ns / nb small enough for an ns >= 256) the fused engine wins:
  // C1 stage, nq = 10^4, d = 96, ms fused / matrix: nlist 8 192: nprobe 32 0.58 / 0.73; 16 384: 64 0.68 / 0.97;
  // 32 768: 128 1.01 / 1.49; 65 536: 16 1.34 / 2.85, 256 1.84 / 3.04; 262 144: 2.7 - 3.2 / > 28.
  // Without one (large nprobe over a small quantizer) the two-step form does: 8 192: 256 2.45 / 0.79;
  // 16 384: 128 2.09 / 1.00; 32 768: 256 5.24 / 1.53.
  if (flat_tc_plan(nq, nlist, d, nprobe).ns > 0) return false;
  return nlist <= 16384 || (nprobe >= 128 && nlist <= 131072) || nprobe >= 256;
}

// C1 through the distance matrix: int32 column numbers -> int64 list numbers, values -> the coarse
// distances without ||x||^2 (the scan adds it)
__global__ void widen_ids_kernel(const int32_t* __restrict__ in, const float* __restrict__ val, int64_t* __restrict__ out,
                                 float* __restrict__ cdist, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    out[i] = in[i];
    cdist[i] = val[i];
  }
}

struct SearchPlan {
  int G, ngroups, K;
  bool qscan;  // M = 8 / 16: the per-query table scan
  FlatPlan coarse;
  size_t off_cdist, off_cids, off_W, off_work, off_tq, off_meta, off_bmax, off_D, off_cval, off_cidx, off_ksws, bytes;
  int64_t c1_chunk, c1_ld;  // C1 through a distance matrix: queries per pass (0 = fused engine), row stride
};

SearchPlan search_plan(const fs_ivfpq* ix, int64_t nq, int nprobe, int k) {
  SearchPlan p;
  p.K = 32 << k_class(k);
  p.qscan = ix->permuted();
  // enough CTAs to fill the GPU twice over, but never more groups than probes
  const int64_t target = (int64_t)sm_count() * (p.qscan ? 2 * QS_CTAS : 4);
  int64_t ng = nq > 0 ? ceil_div(target, nq) : 1;
  if (ng > nprobe) ng = nprobe;
  if (ng < 1) ng = 1;
  p.G = (int)ceil_div(nprobe, ng);
  if (p.qscan && p.G > QS_MAXG) p.G = QS_MAXG;
  p.ngroups = (int)ceil_div(nprobe, p.G);
  p.coarse = flat_plan(nq, ix->nlist, ix->d, nprobe);
  size_t o = align_up(p.coarse.bytes, 256);
  p.c1_chunk = 0;
  p.c1_ld = 0;
  if (c1_matrix(nq, ix->nlist, nprobe, ix->d)) {
    p.c1_ld = (ix->nlist + 3) & ~(int64_t)3;
    static int64_t budget = 0;  // bytes of distances per pass: 1 GB; FS_IVFPQ_C1_BYTES overrides (tests)
    if (budget == 0) {
      const char* e = getenv("FS_IVFPQ_C1_BYTES");
      budget = e && atoll(e) > 0 ? atoll(e) : ((int64_t)1 << 30);
    }
    int64_t c = budget / (p.c1_ld * 4);
    if (c < 128) c = 128;
    p.c1_chunk = c < nq ? c : nq;
    // two pass sizes occur (full passes and the last one): the workspaces take the larger plan
    const int64_t last = nq % p.c1_chunk;
    size_t fb = flat_plan(p.c1_chunk, ix->nlist, ix->d, 1).bytes;
    if (last > 0) fb = std::max(fb, flat_plan(last, ix->nlist, ix->d, 1).bytes);
    if (fb > o) o = align_up(fb, 256);
  }
  p.off_cdist = o;
  o += align_up((size_t)nq * nprobe * sizeof(float), 256);
  p.off_cids = o;
  o += align_up((size_t)nq * nprobe * sizeof(int64_t), 256);
  p.off_work = o;
  o += 256;
  p.off_bmax = o;
  o += 256;
  p.off_tq = p.off_meta = o;
  if (p.qscan) {
    o += align_up((size_t)nq * 256 * ix->M * sizeof(uint32_t), 256);
    p.off_meta = o;
    o += align_up((size_t)nq * sizeof(QMeta), 256);
  }
  p.off_D = p.off_cval = p.off_cidx = p.off_ksws = o;
  if (p.c1_chunk > 0) {
    p.off_D = o;
    o += align_up((size_t)p.c1_chunk * p.c1_ld * sizeof(float), 256);
    p.off_cval = o;
    o += align_up((size_t)p.c1_chunk * nprobe * sizeof(float), 256);
    p.off_cidx = o;
    o += align_up((size_t)p.c1_chunk * nprobe * sizeof(int32_t), 256);
    p.off_ksws = o;
    const int64_t last = nq % p.c1_chunk;
    size_t kb = kselect_ws_bytes(p.c1_chunk, ix->nlist, nprobe);
    if (last > 0) kb = std::max(kb, kselect_ws_bytes(last, ix->nlist, nprobe));
    o += align_up(kb, 256);
  }
  p.off_W = o;
  o += align_up((size_t)nq * p.ngroups * p.K * sizeof(uint64_t), 256);
  p.bytes = o;
  return p;
}

template <int NQ>
int launch_scan_pair(const ScanArgs& a, int64_t nq, cudaStream_t s) {
  constexpr int K = 32 * NQ;
  const size_t smem = (size_t)(((a.d + 3) & ~3) + a.M * 256) * sizeof(float) +
                      (size_t)(SCAN_WARPS * warp_select_smem_keys<2>() + SCAN_WARPS * K) * sizeof(uint64_t);
  if (smem > 227 * 1024) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: shared memory (%zu B) exceeds 227 KB", smem);
  FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int64_t grid = nq * a.ngroups;
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: nq * groups too large");
  ivfpq_scan_kernel<NQ><<<(unsigned)grid, SCAN_THREADS, smem, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
}

template <int NQ, int M>
int launch_scan_q(const ScanArgs& a, int64_t nq, const uint32_t* Tq, const QMeta* meta, unsigned int* work,
                  cudaStream_t s) {
  const size_t smem = qs_smem_bytes<NQ>(a.d);
  FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_q_kernel<NQ, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_q_kernel<NQ, M>, cudaFuncAttributePreferredSharedMemoryCarveout,
                               cudaSharedmemCarveoutMaxShared));
  int occ = 0;
  FS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ivfpq_scan_q_kernel<NQ, M>, SCAN_THREADS, smem));
  if (occ < 1) occ = 1;
  const int64_t n_items = nq * a.ngroups;
  int64_t grid = (int64_t)sm_count() * occ;
  if (grid > n_items) grid = n_items;
  FS_CUDA(cudaMemsetAsync(work, 0, sizeof(unsigned int), s));
  ivfpq_scan_q_kernel<NQ, M><<<(unsigned)grid, SCAN_THREADS, smem, s>>>(a, Tq, meta, work, n_items);
  FS_LAUNCHED();
  return FS_OK;
}

}  // namespace

size_t ivfpq_search_ws(const fs_ivfpq* ix, int64_t nq, int nprobe, int k) {
  return search_plan(ix, nq, nprobe, k).bytes;
}

int ivfpq_search_device(fs_ivfpq* ix, const float* xq, int64_t nq, int nprobe, int k,
                        float* out_dist, int64_t* out_ids, int32_t* out_probed, void* ws,
                        cudaStream_t s) {
  const SearchPlan p = search_plan(ix, nq, nprobe, k);
  char* w = static_cast<char*>(ws);
  float* cdist = reinterpret_cast<float*>(w + p.off_cdist);
  int64_t* cids = reinterpret_cast<int64_t*>(w + p.off_cids);
  uint64_t* Wg = reinterpret_cast<uint64_t*>(w + p.off_W);
  int rc;
  ix->ev_valid = false;
  FS_CUDA(cudaEventRecord(ix->ev[0], s));
  // C1 (the centroids are a prepared database: their norms and operand split were made when they were set)
  const FlatPrep cview = flat_prep_view(ix->cprep.p, ix->nlist, ix->d);
  if (p.c1_chunk > 0) {
    float* D = reinterpret_cast<float*>(w + p.off_D);
    float* cval = reinterpret_cast<float*>(w + p.off_cval);
    int32_t* cidx = reinterpret_cast<int32_t*>(w + p.off_cidx);
    for (int64_t q0 = 0; q0 < nq; q0 += p.c1_chunk) {
      const int64_t n = nq - q0 < p.c1_chunk ? nq - q0 : p.c1_chunk;
      rc = flat_knn_tc_device(xq + q0 * ix->d, n, ix->coarse.as<float>(), ix->nlist, ix->d, 1, nullptr, nullptr, w, s,
                              D, p.c1_ld, &cview);
      if (rc != FS_OK) return rc;
      rc = kselect_device(D, n, ix->nlist, p.c1_ld, nprobe, cval, cidx, w + p.off_ksws, s, false);
      if (rc != FS_OK) return rc;
      widen_ids_kernel<<<(unsigned)ceil_div(n * nprobe, 256), 256, 0, s>>>(cidx, cval, cids + q0 * nprobe,
                                                                          cdist + q0 * nprobe, n * nprobe);
      FS_LAUNCHED();
    }
  } else {
    rc = flat_knn_device(xq, nq, ix->coarse.as<float>(), ix->nlist, ix->d, nprobe,
                         ix->cnorm.as<float>(), cdist, cids, w, s, &cview);
    if (rc != FS_OK) return rc;
  }
  FS_CUDA(cudaEventRecord(ix->ev[1], s));
  FS_CUDA(cudaMemsetAsync(ix->scanned.p, 0, sizeof(unsigned long long), s));
  // C2-C4
  ScanArgs a;
  a.xq = xq;
  a.coarse = ix->coarse.as<float>();
  a.pq = ix->pq.as<float>();
  a.probe_ids = cids;
  a.cdist = cdist;
  a.cd_partial = p.c1_chunk > 0;
  a.offsets = ix->offsets.as<int64_t>();
  a.codes = ix->codes.as<uint8_t>();
  a.s1 = ix->s1.as<float>();
  a.Wg = Wg;
  a.scanned = ix->scanned.as<unsigned long long>();
  a.out_probed = out_probed;
  a.d = ix->d;
  a.M = ix->M;
  a.dsub = ix->dsub;
  a.nprobe = nprobe;
  a.G = p.G;
  a.ngroups = p.ngroups;
  a.k = k;
  if (p.qscan) {
    float* bmax = reinterpret_cast<float*>(w + p.off_bmax);
    uint32_t* Tq = reinterpret_cast<uint32_t*>(w + p.off_tq);
    QMeta* meta = reinterpret_cast<QMeta*>(w + p.off_meta);
    unsigned int* work = reinterpret_cast<unsigned int*>(w + p.off_work);
    pq_bmax_kernel<<<ix->M, 32, 0, s>>>(a.pq, bmax, ix->dsub);
    FS_LAUNCHED();
    if (ix->M == 16)
      ivfpq_qtable_kernel<16><<<(unsigned)ceil_div(nq, (int64_t)QT_QPB), 256, 0, s>>>(xq, a.pq, bmax, ix->d, ix->dsub, Tq, meta, nq, QT_QPB);
    else
      ivfpq_qtable_kernel<8><<<(unsigned)ceil_div(nq, (int64_t)QT_QPB), 256, 0, s>>>(xq, a.pq, bmax, ix->d, ix->dsub, Tq, meta, nq, QT_QPB);
    FS_LAUNCHED();
#define FS_QS(NQ)                                                                          \
  (ix->M == 16 ? launch_scan_q<NQ, 16>(a, nq, Tq, meta, work, s) : launch_scan_q<NQ, 8>(a, nq, Tq, meta, work, s))
    switch (k_class(k)) {
      case 0: rc = FS_QS(1); break;
      case 1: rc = FS_QS(2); break;
      case 2: rc = FS_QS(4); break;
      case 3: rc = FS_QS(8); break;
      case 4: rc = FS_QS(16); break;
      default: rc = FS_QS(32); break;
    }
#undef FS_QS
  } else {
    switch (k_class(k)) {
      case 0: rc = launch_scan_pair<1>(a, nq, s); break;
      case 1: rc = launch_scan_pair<2>(a, nq, s); break;
      case 2: rc = launch_scan_pair<4>(a, nq, s); break;
      case 3: rc = launch_scan_pair<8>(a, nq, s); break;
      case 4: rc = launch_scan_pair<16>(a, nq, s); break;
      default: rc = launch_scan_pair<32>(a, nq, s); break;
    }
  }
  if (rc != FS_OK) return rc;
  FS_CUDA(cudaEventRecord(ix->ev[2], s));
  // C5
  FinishExtra fx;
  fx.packed = true;  // the scan parks sorted queues: keys first
  rc = launch_flat_finish(Wg, nq, p.ngroups, k, nullptr, out_dist, out_ids, s, &fx);
  if (rc != FS_OK) return rc;
  if ((rc = launch_resolve_ids(out_dist, out_ids, ix->ids.as<int64_t>(), nq, k, s)) != FS_OK) return rc;
  FS_CUDA(cudaEventRecord(ix->ev[3], s));
  ix->ev_valid = true;
  return FS_OK;
}

}  // namespace fs
