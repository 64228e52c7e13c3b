// ivfpq_search.cu -- fs_ivfpq_search: Alg. 4, SURVEY 8a rows C1-C5.
//
//   C1 coarse quantizer  L_IVF = tau-argmin_c ||x - c||^2 (Eq. 5): the
//                        exact-search engine over the centroids with k = nprobe
//   C2 lookup tables     per (query, probed list): r = x - c_L,
//                        T_m[c] = ||r^m - B[m][c]||^2 (Eq. 10), built in
//                        SHARED memory by the CTA that scans the list (P:L317 has a
//                        separate kernel write them to global memory; here they never
//                        leave the SM)
//   C3 list scan         dist = sum_m T_m[code_m] over the list's codes, streamed
//                        from HBM (Alg. 4)
//   C4 pass-1 selection  fused: every warp k-selects the distances it produces in a
//                        register queue; a CTA covers a GROUP of G probed lists of
//                        one query, so one partial list of k leaves the SM per group
//                        (the paper writes all distances out first, and
//                        found the fused form <= 15 % faster on Maxwell)
//   C5 pass-2 + ids      the groups' partial lists are selected again to k; int64
//                        ids are fetched for the winners only
#include <cstdlib>
#include <cstring>

#include "flat.cuh"
#include "ivfpq.cuh"
#include "ivfpq_scan.cuh"
#include "select.cuh"

namespace fs {

namespace {

constexpr int SCAN_WARPS = 8;
constexpr int SCAN_THREADS = SCAN_WARPS * 32;

// dist += T_m[byte m of the code] for m = m0 .. MT-1.  Tb = shared-space address of T, 1 KB aligned:
// the lookup address is one shift and one LOP3, the table offset m * 1 KB is an immediate.
template <int OFF>
__device__ __forceinline__ float lds_f32_off(uint32_t addr) {
  float t;
  asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(t) : "r"(addr), "n"(OFF));
  return t;
}
template <int m, int MT>
__device__ __forceinline__ void lookup_all(const uint32_t* cw, uint32_t Tb, float& dist) {
  if constexpr (m < MT) {
    const uint32_t w = cw[m >> 2];
    constexpr int j = m & 3;
    const uint32_t sh = j == 0 ? (w << 2) : (w >> (8 * j - 2));
    dist += lds_f32_off<m * 1024>((sh & 0x3FCu) | Tb);
    lookup_all<m + 1, MT>(cw, Tb, dist);
  }
}

// Shared memory: T[M][256] | r[d] | per-warp batches | merge area [SCAN_WARPS][K]
// MT = M when M is 8 or 16 (code loaded with one 8 / 16-byte load, lookups unrolled), else 0;
// DS = d / M when it is 6 or 12 and MT != 0 (table build unrolled, 8 / 16-byte codebook loads), else 0.
template <int NQ, int MT, int DS>
__global__ void __launch_bounds__(SCAN_THREADS) ivfpq_scan_kernel(const ScanArgs a) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  // T first: each table starts on a 1 KB boundary, so a lookup address is (4 * byte) | base
  float* T = reinterpret_cast<float*>(scan_smem);
  float* r = T + a.M * 256;
  uint64_t* bufs = reinterpret_cast<uint64_t*>(r + ((a.d + 3) & ~3));
  uint64_t* merge = bufs + SCAN_WARPS * warp_select_smem_keys<NB>();
  const uint32_t Tb = (uint32_t)__cvta_generic_to_shared(T);
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
    // the first code of every thread is requested before the table is built, and inside the
    // scan every thread holds the code of its next vector: the load latency is off the path
    const uint8_t* cl = a.codes + lb * M;
    constexpr int CW = MT >= 4 ? MT / 4 : 2;
    uint32_t nxt[CW] = {};
    if (MT != 0 && tid < len) load_code<CW>(cl + (size_t)tid * MT, nxt);
    // C2: residual and tables
    for (int j = tid; j < d; j += SCAN_THREADS) r[j] = a.xq[q * d + j] - a.coarse[L * d + j];
    __syncthreads();
    if (MT != 0 && DS != 0) {
      // thread t builds entry c = t of every table m (SCAN_THREADS == 256): unrolled, vector loads
      // a.pq_t: the codebook regrouped as [m][DS / VW][256 codewords][VW] so that the 32 lanes of a
      // warp (32 consecutive codewords) read 32 consecutive 8 / 16-byte pieces: 2 / 4 wavefronts
      // per load instead of the 6 / 12 lines a [m][c][DS] row layout touches
      constexpr int VW = DS == 6 ? 2 : 4;  // floats per load: 8-byte (DS = 6) or 16-byte (DS = 12)
      constexpr int NV = DS / VW;
#pragma unroll 4
      for (int m = 0; m < MT; ++m) {
        const float* rm = r + m * DS;
        float acc = 0.f;
#pragma unroll
        for (int j = 0; j < NV; ++j) {
          float bv[VW], rv[VW];
          if (VW == 2) {
            const float2 t = __ldg(reinterpret_cast<const float2*>(a.pq_t) + (m * NV + j) * 256 + tid);
            const float2 u = reinterpret_cast<const float2*>(rm)[j];
            bv[0] = t.x; bv[1] = t.y; rv[0] = u.x; rv[1] = u.y;
          } else {
            const float4 t = __ldg(reinterpret_cast<const float4*>(a.pq_t) + (m * NV + j) * 256 + tid);
            const float4 u = reinterpret_cast<const float4*>(rm)[j];
            bv[0] = t.x; bv[1] = t.y; bv[VW - 2] = t.z; bv[VW - 1] = t.w;
            rv[0] = u.x; rv[1] = u.y; rv[VW - 2] = u.z; rv[VW - 1] = u.w;
          }
#pragma unroll
          for (int i = 0; i < VW; ++i) {
            const float df = rv[i] - bv[i];
            acc = fmaf(df, df, acc);
          }
        }
        T[m * 256 + tid] = acc;
      }
    } else {
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
    }
    __syncthreads();
    // C3 + C4: scan and select
    bytes += (unsigned long long)len * M;
    // 32-bit indices inside a piece of at most 2^30 vectors (one piece unless a list is enormous)
    for (int64_t c0 = 0; c0 < len; c0 += (int64_t)1 << 30) {
      const int n = (int)((len - c0) < ((int64_t)1 << 30) ? (len - c0) : ((int64_t)1 << 30));
      const uint8_t* cc = cl + c0 * M;
      const uint32_t pos0 = (uint32_t)(lb + c0);
      if (MT != 0 && c0 != 0 && tid < n) load_code<CW>(cc + (size_t)tid * MT, nxt);
      for (int v0 = 0; v0 < n; v0 += SCAN_THREADS) {
        const int v = v0 + tid;
        const bool ok = v < n;
        float dist = 0.f;
        uint32_t cw[CW];
        if (MT != 0) {
#pragma unroll
          for (int i = 0; i < CW; ++i) cw[i] = nxt[i];
          if (v + SCAN_THREADS < n) load_code<CW>(cc + (size_t)(uint32_t)(v + SCAN_THREADS) * MT, nxt);
        }
        if (ok) {
          if (MT == 8 || MT == 16) {
            lookup_all<0, MT>(cw, Tb, dist);
          } else {
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

// C5 second half: positions -> ids; entries with bitwise-equal distance are put
// in ascending id order (positions order them by list and append order, which is
// ascending id only inside a list filled in ascending id order).  One warp per query.
__global__ void __launch_bounds__(128)
    ivfpq_resolve_kernel(float* __restrict__ dist, int64_t* __restrict__ ids_io,
                         const int64_t* __restrict__ ids, int64_t nq, int k) {
  extern __shared__ __align__(16) unsigned char res_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t q = (int64_t)blockIdx.x * 4 + warp;
  if (q >= nq) return;
  int64_t* sid = reinterpret_cast<int64_t*>(res_smem) + (size_t)warp * k;
  float* sd = reinterpret_cast<float*>(reinterpret_cast<int64_t*>(res_smem) + (size_t)4 * k) +
              (size_t)warp * k;
  for (int i = lane; i < k; i += 32) {
    const int64_t pos = ids_io[q * k + i];
    sid[i] = pos < 0 ? -1 : ids[pos];
    sd[i] = dist[q * k + i];
  }
  __syncwarp();
  for (int i = lane; i < k; i += 32) {
    const float di = sd[i];
    const int64_t id = sid[i];
    int rank = i;
    if (id >= 0) {
      int s = i, e = i;
      while (s > 0 && sd[s - 1] == di && sid[s - 1] >= 0) --s;
      while (e + 1 < k && sd[e + 1] == di && sid[e + 1] >= 0) ++e;
      if (e > s) {
        rank = s;
        for (int j = s; j <= e; ++j) rank += (sid[j] < id) || (sid[j] == id && j < i);
      }
    }
    ids_io[q * k + rank] = id;
  }
}

// The codebook regrouped for the vectorised table build: pq [M][256][dsub] ->
// pq_t [M][dsub / vw][256][vw] (a few hundred KB at most; redone per search, it is ~2 us).
__global__ void pq_regroup_kernel(const float* __restrict__ pq, float* __restrict__ pq_t, int M, int dsub,
                                  int vw) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M * 256 * dsub) return;
  const int m = i / (256 * dsub);
  const int rem = i - m * 256 * dsub;
  const int c = rem / dsub, j = rem - c * dsub;
  pq_t[((m * (dsub / vw) + j / vw) * 256 + c) * vw + (j % vw)] = pq[i];
}

struct SearchPlan {
  int G, ngroups, K;
  FlatPlan coarse;
  size_t off_cdist, off_cids, off_W, off_work, off_pqt, bytes;
};

SearchPlan search_plan(const fs_ivfpq* ix, int64_t nq, int nprobe, int k) {
  SearchPlan p;
  p.K = 32 << k_class(k);
  // enough CTAs to fill the GPU twice over, but never more groups than probes
  const int64_t target = (int64_t)sm_count() * 4;
  int64_t ng = nq > 0 ? ceil_div(target, nq) : 1;
  if (ng > nprobe) ng = nprobe;
  if (ng < 1) ng = 1;
  p.G = (int)ceil_div(nprobe, ng);
  p.ngroups = (int)ceil_div(nprobe, p.G);
  p.coarse = flat_plan(nq, ix->nlist, ix->d, nprobe);
  size_t o = align_up(p.coarse.bytes, 256);
  p.off_cdist = o;
  o += align_up((size_t)nq * nprobe * sizeof(float), 256);
  p.off_cids = o;
  o += align_up((size_t)nq * nprobe * sizeof(int64_t), 256);
  p.off_work = o;
  o += 256;
  p.off_pqt = o;
  o += align_up((size_t)256 * ix->d * sizeof(float), 256);
  p.off_W = o;
  const int qpi = scan2_supported(ix->d, ix->M, k) ? scan2_queues_per_item() : 1;
  o += align_up((size_t)nq * p.ngroups * qpi * p.K * sizeof(uint64_t), 256);
  p.bytes = o;
  return p;
}

// ---------------------------------------------------------------------------
// M = 8 or 16: the same scan with a bank-conflict-free gather.
//   * the table is stored as lut[c][b], b = 0..31: word (c, b) lives in shared-memory bank b and
//     holds T_{b mod M}[c] (32 / M replicas of every table); lane l adds its sub-quantizers in
//     the rotated order m = (s + l) mod M, so at step s the 32 lanes read 32 different banks;
//     lane l rotates its code by l mod M bytes once per vector (funnel shifts);
//   * so that the rotated order cannot change the sum, the entries are FIXED-POINT: the CTA
//     scales every table of the (query, list) pair by one power of two such that the largest
//     entry is < 2^27, rounds to integers, and the scan adds integers (exact, associative).
//     Identical codes therefore give identical distances whatever lane scans them (reading
//     C-6).  Quantisation: <= 2^-28 of the largest table entry per entry, M times that per
//     distance -- far inside the 1e-3 relative tolerance for every distance that is not
//     ~5 orders of magnitude below the largest entry of its tables.
// Shared memory: r[d] | Tn[M][257] | lut[256][32] | red[8] | select batches | merge area
// ---------------------------------------------------------------------------
template <int NQ, int M>
__global__ void __launch_bounds__(SCAN_THREADS) ivfpq_scan_rot_kernel(const ScanArgs a) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int TS = 257;  // row stride of the natural table: conflict-free reads by m
  const int d = a.d, dsub = a.dsub;
  float* r = reinterpret_cast<float*>(scan_smem);
  float* Tn = r + ((d + 3) & ~3);
  uint32_t* lut = reinterpret_cast<uint32_t*>(Tn + ((M * TS + 3) & ~3));
  float* red = reinterpret_cast<float*>(lut + 256 * 32);
  uint64_t* bufs = reinterpret_cast<uint64_t*>(red + 8);
  uint64_t* merge = bufs + SCAN_WARPS * warp_select_smem_keys<NB>();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t q = blockIdx.x / a.ngroups;
  const int g = (int)(blockIdx.x - q * a.ngroups);
  const int p_begin = g * a.G;
  const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;

  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  unsigned long long bytes = 0;
  const int rot = lane % M;

  for (int p = p_begin; p < p_end; ++p) {
    const int64_t L = a.probe_ids[q * a.nprobe + p];
    if (a.out_probed && tid == 0) a.out_probed[q * a.nprobe + p] = (int32_t)L;
    if (L < 0) continue;
    const int64_t lb = a.offsets[L], le = a.offsets[L + 1];
    const int64_t len = le - lb;
    if (len == 0) continue;  // empty lists are probed and contribute nothing
    __syncthreads();         // previous list's tables are no longer read
    for (int j = tid; j < d; j += SCAN_THREADS) r[j] = a.xq[q * d + j] - a.coarse[L * d + j];
    __syncthreads();
    // C2, step 1: T_m[c] = ||r^m - B[m][c]||^2 (Eq. 10) in the natural layout, and its maximum
    float mx = 0.f;
    for (int e = tid; e < M * 256; e += SCAN_THREADS) {
      const int m = e >> 8;
      const float* b = a.pq + (int64_t)e * dsub;
      const float* rm = r + m * dsub;
      float acc = 0.f;
      if (dsub == 6) {
        const float2* b2 = reinterpret_cast<const float2*>(b);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const float2 bb = __ldg(b2 + j);
          const float t0 = rm[2 * j] - bb.x, t1 = rm[2 * j + 1] - bb.y;
          acc = fmaf(t0, t0, acc);
          acc = fmaf(t1, t1, acc);
        }
      } else if (dsub == 12) {
        const float4* b4 = reinterpret_cast<const float4*>(b);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const float4 bb = __ldg(b4 + j);
          const float t0 = rm[4 * j] - bb.x, t1 = rm[4 * j + 1] - bb.y, t2 = rm[4 * j + 2] - bb.z,
                      t3 = rm[4 * j + 3] - bb.w;
          acc = fmaf(t0, t0, acc);
          acc = fmaf(t1, t1, acc);
          acc = fmaf(t2, t2, acc);
          acc = fmaf(t3, t3, acc);
        }
      } else {
        for (int j = 0; j < dsub; ++j) {
          const float t = rm[j] - b[j];
          acc = fmaf(t, t, acc);
        }
      }
      Tn[m * TS + (e & 255)] = acc;
      mx = fmaxf(mx, acc);
    }
#pragma unroll
    for (int sft = 16; sft >= 1; sft >>= 1) mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, sft));
    if (lane == 0) red[warp] = mx;
    __syncthreads();
    // C2, step 2: one power-of-two scale for the pair, integer entries into the banked layout
    mx = red[0];
#pragma unroll
    for (int w = 1; w < SCAN_WARPS; ++w) mx = fmaxf(mx, red[w]);
    int ex = 0;
    if (mx > 0.f && mx < 3.0e38f) frexpf(mx, &ex);  // mx < 2^ex
    int se = 27 - ex;                               // scale = 2^se: scaled entries < 2^27
    se = se > 100 ? 100 : (se < -100 ? -100 : se);
    const float scale = __uint_as_float((uint32_t)(127 + se) << 23);
    const float inv_scale = __uint_as_float((uint32_t)(127 - se) << 23);
    {
      const int m = lane % M, cofs = lane / M;
      for (int c0 = warp * REP; c0 < 256; c0 += SCAN_WARPS * REP) {
        const int c = c0 + cofs;
        const uint32_t v = __float2uint_rn(Tn[m * TS + c] * scale);
#pragma unroll
        for (int rep = 0; rep < REP; ++rep) lut[c * 32 + m + rep * M] = v;
      }
    }
    __syncthreads();
    // C3 + C4: scan and select
    bytes += (unsigned long long)len * M;
    const uint8_t* cl = a.codes + lb * M;
    const char* lutb = reinterpret_cast<const char*>(lut);
    for (int64_t v0 = 0; v0 < len; v0 += SCAN_THREADS) {
      const int64_t v = v0 + tid;
      const bool ok = v < len;
      float dist = 0.f;
      if (ok) {
        uint32_t w[MW];
        load_code<MW>(cl + v * M, w);
        rotate_bytes<MW>(w, rot);
        uint32_t acc = 0u;
#pragma unroll
        for (int s2 = 0; s2 < M; ++s2) {
          const uint32_t c = (w[s2 >> 2] >> (8 * (s2 & 3))) & 255u;
          acc += *reinterpret_cast<const uint32_t*>(lutb + c * 128 + (((s2 + lane) & 31) << 2));
        }
        dist = (float)acc * inv_scale;
      }
      const bool cand = ok && sel.maybe(dist);
      if (__any_sync(kFull, cand)) {
        const uint64_t key = make_key(dist, (uint32_t)(lb + v));
        sel.push(cand && sel.wants(key), key);
      }
    }
  }
  sel.finish();
  if (tid == 0 && bytes) atomicAdd(a.scanned, bytes);

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

template <int NQ, int M>
int launch_scan_rot(const ScanArgs& a, int64_t nq, cudaStream_t s) {
  constexpr int K = 32 * NQ;
  const size_t smem = (size_t)(((a.d + 3) & ~3) + ((M * 257 + 3) & ~3) + 256 * 32 + 8) * sizeof(float) +
                      (size_t)(SCAN_WARPS * warp_select_smem_keys<2>() + SCAN_WARPS * K) * sizeof(uint64_t);
  if (smem > 227 * 1024) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: shared memory (%zu B) exceeds 227 KB", smem);
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_rot_kernel<NQ, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const char* e = getenv("FS_IVFPQ_CARVEOUT");
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_rot_kernel<NQ, M>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 e ? atoi(e) : 100));
    attr_smem = smem;
  }
  const int64_t grid = nq * a.ngroups;
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: nq * groups too large");
  ivfpq_scan_rot_kernel<NQ, M><<<(unsigned)grid, SCAN_THREADS, smem, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
}

template <int NQ, int MT, int DS>
int launch_scan_m(const ScanArgs& a, int64_t nq, cudaStream_t s) {
  constexpr int K = 32 * NQ;
  const size_t smem = (size_t)(((a.d + 3) & ~3) + a.M * 256) * sizeof(float) +
                      (size_t)(SCAN_WARPS * warp_select_smem_keys<2>() + SCAN_WARPS * K) * sizeof(uint64_t);
  if (smem > 227 * 1024) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: shared memory (%zu B) exceeds 227 KB", smem);
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_kernel<NQ, MT, DS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // Leave part of the unified L1 / shared memory to L1: every CTA re-reads the PQ codebook
    // (256 d floats, 96 KB at d = 96) for every table it builds; with the maximum shared-memory
    // carve-out those reads all go to L2.
    const char* e = getenv("FS_IVFPQ_CARVEOUT");
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_kernel<NQ, MT, DS>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 e ? atoi(e) : 65));
    attr_smem = smem;
  }
  const int64_t grid = nq * a.ngroups;
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: nq * groups too large");
  ivfpq_scan_kernel<NQ, MT, DS><<<(unsigned)grid, SCAN_THREADS, smem, s>>>(a);
  FS_LAUNCHED();
  return FS_OK;
}

template <int NQ>
int launch_scan(const ScanArgs& a, int64_t nq, cudaStream_t s) {
  // FS_IVFPQ_SCAN=rot selects the bank-conflict-free fixed-point kernel (A/B runs): correct, but
  // its second table pass and larger footprint cost more than the conflicts (profiles/r01_ivfpq.md)
  static int plain = -1;
  if (plain < 0) {
    const char* e = getenv("FS_IVFPQ_SCAN");
    plain = (e && strcmp(e, "rot") == 0) ? 0 : 1;
  }
  if (!plain && NQ <= 8 && a.M == 16) return launch_scan_rot<NQ, 16>(a, nq, s);
  if (!plain && NQ <= 8 && a.M == 8) return launch_scan_rot<NQ, 8>(a, nq, s);
  if (a.M == 16 && a.dsub == 6) return launch_scan_m<NQ, 16, 6>(a, nq, s);
  if (a.M == 8 && a.dsub == 12) return launch_scan_m<NQ, 8, 12>(a, nq, s);
  if (a.M == 16) return launch_scan_m<NQ, 16, 0>(a, nq, s);
  if (a.M == 8) return launch_scan_m<NQ, 8, 0>(a, nq, s);
  return launch_scan_m<NQ, 0, 0>(a, nq, s);
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
  // C1
  rc = flat_knn_device(xq, nq, ix->coarse.as<float>(), ix->nlist, ix->d, nprobe,
                       ix->cnorm.as<float>(), cdist, cids, w, s);
  if (rc != FS_OK) return rc;
  FS_CUDA(cudaMemsetAsync(ix->scanned.p, 0, sizeof(unsigned long long), s));
  // C2-C4
  ScanArgs a;
  a.xq = xq;
  a.coarse = ix->coarse.as<float>();
  a.pq = ix->pq.as<float>();
  a.pq_t = nullptr;
  if ((ix->M == 16 && ix->dsub == 6) || (ix->M == 8 && ix->dsub == 12)) {
    float* pq_t = reinterpret_cast<float*>(w + p.off_pqt);
    const int n = 256 * ix->d;
    pq_regroup_kernel<<<ceil_div(n, 256), 256, 0, s>>>(a.pq, pq_t, ix->M, ix->dsub, ix->dsub == 6 ? 2 : 4);
    FS_LAUNCHED();
    a.pq_t = pq_t;
  }
  a.probe_ids = cids;
  a.offsets = ix->offsets.as<int64_t>();
  a.codes = ix->codes.as<uint8_t>();
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
  const bool persistent = ix->ntotal() < ((int64_t)1 << 31) && scan2_supported(ix->d, ix->M, k);  // 32-bit list lengths
  const int qpi = persistent ? scan2_queues_per_item() : 1;
  if (persistent)
    rc = launch_scan2(a, nq, k, reinterpret_cast<unsigned int*>(w + p.off_work), s);
  else
  switch (k_class(k)) {
    case 0: rc = launch_scan<1>(a, nq, s); break;
    case 1: rc = launch_scan<2>(a, nq, s); break;
    case 2: rc = launch_scan<4>(a, nq, s); break;
    case 3: rc = launch_scan<8>(a, nq, s); break;
    case 4: rc = launch_scan<16>(a, nq, s); break;
    default: rc = launch_scan<32>(a, nq, s); break;
  }
  if (rc != FS_OK) return rc;
  // C5
  rc = launch_flat_finish(Wg, nq, p.ngroups * qpi, k, nullptr, out_dist, out_ids, s);
  if (rc != FS_OK) return rc;
  const size_t smem = (size_t)4 * k * (sizeof(int64_t) + sizeof(float));
  ivfpq_resolve_kernel<<<(unsigned)ceil_div(nq, 4), 128, smem, s>>>(out_dist, out_ids,
                                                                    ix->ids.as<int64_t>(), nq, k);
  FS_LAUNCHED();
  return FS_OK;
}

}  // namespace fs
