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
                   int32_t* out_idx, void* ws, cudaStream_t s);

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
// DS = d / M when it is 6, 8, 12 or 16 and MT != 0 (table build unrolled, 8 / 16-byte codebook loads), else 0.
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

// The codebook regrouped for the vectorised table builds (a few hundred KB at most; redone per
// search, it is ~2 us):
//   pq_t [M][dsub / vw][256][vw]            thread c builds entry c of every table (float kernel)
//   pq_r [256 / REP][dsub / vw][32][vw]     lane l = cofs * M + m builds entry (m, c0 + cofs) (rot kernel)
//   bmax [M]                                max_c ||B[m][c]|| (bound of the fixed-point scale)
__global__ void pq_regroup_kernel(const float* __restrict__ pq, float* __restrict__ pq_t, float* __restrict__ pq_r,
                                  int M, int dsub, int vw) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M * 256 * dsub) return;
  const int m = i / (256 * dsub);
  const int rem = i - m * 256 * dsub;
  const int c = rem / dsub, j = rem - c * dsub;
  const int nv = dsub / vw, rep = 32 / M;
  pq_t[((m * nv + j / vw) * 256 + c) * vw + (j % vw)] = pq[i];
  pq_r[(((c / rep) * nv + j / vw) * 32 + (c % rep) * M + m) * vw + (j % vw)] = pq[i];
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
  // measured (nq = 10^4, d = 96; search of a tiny index, ms, fused / matrix): nlist 8 192: nprobe 64
  // 2.79 / 1.95, 256 8.25 / 6.30; nlist 65 536: 16 1.71 / 2.41, 64 2.85 / 2.97, 256 9.24 / 4.93;
  // nlist 262 144: 64 4.98 / 11.1, 256 14.4 / 13.6
  return nlist <= 16384 || (nprobe >= 128 && nlist <= 131072) || nprobe >= 256;
}

int scan_forced_mode() {  // 0 none, 1 rot, 2 grp, 3 pair, 4 pre
  static int forced = -1;
  if (forced < 0) {
    const char* e = getenv("FS_IVFPQ_SCAN");
    forced = !e ? 0 : strcmp(e, "pair") == 0 ? 3 : strcmp(e, "rot") == 0 ? 1 : strcmp(e, "grp") == 0 ? 2 : strcmp(e, "pre") == 0 ? 4 : 0;
  }
  return forced;
}
bool scan_forced_pre() { return scan_forced_mode() == 4; }
// (M = 8: half the lookups per vector, the float kernel stays ahead: 7.7 against 9.7 ms, cfg5 shape)
bool scan_auto_grouped(int M, int G, int64_t n_items) {
  return scan_forced_mode() == 0 && M == 16 && G >= 32 && n_items >= (int64_t)9 * sm_count();  // 3 rounds of 3 groups per SM
}

// The decomposed table build (FS_IVFPQ_SCAN=pre) needs M = 8 / 16 and nlist * M * 1 KB of device memory
// (<= 4 GB here).  Measured level with the direct build once both scans use the XOR order (9.26 against
// 8.89 ms at nprobe 64): kept as a forced variant, not the default.
bool want_term1(const fs_ivfpq* ix) {
  return scan_forced_pre() && (ix->M == 16 || ix->M == 8) && ix->d <= SCAN_THREADS &&
         (size_t)ix->nlist * ix->M * 256 * sizeof(float) <= ((size_t)4 << 30);
}

__global__ void widen_ids_kernel(const int32_t* __restrict__ in, int64_t* __restrict__ out, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = in[i];
}

struct SearchPlan {
  int G, ngroups, K;
  FlatPlan coarse;
  size_t off_cdist, off_cids, off_W, off_work, off_pqt, off_pqr, off_D, off_cval, off_cidx, off_ksws, bytes;
  int64_t c1_chunk, c1_ld;  // C1 through a distance matrix: queries per pass (0 = fused engine), row stride
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
  p.off_pqt = o;
  o += align_up((size_t)256 * ix->d * sizeof(float), 256);
  p.off_pqr = o;
  o += align_up((size_t)256 * ix->d * sizeof(float), 256) + 256;  // + bmax[M]
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
  const int qpi = scan2_supported(ix->d, ix->M, k) ? scan2_queues_per_item() : 1;
  o += align_up((size_t)nq * p.ngroups * qpi * p.K * sizeof(uint64_t), 256);
  p.bytes = o;
  return p;
}

// ---------------------------------------------------------------------------
// M = 8 or 16, dsub = 6 or 12: the same scan with a bank-conflict-free gather (FS_IVFPQ_SCAN=rot).
//   * the table is stored as lut[c][b], b = 0..31: word (c, b) lives in shared-memory bank b and
//     holds T_{b mod M}[c] (32 / M replicas of every table); lane l adds its sub-quantizers in
//     the rotated order m = (s + l) mod M, so at step s the 32 lanes read 32 different banks;
//     lane l rotates its code by l mod M bytes once per vector (funnel shifts);
//   * so that the rotated order cannot change the sum, the entries are FIXED-POINT: one power-of-two
//     scale per (query, list) pair, from the bound (||r^m|| + max_c ||B[m][c]||)^2 >= every entry of
//     T_m, makes every entry an integer < 2^27; the scan adds integers (exact, associative), so
//     identical codes give identical distances whatever lane scans them (reading C-6).
//     Quantisation: <= 2^-27 of the bound per entry, M times that per distance;
//   * build: lane l of a warp computes entry (m = l mod M, c = c0 + l / M) from a codebook that
//     pq_regroup_kernel lays out so that the warp's loads are 32 consecutive 8 / 16-byte pieces,
//     and stores its 32 / M replicas in rotated replica order: loads coalesced, stores conflict-free.
// Shared memory: lut[256][32] | r[d] | select batches | merge area
// ---------------------------------------------------------------------------
template <int s, int M>
__device__ __forceinline__ void rot_gather(const uint32_t* w, const uint32_t* base, uint32_t& acc) {
  if constexpr (s < M) {
    const uint32_t c = __byte_perm(w[s >> 2], 0u, 0x4440u + (s & 3));  // byte s, zero-extended
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(base[s] + c * 128u));
    acc += v;
    rot_gather<s + 1, M>(w, base, acc);
  }
}

// acc += lut[byte s of w][bank lane ^ s] for s = s0 .. M-1; A = table + 4 * lane (table 128-byte aligned)
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

template <int NQ, int M, int DS>
__global__ void __launch_bounds__(SCAN_THREADS, 3) ivfpq_scan_rot_kernel(const ScanArgs a) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int VW = DS == 6 ? 2 : 4;
  constexpr int NV = DS / VW;
  const int d = a.d;
  uint32_t* lut = reinterpret_cast<uint32_t*>(scan_smem);
  float* r = reinterpret_cast<float*>(lut + 256 * 32);
  uint64_t* bufs = reinterpret_cast<uint64_t*>(r + ((d + 3) & ~3));
  uint64_t* merge = bufs + SCAN_WARPS * warp_select_smem_keys<NB>();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t q = blockIdx.x / a.ngroups;
  const int g = (int)(blockIdx.x - q * a.ngroups);
  const int p_begin = g * a.G;
  const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;

  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  unsigned long long bytes = 0;
  __shared__ uint32_t cta_bound;
  if (tid == 0) cta_bound = 0x7F800000u;
  const int rot = lane % M;
  const int my_m = lane % M, cofs = lane / M;
  const float my_bmax = a.bmax[my_m];
  const uint32_t lutb = (uint32_t)__cvta_generic_to_shared(lut);
  uint32_t base[M];
#pragma unroll
  for (int s = 0; s < M; ++s) base[s] = lutb + (((lane + s) & 31) << 2);

  for (int p = p_begin; p < p_end; ++p) {
    const int64_t L = a.probe_ids[q * a.nprobe + p];
    if (a.out_probed && tid == 0) a.out_probed[q * a.nprobe + p] = (int32_t)L;
    if (L < 0) continue;
    const int64_t lb = a.offsets[L], le = a.offsets[L + 1];
    const int64_t len64 = le - lb;
    if (len64 == 0) continue;  // empty lists are probed and contribute nothing
    const int len = (int)len64;  // the caller routes indexes of 2^31 vectors or more to the float kernel
    __syncthreads();             // previous list's table is no longer read
    const uint8_t* cl = a.codes + lb * M;
    uint32_t nxt[MW] = {};
    if (tid < len) load_code<MW>(cl + (size_t)tid * M, nxt);
    for (int j = tid; j < d; j += SCAN_THREADS) r[j] = a.xq[q * d + j] - a.coarse[L * d + j];
    __syncthreads();
    // C2: scale from the bound, then the fixed-point table (Eq. 10)
    float rm[DS];
    float n = 0.f;
#pragma unroll
    for (int j = 0; j < DS; ++j) {
      rm[j] = r[my_m * DS + j];
      n = fmaf(rm[j], rm[j], n);
    }
    float u = sqrtf(n) + my_bmax;
    u = u * u * 1.001f;  // >= every entry of T_m as the float code below computes it
#pragma unroll
    for (int sft = 16; sft >= 1; sft >>= 1) u = fmaxf(u, __shfl_xor_sync(kFull, u, sft));
    int ex = 0;
    if (u > 0.f && u < 3.0e38f) frexpf(u, &ex);  // u < 2^ex
    int se = 27 - ex;                            // scaled entries < 2^27
    se = se > 100 ? 100 : (se < -100 ? -100 : se);
    const float scale = __uint_as_float((uint32_t)(127 + se) << 23);
    const float inv_scale = __uint_as_float((uint32_t)(127 - se) << 23);
#pragma unroll 2
    for (int c0 = warp * REP; c0 < 256; c0 += SCAN_WARPS * REP) {
      const int c = c0 + cofs;
      float t = 0.f;
#pragma unroll
      for (int jv = 0; jv < NV; ++jv) {
        float bv[VW];
        if (VW == 2) {
          const float2 x = __ldg(reinterpret_cast<const float2*>(a.pq_r) + ((c0 / REP) * NV + jv) * 32 + lane);
          bv[0] = x.x; bv[1] = x.y;
        } else {
          const float4 x = __ldg(reinterpret_cast<const float4*>(a.pq_r) + ((c0 / REP) * NV + jv) * 32 + lane);
          bv[0] = x.x; bv[1] = x.y; bv[VW - 2] = x.z; bv[VW - 1] = x.w;
        }
#pragma unroll
        for (int i = 0; i < VW; ++i) {
          const float df = rm[jv * VW + i] - bv[i];
          t = fmaf(df, df, t);
        }
      }
      const uint32_t v = __float2uint_rn(t * scale);
      // replica (rep + cofs) mod REP at store rep: the 32 lanes write 32 different banks
#pragma unroll
      for (int rep = 0; rep < REP; ++rep) lut[c * 32 + my_m + ((rep + cofs) % REP) * M] = v;
    }
    __syncthreads();
    // C3 + C4: scan and select
    bytes += (unsigned long long)len * M;
    const uint32_t pos0 = (uint32_t)lb;
    for (int v0 = warp * 32; v0 < len; v0 += SCAN_THREADS) {  // a warp stops after its last 32 vectors
      const int v = v0 + lane;
      const bool ok = v < len;
      uint32_t w[MW];
#pragma unroll
      for (int i = 0; i < MW; ++i) w[i] = nxt[i];
      if (v + SCAN_THREADS < len) load_code<MW>(cl + (size_t)(uint32_t)(v + SCAN_THREADS) * M, nxt);
      float dist = 0.f;
      if (ok) {
        rotate_bytes<MW>(w, rot);
        uint32_t acc = 0u;
        rot_gather<0, M>(w, base, acc);
        dist = (float)acc * inv_scale;
      }
      const float bound = fminf(sel.thr_val, __uint_as_float(*reinterpret_cast<volatile uint32_t*>(&cta_bound)));
      const bool cand = ok && !(dist > bound);
      if (__any_sync(kFull, cand)) {
        const uint64_t key = make_key(dist, pos0 + (uint32_t)v);
        const uint64_t thr_before = sel.thr;
        sel.push(cand && sel.wants(key), key);
        if (sel.thr != thr_before && lane == 0) atomicMin(&cta_bound, __float_as_uint(sel.thr_val));
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

// ---------------------------------------------------------------------------
// The same fixed-point scan, persistent (FS_IVFPQ_SCAN=grp): one CTA of GRP_N groups of 8 warps per
// SM.  The regrouped codebook (pq_r, 256 d floats) is resident in shared memory, shared by the
// groups; every group owns one table and walks its own (query, list group) items, handed out by
// an atomic counter, synchronising with a named barrier: the groups overlap each other's table
// builds and scans like independent CTAs would, but no table build reads global memory.
// Shared memory: cb[256 d] | per group: lut[256][32] (merge area aliases it) | r[d] | select batches
// ---------------------------------------------------------------------------
constexpr int GRP_N = 3;
constexpr int GRP_THREADS = SCAN_THREADS * GRP_N;

__device__ __forceinline__ void group_sync(int gid) {
  asm volatile("bar.sync %0, %1;" ::"r"(gid + 1), "n"(SCAN_THREADS) : "memory");
}

template <int NQ, int M, int DS>
__global__ void __launch_bounds__(GRP_THREADS, 1) ivfpq_scan_grp_kernel(const ScanArgs a, unsigned int* __restrict__ work,
                                                                         int64_t n_items) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int VW = DS == 6 ? 2 : 4;
  constexpr int NV = DS / VW;
  static_assert(SCAN_WARPS * K * 8 <= 256 * 32 * 4, "merge area must fit the table it aliases");
  const int d = a.d, dpad = (d + 3) & ~3;
  const int gid = threadIdx.x / SCAN_THREADS, tid = threadIdx.x % SCAN_THREADS, lane = tid & 31, warp = tid >> 5;
  float* cb = reinterpret_cast<float*>(scan_smem);  // pq_r, as laid out by pq_regroup_kernel
  const size_t grp_bytes = (size_t)256 * 32 * 4 + (size_t)dpad * 4 + (size_t)SCAN_WARPS * warp_select_smem_keys<NB>() * 8;
  unsigned char* gbase = scan_smem + (size_t)256 * d * 4 + gid * grp_bytes;
  uint32_t* lut = reinterpret_cast<uint32_t*>(gbase);
  float* r = reinterpret_cast<float*>(lut + 256 * 32);
  uint64_t* bufs = reinterpret_cast<uint64_t*>(r + dpad);
  uint64_t* merge = reinterpret_cast<uint64_t*>(lut);  // the table is dead when the queues are merged
  __shared__ uint32_t grp_bound[GRP_N];
  __shared__ int grp_item[GRP_N];

  for (int i = threadIdx.x; i < 256 * d / 4; i += GRP_THREADS)
    reinterpret_cast<float4*>(cb)[i] = __ldg(reinterpret_cast<const float4*>(a.pq_r) + i);
  __syncthreads();

  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  unsigned long long bytes = 0;
  const int rot = lane % M;
  const int my_m = lane % M, cofs = lane / M;
  const float my_bmax = a.bmax[my_m];
  const uint32_t lutb = (uint32_t)__cvta_generic_to_shared(lut);
  const uint32_t lane_base = lutb + ((uint32_t)lane << 2);  // step s reads bank lane ^ s

  while (true) {
    group_sync(gid);  // the previous item's merge is done with the table / merge area
    if (tid == 0) {
      grp_item[gid] = (int)atomicAdd(work, 1u);
      grp_bound[gid] = 0x7F800000u;
    }
    group_sync(gid);
    const int64_t item = grp_item[gid];
    if (item >= n_items) break;
    const int64_t q = item / a.ngroups;
    const int g = (int)(item - q * a.ngroups);
    const int p_begin = g * a.G;
    const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;
    sel.reset();

    // The dependent loads of a list (probe id -> list bounds, centroid) are issued one and two
    // lists ahead and stay in registers: none of their latency is on the path.
    const float xj = tid < d ? a.xq[q * d + tid] : 0.f;
    const int64_t* pid = a.probe_ids + q * a.nprobe;
    int64_t L1 = pid[p_begin];                                // list of the coming iteration
    int64_t L2 = p_begin + 1 < p_end ? pid[p_begin + 1] : -1;  // and of the one after
    int64_t lb1 = 0, le1 = 0;
    float c1 = 0.f;
    if (L1 >= 0) {
      lb1 = a.offsets[L1];
      le1 = a.offsets[L1 + 1];
      if (tid < d) c1 = a.coarse[L1 * d + tid];
    }
    for (int p = p_begin; p < p_end; ++p) {
      const int64_t L = L1, lb = lb1, le = le1;
      const float cj = c1;
      L1 = L2;
      if (L1 >= 0) {
        lb1 = a.offsets[L1];
        le1 = a.offsets[L1 + 1];
        if (tid < d) c1 = a.coarse[L1 * d + tid];
      }
      L2 = p + 2 < p_end ? pid[p + 2] : -1;
      if (a.out_probed && tid == 0) a.out_probed[q * a.nprobe + p] = (int32_t)L;
      if (L < 0 || le == lb) continue;  // empty lists are probed and contribute nothing
      const int len = (int)(le - lb);
      group_sync(gid);  // previous list's table is no longer read
      const uint8_t* cl = a.codes + lb * M;
      uint32_t nxt[MW] = {};
      if (tid < len) load_code<MW>(cl + (size_t)tid * M, nxt);
      if (tid < d) r[tid] = xj - cj;
      group_sync(gid);
      // C2: scale from the bound, then the fixed-point table (Eq. 10)
      float rm[DS];
      float n = 0.f;
#pragma unroll
      for (int j = 0; j < DS; ++j) {
        rm[j] = r[my_m * DS + j];
        n = fmaf(rm[j], rm[j], n);
      }
      uint64_t rm2[DS / 2];  // the residual sub-vector as packed pairs (FADD2 / FFMA2 below)
#pragma unroll
      for (int j = 0; j < DS / 2; ++j) rm2[j] = f2_pack(rm[2 * j], rm[2 * j + 1]);
      float u = sqrtf(n) + my_bmax;
      u = u * u * 1.001f;  // >= every entry of T_m as the float code below computes it
#pragma unroll
      for (int sft = 16; sft >= 1; sft >>= 1) u = fmaxf(u, __shfl_xor_sync(kFull, u, sft));
      int ex = 0;
      if (u > 0.f && u < 3.0e38f) frexpf(u, &ex);  // u < 2^ex
      int se = 27 - ex;                            // scaled entries < 2^27
      se = se > 100 ? 100 : (se < -100 ? -100 : se);
      const float scale = __uint_as_float((uint32_t)(127 + se) << 23);
      const float inv_scale = __uint_as_float((uint32_t)(127 - se) << 23);
#pragma unroll 4
      for (int c0 = warp * REP; c0 < 256; c0 += SCAN_WARPS * REP) {
        const int c = c0 + cofs;
        // even and odd dimensions accumulate in the two halves of one packed register
        uint64_t acc2 = 0ull;
#pragma unroll
        for (int jv = 0; jv < NV; ++jv) {
          if (VW == 2) {
            const uint64_t b2 = reinterpret_cast<const uint64_t*>(cb)[((c0 / REP) * NV + jv) * 32 + lane];
            const uint64_t d2 = f2_sub(rm2[jv], b2);
            acc2 = f2_fma(d2, d2, acc2);
          } else {
            const ulonglong2 b4 = reinterpret_cast<const ulonglong2*>(cb)[((c0 / REP) * NV + jv) * 32 + lane];
            const uint64_t d2a = f2_sub(rm2[(2 * jv) % (DS / 2)], b4.x);
            acc2 = f2_fma(d2a, d2a, acc2);
            const uint64_t d2b = f2_sub(rm2[(2 * jv + 1) % (DS / 2)], b4.y);
            acc2 = f2_fma(d2b, d2b, acc2);
          }
        }
        const float t = f2_hsum(acc2);
        const uint32_t v = __float2uint_rn(t * scale);
#pragma unroll
        for (int rep = 0; rep < REP; ++rep) lut[c * 32 + my_m + ((rep + cofs) % REP) * M] = v;
      }
      group_sync(gid);
      // C3 + C4: scan and select
      if (tid == 0) bytes += (unsigned long long)len * M;
      const uint32_t pos0 = (uint32_t)lb;
      for (int v0 = warp * 32; v0 < len; v0 += SCAN_THREADS) {  // a warp stops after its last 32 vectors
        const int v = v0 + lane;
        const bool ok = v < len;
        uint32_t w[MW];
#pragma unroll
        for (int i = 0; i < MW; ++i) w[i] = nxt[i];
        if (v + SCAN_THREADS < len) load_code<MW>(cl + (size_t)(uint32_t)(v + SCAN_THREADS) * M, nxt);
        float dist = 0.f;
        if (ok) {
          xor_permute_bytes<MW>(w, rot);
          uint32_t acc = 0u;
          xor_gather<0, M>(w, lane_base, acc);
          dist = (float)acc * inv_scale;
        }
        const float bound = fminf(sel.thr_val, __uint_as_float(*reinterpret_cast<volatile uint32_t*>(grp_bound + gid)));
        const bool cand = ok && !(dist > bound);
        if (__any_sync(kFull, cand)) {
          const uint64_t key = make_key(dist, pos0 + (uint32_t)v);
          const uint64_t thr_before = sel.thr;
          sel.push(cand && sel.wants(key), key);
          if (sel.thr != thr_before && lane == 0) atomicMin(grp_bound + gid, __float_as_uint(sel.thr_val));
        }
      }
    }
    sel.finish();
    group_sync(gid);  // every warp is done with the table: the merge area takes its place
#pragma unroll
    for (int rr = 0; rr < NQ; ++rr) merge[warp * K + rr * 32 + lane] = sel.W[rr];
    group_sync(gid);
    if (warp == 0) {
      sel.reset();
      for (int e0 = 0; e0 < SCAN_WARPS * K; e0 += 32) {
        const uint64_t key = merge[e0 + lane];
        sel.push(key < sel.thr, key);
      }
      sel.finish();
      uint64_t* W = a.Wg + item * K;
#pragma unroll
      for (int rr = 0; rr < NQ; ++rr) W[rr * 32 + lane] = sel.W[rr];
    }
  }
  if (tid == 0 && bytes) atomicAdd(a.scanned, bytes);
}

// ---------------------------------------------------------------------------
// The grouped fixed-point scan with the paper's table decomposition (Eq. 11, P:L300-311;
// FS_IVFPQ_SCAN=pre):  T_m[c] = ||x^m - c_L^m - B[m][c]||^2
//     = (||B[m][c]||^2 + 2 <c_L^m, B[m][c]>)      term 1: per list, precomputed (ivfpq_term1_kernel)
//     + ||x^m - c_L^m||^2                          term 2: per (query, list, m), constant over c
//     + (-2 <x^m, B[m][c]>)                        term 3: per query, built once per work item
// so the table of a (query, list) pair costs one load, two adds and the conversion per entry
// instead of 2 dsub flops, and no codebook is needed in shared memory (any dsub).  Entries are
// clamped at 0 before the fixed-point conversion (the three terms cancel to rounding).
// Shared memory per group: lut[256][32] (merge area aliases it) | t3[M * 256] | r[d] | select batches
// ---------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(256) ivfpq_term1_kernel(const float* __restrict__ coarse, const float* __restrict__ pq,
                                                          float* __restrict__ term1, int d, int dsub) {
  constexpr int REP = 32 / M;
  const int64_t L = blockIdx.x;
  const float* cL = coarse + L * d;
  for (int e = threadIdx.x; e < M * 256; e += 256) {
    const int st = e >> 5, lane = e & 31;
    const int m = lane % M, c = st * REP + lane / M;
    const float* b = pq + ((int64_t)m * 256 + c) * dsub;
    float bn = 0.f, cb = 0.f;
    for (int j = 0; j < dsub; ++j) {
      bn = fmaf(b[j], b[j], bn);
      cb = fmaf(cL[m * dsub + j], b[j], cb);
    }
    term1[L * (M * 256) + e] = fmaf(2.f, cb, bn);
  }
}

#ifndef FS_PRE_N
#define FS_PRE_N 3
#endif
constexpr int PRE_N = FS_PRE_N;  // groups per CTA (a fourth fits -- no resident codebook -- but measures the same)
constexpr int PRE_THREADS = SCAN_THREADS * PRE_N;

template <int NQ, int M>
__global__ void __launch_bounds__(PRE_THREADS, 1) ivfpq_scan_pre_kernel(const ScanArgs a, unsigned int* __restrict__ work,
                                                                         int64_t n_items) {
  extern __shared__ __align__(1024) unsigned char scan_smem[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int NE = M * 256 / SCAN_THREADS;  // table entries per thread
  static_assert(SCAN_WARPS * K * 8 <= 256 * 32 * 4, "merge area must fit the table it aliases");
  const int d = a.d, dsub = a.dsub, dpad = (d + 3) & ~3;
  const int gid = threadIdx.x / SCAN_THREADS, tid = threadIdx.x % SCAN_THREADS, lane = tid & 31, warp = tid >> 5;
  const size_t grp_bytes = (size_t)256 * 32 * 4 + (size_t)M * 256 * 4 + (size_t)dpad * 4 +
                           (size_t)SCAN_WARPS * warp_select_smem_keys<NB>() * 8;
  unsigned char* gbase = scan_smem + gid * grp_bytes;
  uint32_t* lut = reinterpret_cast<uint32_t*>(gbase);
  float* t3 = reinterpret_cast<float*>(lut + 256 * 32);
  float* r = t3 + M * 256;
  uint64_t* bufs = reinterpret_cast<uint64_t*>(r + dpad);
  uint64_t* merge = reinterpret_cast<uint64_t*>(lut);  // the table is dead when the queues are merged
  __shared__ uint32_t grp_bound[PRE_N];
  __shared__ int grp_item[PRE_N];

  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  unsigned long long bytes = 0;
  const int rot = lane % M;
  const int my_m = lane % M, cofs = lane / M;
  const float my_bmax = a.bmax[my_m];
  const uint32_t lutb = (uint32_t)__cvta_generic_to_shared(lut);

  while (true) {
    group_sync(gid);  // the previous item's merge is done with the table / merge area
    if (tid == 0) {
      grp_item[gid] = (int)atomicAdd(work, 1u);
      grp_bound[gid] = 0x7F800000u;
    }
    group_sync(gid);
    const int64_t item = grp_item[gid];
    if (item >= n_items) break;
    const int64_t q = item / a.ngroups;
    const int g = (int)(item - q * a.ngroups);
    const int p_begin = g * a.G;
    const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;
    sel.reset();
    // term 3 of this query, in the lane order of the build: entry e = step * 32 + lane
    for (int e = tid; e < M * 256; e += SCAN_THREADS) {
      const int st = e >> 5, ln = e & 31;
      const int m = ln % M, c = st * REP + ln / M;
      const float* b = a.pq + ((int64_t)m * 256 + c) * dsub;
      const float* xm = a.xq + q * d + m * dsub;
      float acc = 0.f;
      for (int j = 0; j < dsub; ++j) acc = fmaf(__ldg(xm + j), __ldg(b + j), acc);
      t3[e] = -2.f * acc;
    }

    // The dependent loads of a list (probe id -> list bounds, centroid) are issued one and two
    // lists ahead and stay in registers: none of their latency is on the path.
    const float xj = tid < d ? a.xq[q * d + tid] : 0.f;
    const int64_t* pid = a.probe_ids + q * a.nprobe;
    int64_t L1 = pid[p_begin];
    int64_t L2 = p_begin + 1 < p_end ? pid[p_begin + 1] : -1;
    int64_t lb1 = 0, le1 = 0;
    float c1 = 0.f;
    if (L1 >= 0) {
      lb1 = a.offsets[L1];
      le1 = a.offsets[L1 + 1];
      if (tid < d) c1 = a.coarse[L1 * d + tid];
    }
    for (int p = p_begin; p < p_end; ++p) {
      const int64_t L = L1, lb = lb1, le = le1;
      const float cj = c1;
      L1 = L2;
      if (L1 >= 0) {
        lb1 = a.offsets[L1];
        le1 = a.offsets[L1 + 1];
        if (tid < d) c1 = a.coarse[L1 * d + tid];
      }
      L2 = p + 2 < p_end ? pid[p + 2] : -1;
      if (a.out_probed && tid == 0) a.out_probed[q * a.nprobe + p] = (int32_t)L;
      if (L < 0 || le == lb) continue;  // empty lists are probed and contribute nothing
      const int len = (int)(le - lb);
      // term 1 of this list: this thread's NE entries, requested before anything waits
      float t1[NE];
      const float* t1g = a.term1 + L * (M * 256) + warp * 32 + lane;
#pragma unroll
      for (int i = 0; i < NE; ++i) t1[i] = __ldg(t1g + i * SCAN_THREADS);
      group_sync(gid);  // previous list's table is no longer read (and t3 is complete)
      const uint8_t* cl = a.codes + lb * M;
      uint32_t nxt[MW] = {};
      if (tid < len) load_code<MW>(cl + (size_t)tid * M, nxt);
      if (tid < d) r[tid] = xj - cj;
      group_sync(gid);
      // term 2 of this lane's sub-quantizer, and the scale from the bound
      float n = 0.f;
      for (int j = 0; j < dsub; ++j) {
        const float v = r[my_m * dsub + j];
        n = fmaf(v, v, n);
      }
      float u = sqrtf(n) + my_bmax;
      u = u * u * 1.001f;
#pragma unroll
      for (int sft = 16; sft >= 1; sft >>= 1) u = fmaxf(u, __shfl_xor_sync(kFull, u, sft));
      int ex = 0;
      if (u > 0.f && u < 3.0e38f) frexpf(u, &ex);  // u < 2^ex
      int se = 27 - ex;                            // scaled entries < 2^27
      se = se > 100 ? 100 : (se < -100 ? -100 : se);
      const float scale = __uint_as_float((uint32_t)(127 + se) << 23);
      const float inv_scale = __uint_as_float((uint32_t)(127 - se) << 23);
      const float cap = u;  // the bound also clamps from above: rounding cannot push an entry past it
#pragma unroll
      for (int i = 0; i < NE; ++i) {
        const int st = warp + i * SCAN_WARPS;  // entry e = st * 32 + lane
        const int c = st * REP + cofs;
        float t = (t1[i] + t3[st * 32 + lane]) + n;
        t = fminf(fmaxf(t, 0.f), cap);
        const uint32_t v = __float2uint_rn(t * scale);
#pragma unroll
        for (int rep = 0; rep < REP; ++rep) lut[c * 32 + my_m + ((rep + cofs) % REP) * M] = v;
      }
      group_sync(gid);
      // C3 + C4: scan and select
      const uint32_t lane_base = lutb + ((uint32_t)lane << 2);  // step s reads bank lane ^ s
      if (tid == 0) bytes += (unsigned long long)len * M;
      const uint32_t pos0 = (uint32_t)lb;
      for (int v0 = warp * 32; v0 < len; v0 += SCAN_THREADS) {
        const int v = v0 + lane;
        const bool ok = v < len;
        uint32_t w[MW];
#pragma unroll
        for (int i = 0; i < MW; ++i) w[i] = nxt[i];
        if (v + SCAN_THREADS < len) load_code<MW>(cl + (size_t)(uint32_t)(v + SCAN_THREADS) * M, nxt);
        float dist = 0.f;
        if (ok) {
          xor_permute_bytes<MW>(w, rot);
          uint32_t acc = 0u;
          xor_gather<0, M>(w, lane_base, acc);
          dist = (float)acc * inv_scale;
        }
        const float bound = fminf(sel.thr_val, __uint_as_float(*reinterpret_cast<volatile uint32_t*>(grp_bound + gid)));
        const bool cand = ok && !(dist > bound);
        if (__any_sync(kFull, cand)) {
          const uint64_t key = make_key(dist, pos0 + (uint32_t)v);
          const uint64_t thr_before = sel.thr;
          sel.push(cand && sel.wants(key), key);
          if (sel.thr != thr_before && lane == 0) atomicMin(grp_bound + gid, __float_as_uint(sel.thr_val));
        }
      }
    }
    sel.finish();
    group_sync(gid);  // every warp is done with the table: the merge area takes its place
#pragma unroll
    for (int rr = 0; rr < NQ; ++rr) merge[warp * K + rr * 32 + lane] = sel.W[rr];
    group_sync(gid);
    if (warp == 0) {
      sel.reset();
      for (int e0 = 0; e0 < SCAN_WARPS * K; e0 += 32) {
        const uint64_t key = merge[e0 + lane];
        sel.push(key < sel.thr, key);
      }
      sel.finish();
      uint64_t* W = a.Wg + item * K;
#pragma unroll
      for (int rr = 0; rr < NQ; ++rr) W[rr * 32 + lane] = sel.W[rr];
    }
  }
  if (tid == 0 && bytes) atomicAdd(a.scanned, bytes);
}

template <int NQ, int M>
int launch_scan_pre(const ScanArgs& a, int64_t nq, unsigned int* work, cudaStream_t s) {
  const size_t grp_bytes = (size_t)256 * 32 * 4 + (size_t)M * 256 * 4 + (size_t)((a.d + 3) & ~3) * 4 +
                           (size_t)SCAN_WARPS * warp_select_smem_keys<2>() * 8;
  const size_t smem = PRE_N * grp_bytes;
  if (smem > 227 * 1024) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: shared memory (%zu B) exceeds 227 KB", smem);
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_pre_kernel<NQ, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_smem = smem;
  }
  const int64_t n_items = nq * a.ngroups;
  int64_t grid = sm_count();
  if (grid * PRE_N > n_items) grid = ceil_div(n_items, (int64_t)PRE_N);
  FS_CUDA(cudaMemsetAsync(work, 0, sizeof(unsigned int), s));
  ivfpq_scan_pre_kernel<NQ, M><<<(unsigned)grid, PRE_THREADS, smem, s>>>(a, work, n_items);
  FS_LAUNCHED();
  return FS_OK;
}

template <int NQ, int M, int DS>
int launch_scan_grp(const ScanArgs& a, int64_t nq, unsigned int* work, cudaStream_t s) {
  const size_t grp_bytes = (size_t)256 * 32 * 4 + (size_t)((a.d + 3) & ~3) * 4 +
                           (size_t)SCAN_WARPS * warp_select_smem_keys<2>() * 8;
  const size_t smem = (size_t)256 * a.d * 4 + GRP_N * grp_bytes;
  if (smem > 227 * 1024) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: shared memory (%zu B) exceeds 227 KB", smem);
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_grp_kernel<NQ, M, DS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_smem = smem;
  }
  const int64_t n_items = nq * a.ngroups;
  int64_t grid = sm_count();
  if (grid * GRP_N > n_items) grid = ceil_div(n_items, (int64_t)GRP_N);
  FS_CUDA(cudaMemsetAsync(work, 0, sizeof(unsigned int), s));
  ivfpq_scan_grp_kernel<NQ, M, DS><<<(unsigned)grid, GRP_THREADS, smem, s>>>(a, work, n_items);
  FS_LAUNCHED();
  return FS_OK;
}

template <int NQ, int M, int DS>
int launch_scan_rot(const ScanArgs& a, int64_t nq, cudaStream_t s) {
  constexpr int K = 32 * NQ;
  const size_t smem = (size_t)(256 * 32 + ((a.d + 3) & ~3)) * sizeof(float) +
                      (size_t)(SCAN_WARPS * warp_select_smem_keys<2>() + SCAN_WARPS * K) * sizeof(uint64_t);
  if (smem > 227 * 1024) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: shared memory (%zu B) exceeds 227 KB", smem);
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_rot_kernel<NQ, M, DS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const char* e = getenv("FS_IVFPQ_CARVEOUT");
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan_rot_kernel<NQ, M, DS>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                 e ? atoi(e) : 60));
    attr_smem = smem;
  }
  const int64_t grid = nq * a.ngroups;
  if (grid > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: nq * groups too large");
  ivfpq_scan_rot_kernel<NQ, M, DS><<<(unsigned)grid, SCAN_THREADS, smem, s>>>(a);
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
  // Scan kernels (profiles/r01_ivfpq.md): pair = float tables, one CTA per item; rot = fixed-point
  // conflict-free tables, one CTA per item; grp = the same in persistent groups with the codebook
  // resident in shared memory; pre = grp with the table built from the Eq. 11 terms.  Default: grp
  // where it is measured faster (M = 16, items of >= 32 lists, enough items to fill the persistent
  // groups), else pair.  FS_IVFPQ_SCAN=pair|rot|grp|pre forces one (A/B runs).
  const int forced = scan_forced_mode();
  int mode = forced == 3 ? 0 : forced;
  if (forced == 0 && scan_auto_grouped(a.M, a.G, nq * a.ngroups)) mode = 2;
  if constexpr (NQ <= 8) {
    if (mode == 4 && a.len32 && a.term1 && a.bmax && a.d <= SCAN_THREADS && a.M == 16)
      return launch_scan_pre<NQ, 16>(a, nq, a.work, s);
    if (mode == 4 && a.len32 && a.term1 && a.bmax && a.d <= SCAN_THREADS && a.M == 8)
      return launch_scan_pre<NQ, 8>(a, nq, a.work, s);
    const bool fx = a.len32 && a.pq_r;
    if (mode == 2 && fx && a.d <= SCAN_THREADS && a.M == 16 && a.dsub == 6) return launch_scan_grp<NQ, 16, 6>(a, nq, a.work, s);
    if (mode == 2 && fx && a.d <= SCAN_THREADS && a.M == 8 && a.dsub == 12) return launch_scan_grp<NQ, 8, 12>(a, nq, a.work, s);
    if (mode == 1 && fx && a.M == 16 && a.dsub == 6) return launch_scan_rot<NQ, 16, 6>(a, nq, s);
    if (mode == 1 && fx && a.M == 8 && a.dsub == 12) return launch_scan_rot<NQ, 8, 12>(a, nq, s);
  }
  if (a.pq_t && a.M == 16 && a.dsub == 6) return launch_scan_m<NQ, 16, 6>(a, nq, s);
  if (a.pq_t && a.M == 8 && a.dsub == 12) return launch_scan_m<NQ, 8, 12>(a, nq, s);
  if (a.pq_t && a.M == 16 && a.dsub == 8) return launch_scan_m<NQ, 16, 8>(a, nq, s);   // d = 128
  if (a.pq_t && a.M == 8 && a.dsub == 16) return launch_scan_m<NQ, 8, 16>(a, nq, s);   // d = 128
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
  ix->ev_valid = false;
  FS_CUDA(cudaEventRecord(ix->ev[0], s));
  // C1
  if (p.c1_chunk > 0) {
    float* D = reinterpret_cast<float*>(w + p.off_D);
    float* cval = reinterpret_cast<float*>(w + p.off_cval);
    int32_t* cidx = reinterpret_cast<int32_t*>(w + p.off_cidx);
    for (int64_t q0 = 0; q0 < nq; q0 += p.c1_chunk) {
      const int64_t n = nq - q0 < p.c1_chunk ? nq - q0 : p.c1_chunk;
      rc = flat_knn_tc_device(xq + q0 * ix->d, n, ix->coarse.as<float>(), ix->nlist, ix->d, 1, nullptr, nullptr, w, s,
                              D, p.c1_ld);
      if (rc != FS_OK) return rc;
      rc = kselect_device(D, n, ix->nlist, p.c1_ld, nprobe, cval, cidx, w + p.off_ksws, s);
      if (rc != FS_OK) return rc;
      widen_ids_kernel<<<(unsigned)ceil_div(n * nprobe, 256), 256, 0, s>>>(cidx, cids + q0 * nprobe, n * nprobe);
      FS_LAUNCHED();
    }
  } else {
    rc = flat_knn_device(xq, nq, ix->coarse.as<float>(), ix->nlist, ix->d, nprobe,
                         ix->cnorm.as<float>(), cdist, cids, w, s);
    if (rc != FS_OK) return rc;
  }
  FS_CUDA(cudaEventRecord(ix->ev[1], s));
  FS_CUDA(cudaMemsetAsync(ix->scanned.p, 0, sizeof(unsigned long long), s));
  // C2-C4
  ScanArgs a;
  a.xq = xq;
  a.coarse = ix->coarse.as<float>();
  a.pq = ix->pq.as<float>();
  a.len32 = ix->ntotal() < ((int64_t)1 << 31);
  a.work = reinterpret_cast<unsigned int*>(w + p.off_work);
  a.pq_t = nullptr;
  a.pq_r = nullptr;
  a.bmax = nullptr;
  if ((ix->M == 16 && (ix->dsub == 6 || ix->dsub == 8)) || (ix->M == 8 && (ix->dsub == 12 || ix->dsub == 16))) {
    float* pq_t = reinterpret_cast<float*>(w + p.off_pqt);
    float* pq_r = reinterpret_cast<float*>(w + p.off_pqr);
    const int n = 256 * ix->d;
    pq_regroup_kernel<<<ceil_div(n, 256), 256, 0, s>>>(a.pq, pq_t, pq_r, ix->M, ix->dsub, ix->dsub == 6 ? 2 : 4);
    FS_LAUNCHED();
    a.pq_t = pq_t;
    a.pq_r = pq_r;
  }
  if (ix->M == 16 || ix->M == 8) {
    float* bmax = reinterpret_cast<float*>(w + p.off_pqr) + (size_t)256 * ix->d;
    pq_bmax_kernel<<<ix->M, 32, 0, s>>>(a.pq, bmax, ix->dsub);
    FS_LAUNCHED();
    a.bmax = bmax;
  }
  // Eq. 11 term 1 for every list (16 KB per list at M = 16): built by the first search that wants it
  a.term1 = nullptr;
  if (want_term1(ix)) {
    if (!ix->term1_valid) {
      const size_t tb = (size_t)ix->nlist * ix->M * 256 * sizeof(float);
      if ((rc = ix->term1.ensure(tb, 0, s)) != FS_OK) return rc;
      if (ix->M == 16)
        ivfpq_term1_kernel<16><<<(unsigned)ix->nlist, 256, 0, s>>>(ix->coarse.as<float>(), a.pq, ix->term1.as<float>(),
                                                                  ix->d, ix->dsub);
      else
        ivfpq_term1_kernel<8><<<(unsigned)ix->nlist, 256, 0, s>>>(ix->coarse.as<float>(), a.pq, ix->term1.as<float>(),
                                                                 ix->d, ix->dsub);
      FS_LAUNCHED();
      ix->term1_valid = true;
    }
    a.term1 = ix->term1.as<float>();
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
  FS_CUDA(cudaEventRecord(ix->ev[2], s));
  // C5
  rc = launch_flat_finish(Wg, nq, p.ngroups * qpi, k, nullptr, out_dist, out_ids, s);
  if (rc != FS_OK) return rc;
  const size_t smem = (size_t)4 * k * (sizeof(int64_t) + sizeof(float));
  ivfpq_resolve_kernel<<<(unsigned)ceil_div(nq, 4), 128, smem, s>>>(out_dist, out_ids,
                                                                    ix->ids.as<int64_t>(), nq, k);
  FS_LAUNCHED();
  FS_CUDA(cudaEventRecord(ix->ev[3], s));
  ix->ev_valid = true;
  return FS_OK;
}

}  // namespace fs
