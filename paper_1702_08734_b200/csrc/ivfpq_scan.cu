// ivfpq_scan.cu -- the IVFPQ list scan, persistent form.
//
//   C2 lookup tables   per (query, probed list): r = x - c_L, T_m[c] = ||r^m - B[m][c]||^2
//                      (Eq. 10; direct form), built in shared memory by the CTA that scans
//                      the list from a codebook that is RESIDENT in shared memory
//   C3 list scan       dist = sum_m T_m[code_m] (Alg. 4); one thread per
//                      vector, one 8/16/32-byte load of its code
//   C4 pass-1 select   every warp k-selects what it produces in a register queue; the
//                      CTA's 16 queues are merged per work item
//
// "A significant portion of the runtime is the gather from the T_i in shared memory"
// (P:L325).  On B200 that gather is the co-bound of the scan (one 4-byte lookup per
// code byte), so the table is laid out WITHOUT bank conflicts: word (c, b) of the
// 256 x 32 table lives in bank b and holds T_{b mod M}[c] (32 / M replicas of every
// table), and lane l adds its sub-quantizers in the rotated order m = (s + l) mod M,
// so at step s the 32 lanes read the 32 different banks (s + l) mod 32.  Lane l
// rotates its code by l mod M bytes once per vector (funnel shifts), after which the
// byte of step s sits at a compile-time position.
#include <cstdlib>
#include <cstring>

#include "ivfpq.cuh"
#include "ivfpq_scan.cuh"
#include "select.cuh"

namespace fs {

namespace {

constexpr int SW = 16;              // warps per CTA
constexpr int ST = SW * 32;         // threads per CTA

// Shared memory: cb [256][d+1] | lut [2][256][32] | per-warp select batches | merge area [SW][K]
template <int NQ, int M>
__global__ void __launch_bounds__(ST, 1) ivfpq_scan2_kernel(const ScanArgs a, unsigned int* __restrict__ work,
                                                            int64_t n_items) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int K = 32 * NQ;
  constexpr int NB = 2;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int DSUB_MAX = 16;
  const int d = a.d, dsub = a.dsub, dp = d + 1;
  float* cb = reinterpret_cast<float*>(smem_raw);  // codeword c of all sub-quantizers: cb[c * dp + m * dsub + j]
  float* lut0 = cb + 256 * dp;                     // two tables: the next one is built while slow warps still scan
  uint64_t* bufs = reinterpret_cast<uint64_t*>(lut0 + 2 * 256 * 32);
  uint64_t* merge = bufs + SW * warp_select_smem_keys<NB>();
  __shared__ int s_item;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // the codebook becomes resident: pq [M][256][dsub] -> cb
  for (int e = tid; e < M * 256; e += ST) {
    const int m = e >> 8, c = e & 255;
    for (int j = 0; j < dsub; ++j) cb[c * dp + m * dsub + j] = a.pq[(int64_t)e * dsub + j];
  }
  __syncthreads();

  WarpSelect<NQ, NB> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB>(), lane);
  const int rot = lane % M;
  const int my_m = lane % M, my_cofs = lane / M;
  unsigned long long bytes = 0;
  int which = 0;

  while (true) {
    __syncthreads();
    if (tid == 0) s_item = (int)atomicAdd(work, 1u);
    __syncthreads();
    const int64_t item = s_item;
    if (item >= n_items) break;
    const int64_t q = item / a.ngroups;
    const int g = (int)(item - q * a.ngroups);
    const int p_begin = g * a.G;
    const int p_end = (p_begin + a.G) < a.nprobe ? (p_begin + a.G) : a.nprobe;
    sel.reset();

    for (int p = p_begin; p < p_end; ++p) {
      const int64_t L = a.probe_ids[q * a.nprobe + p];
      if (a.out_probed && tid == 0) a.out_probed[q * a.nprobe + p] = (int32_t)L;
      if (L < 0) continue;
      const int64_t lb = a.offsets[L], le = a.offsets[L + 1];
      const int64_t len = le - lb;
      if (len == 0) continue;  // empty lists are probed and contribute nothing
      // C2: this lane's residual sub-vector r^m = (x - c_L)^m in registers, then its share of
      // the table: entry (m = lane % M, c = c0 + lane / M) goes to the REP banks of table m
      float* lut = lut0 + which * (256 * 32);
      float rm[DSUB_MAX];
#pragma unroll
      for (int j = 0; j < DSUB_MAX; ++j)
        rm[j] = j < dsub ? __ldg(a.xq + q * d + my_m * dsub + j) - __ldg(a.coarse + L * d + my_m * dsub + j) : 0.f;
      for (int c0 = warp * REP; c0 < 256; c0 += SW * REP) {
        const int c = c0 + my_cofs;
        const float* b = cb + c * dp + my_m * dsub;
        float t = 0.f;
#pragma unroll
        for (int j = 0; j < DSUB_MAX; ++j) {
          if (j < dsub) {
            const float df = rm[j] - b[j];
            t = fmaf(df, df, t);
          }
        }
#pragma unroll
        for (int rep = 0; rep < REP; ++rep) lut[c * 32 + my_m + rep * M] = t;
      }
      __syncthreads();  // table complete (and every warp is past the scan that used the other one)
      // C3 + C4: scan and select
      bytes += (unsigned long long)len * M;
      const uint8_t* cl = a.codes + lb * M;
      const char* lutb = reinterpret_cast<const char*>(lut);
      for (int64_t v0 = (int64_t)warp * 32; v0 < len; v0 += ST) {
        const int64_t v = v0 + lane;
        const bool ok = v < len;
        float dist = 0.f;
        if (ok) {
          uint32_t w[MW];
          load_code<MW>(cl + v * M, w);
          rotate_bytes<MW>(w, rot);
#pragma unroll
          for (int s = 0; s < M; ++s) {
            const uint32_t c = (w[s >> 2] >> (8 * (s & 3))) & 255u;
            dist += *reinterpret_cast<const float*>(lutb + c * 128 + (((s + lane) & 31) << 2));
          }
        }
        const bool cand = ok && sel.maybe(dist);
        if (__any_sync(kFull, cand)) {
          const uint64_t key = make_key(dist, (uint32_t)(lb + v));
          sel.push(cand && sel.wants(key), key);
        }
      }
      which ^= 1;
    }
    sel.finish();

    // merge the warps' queues: warp 0 selects again over SW * K keys
    __syncthreads();
#pragma unroll
    for (int rr = 0; rr < NQ; ++rr) merge[warp * K + rr * 32 + lane] = sel.W[rr];
    __syncthreads();
    if (warp == 0) {
      sel.reset();
      for (int e0 = 0; e0 < SW * K; e0 += 32) {
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
size_t scan2_smem(int d) {
  constexpr int K = 32 * NQ;
  return (size_t)(256 * (d + 1) + 2 * 256 * 32) * sizeof(float) +
         (size_t)(SW * warp_select_smem_keys<2>() + SW * K) * sizeof(uint64_t);
}

template <int NQ, int M>
int launch_scan2_t(const ScanArgs& a, int64_t nq, unsigned int* work, cudaStream_t s) {
  const size_t smem = scan2_smem<NQ, M>(a.d);
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan2_kernel<NQ, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_smem = smem;
  }
  const int64_t n_items = nq * a.ngroups;
  int64_t grid = sm_count();
  if (grid > n_items) grid = n_items;
  FS_CUDA(cudaMemsetAsync(work, 0, sizeof(unsigned int), s));
  ivfpq_scan2_kernel<NQ, M><<<(unsigned)grid, ST, smem, s>>>(a, work, n_items);
  FS_LAUNCHED();
  return FS_OK;
}

template <int M>
int launch_scan2_m(int kclass, const ScanArgs& a, int64_t nq, unsigned int* work, cudaStream_t s) {
  switch (kclass) {
    case 0: return launch_scan2_t<1, M>(a, nq, work, s);
    case 1: return launch_scan2_t<2, M>(a, nq, work, s);
    case 2: return launch_scan2_t<4, M>(a, nq, work, s);
    default: return launch_scan2_t<8, M>(a, nq, work, s);
  }
}

}  // namespace

bool scan2_supported(int d, int M, int k) {
  // Opt-in (FS_IVFPQ_SCAN=persistent) until it beats the per-pair kernel of ivfpq_search.cu:
  // with ~1.5 k vectors per list the 16 warps of a CTA spend as long on the table and its
  // barriers as on the scan (profiles/r01_ivfpq_scan.md), and the rotated summation order
  // reorders distances that differ in the last bits.
  static int on = -1;
  if (on < 0) {
    const char* e = getenv("FS_IVFPQ_SCAN");
    on = (e && strcmp(e, "persistent") == 0) ? 1 : 0;
  }
  if (!on) return false;
  if (!(M == 8 || M == 16 || M == 32)) return false;
  const int kc = k_class(k);
  if (kc > 3) return false;  // the merge area of larger queues does not fit beside the codebook
  if (d / M > 16) return false;
  const size_t smem = (size_t)(256 * (d + 1) + 2 * 256 * 32) * sizeof(float) +
                      (size_t)(SW * warp_select_smem_keys<2>() + SW * (32 << kc)) * sizeof(uint64_t);
  return smem <= 224 * 1024;
}

int launch_scan2(const ScanArgs& a, int64_t nq, int k, unsigned int* work, cudaStream_t s) {
  const int kc = k_class(k);
  switch (a.M) {
    case 8: return launch_scan2_m<8>(kc, a, nq, work, s);
    case 16: return launch_scan2_m<16>(kc, a, nq, work, s);
    default: return launch_scan2_m<32>(kc, a, nq, work, s);
  }
}

}  // namespace fs
