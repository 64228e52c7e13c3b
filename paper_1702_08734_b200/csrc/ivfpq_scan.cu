// ivfpq_scan.cu -- the IVFPQ list scan, persistent form.
//
//   C2 lookup tables   per (query, probed list): r = x - c_L, T_m[c] = ||r^m - B[m][c]||^2
//                      (Eq. 10; direct form), built from a codebook that is
//                      RESIDENT in shared memory for the life of the CTA
//   C3 list scan       dist = sum_m T_m[code_m] (Alg. 4); one thread per
//                      vector, one 8 / 16-byte load of its code
//   C4 pass-1 select   every warp k-selects what it produces in a register queue; the
//                      CTA's 16 queues are merged per work item
//
// Why this shape (profiles/r01_ivfpq.md): the per-pair kernel of ivfpq_search.cu runs the
// L1 / shared-memory data pipe at 94 % -- 3.3 wavefronts per table lookup (random banks) and
// the 96 KB codebook re-read through L1 for every pair.  "A significant portion of the
// runtime is the gather from the T_i in shared memory" is still true on B200.  Here
//   * the table is stored as lut[c][b], b = 0..31: word (c, b) lives in bank b and holds
//     T_{b mod M}[c] (32 / M replicas); lane l adds its sub-quantizers in the rotated order
//     m = (s + l) mod M, so at step s the 32 lanes read the 32 different banks (s + l) mod 32:
//     ONE wavefront per lookup.  Lane l rotates its code by l mod M bytes once per vector;
//   * so that the rotated order cannot change the sum, entries are FIXED-POINT: one power-of-two
//     scale per (query, list) pair, from the bound (||r^m|| + max_c ||B[m][c]||)^2 >= every entry
//     of T_m, makes every entry an integer < 2^27; the scan adds integers (exact, associative),
//     so identical codes give identical distances whatever lane scans them (DESIGN reading
//     C-6).  Quantisation: <= 2^-27 of the bound per entry, M times that per distance;
//   * the codebook is read from shared memory, conflict-free (row stride d + 1 words);
//   * one CTA of 16 warps per SM walks its (query, list) pairs in a software pipeline: in
//     phase t it scans pair t with table t & 1 while it builds table (t + 1) & 1 for pair
//     t + 1, and the dependent global loads of later pairs (probe id -> list bounds and
//     coarse centroid -> residual) are issued one hop per phase, two and three pairs ahead,
//     so none of their latency is on the path.  One __syncthreads per pair.
#include <cstdlib>
#include <cstring>

#include "ivfpq.cuh"
#include "ivfpq_scan.cuh"
#include "select.cuh"

namespace fs {

namespace {

constexpr int SW = 16;       // warps per CTA
constexpr int ST = SW * 32;  // threads per CTA
constexpr int NB3 = 2;       // select batch: 32 * NB3 keys per warp

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}

// dist += lut[byte s of w][bank (s + lane) mod 32] for s = s0 .. M-1; base[s] = table + 4 * bank
template <int s, int M>
__device__ __forceinline__ void gather_all(const uint32_t* w, const uint32_t* base, uint32_t& acc) {
  if constexpr (s < M) {
    const uint32_t c = __byte_perm(w[s >> 2], 0u, 0x4440u + (s & 3));  // byte s, zero-extended
    acc += lds_u32(base[s] + c * 128u);
    gather_all<s + 1, M>(w, base, acc);
  }
}

// Shared-memory plan (bytes) -- the kernel carves the same way
struct Scan3Smem {
  size_t lut, cb, rr, bmax, meta, bufs, merge, total;
};
__host__ __device__ inline Scan3Smem scan3_smem(int d, int K) {
  Scan3Smem s;
  size_t o = 0;
  s.lut = o;
  o += (size_t)2 * 256 * 32 * 4;
  s.cb = o;
  o += (size_t)((256 * (d + 1) + 3) & ~3) * 4;
  s.rr = o;
  o += (size_t)2 * ((d + 3) & ~3) * 4;
  s.bmax = o;
  o += 32 * 4;
  s.meta = o;
  o += 4 * 8 + 4 * 8 + 4 * 4 + 4 * 4 + 16;  // lb[4] q[4] len[4] L[4] ithr[2] (+pad)
  s.bufs = o;
  o += (size_t)SW * warp_select_smem_keys<NB3>() * 8;
  s.merge = o;  // (no merge area: every warp's queue goes to global memory, merged by the C5 pass)
  (void)K;
  s.total = o;
  return s;
}

// DS = d / M when it is 6 or 12 (loops unrolled exactly), else 0 (run-time dsub <= 16).
template <int NQ, int M, int DS>
__global__ void __launch_bounds__(ST, 1) ivfpq_scan3_kernel(const ScanArgs a, int64_t n_items) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  constexpr int K = 32 * NQ;
  constexpr int MW = M / 4;
  constexpr int REP = 32 / M;
  constexpr int DSB = DS ? DS : 16;
  const int d = a.d, dsub = DS ? DS : a.dsub, dp = d + 1, dpad = (d + 3) & ~3;
  const Scan3Smem lay = scan3_smem(d, K);
  uint32_t* lut0 = reinterpret_cast<uint32_t*>(smem_raw + lay.lut);  // two tables [256][32]
  float* cb = reinterpret_cast<float*>(smem_raw + lay.cb);           // cb[c * dp + m * dsub + j]
  float* rr = reinterpret_cast<float*>(smem_raw + lay.rr);           // two residuals
  float* bmax = reinterpret_cast<float*>(smem_raw + lay.bmax);       // max_c ||B[m][c]||
  int64_t* m_lb = reinterpret_cast<int64_t*>(smem_raw + lay.meta);   // rings of 4 pairs
  int64_t* m_q = m_lb + 4;
  int* m_len = reinterpret_cast<int*>(m_q + 4);
  int* m_L = m_len + 4;
  uint64_t* bufs = reinterpret_cast<uint64_t*>(smem_raw + lay.bufs);
  uint32_t* ithr = reinterpret_cast<uint32_t*>(m_L + 4);  // per item parity: min over warps of their K-th distance
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // the codebook becomes resident: pq [M][256][dsub] -> cb
  for (int i = tid; i < 256 * d; i += ST) {
    const int m = i / (256 * dsub);
    const int rem = i - m * 256 * dsub;
    const int c = rem / dsub;
    cb[c * dp + m * dsub + (rem - c * dsub)] = a.pq[i];
  }
  if (tid < 2) ithr[tid] = 0x7F800000u;
  if (tid < 4) {
    m_L[tid] = -1;
    m_len[tid] = 0;
    m_lb[tid] = 0;
    m_q[tid] = 0;
  }
  __syncthreads();
  if (warp < M) {  // M <= SW
    float mx = 0.f;
    for (int c = lane; c < 256; c += 32) {
      float n = 0.f;
      for (int j = 0; j < dsub; ++j) {
        const float v = cb[c * dp + warp * dsub + j];
        n = fmaf(v, v, n);
      }
      mx = fmaxf(mx, n);
    }
#pragma unroll
    for (int sft = 16; sft >= 1; sft >>= 1) mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, sft));
    if (lane == 0) bmax[warp] = sqrtf(mx);
  }
  __syncthreads();

  WarpSelect<NQ, NB3> sel;
  sel.init(bufs + warp * warp_select_smem_keys<NB3>(), lane);
  unsigned long long bytes = 0;
  const int rot = lane % M;
  const int my_m = lane % M, cofs = lane / M;
  const int64_t my_items =
      (int64_t)blockIdx.x < n_items ? (n_items - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const int T = (int)(my_items * a.G);  // pairs this CTA walks (an item's tail pairs may be void)

  int li = 0, pg = 0;    // item and pair-in-item of phase ph (valid for ph >= 0)
  int liA = 0, pgA = 0;  // the same for pair ph + 3
  float inv0 = 1.f;      // 1 / scale of the table of pair ph

  for (int ph = -3; ph < T; ++ph) {
    // the bound of the item that ended one phase ago is reset for the item after this one
    if (ph >= 0 && pg == 0 && tid == 0) ithr[(li + 1) & 1] = 0x7F800000u;
    // ---- hop 1 (thread 0): probe id of pair ph + 3
    int A_L = -1, A_p = 0;
    int64_t A_q = 0;
    const bool A_on = tid == 0 && ph + 3 < T;
    if (A_on) {
      const int64_t it = (int64_t)blockIdx.x + (int64_t)liA * gridDim.x;
      A_q = it / a.ngroups;
      A_p = (int)(it - A_q * a.ngroups) * a.G + pgA;
      if (A_p < a.nprobe) A_L = (int)a.probe_ids[A_q * a.nprobe + A_p];
    }
    // ---- hop 2: list bounds and residual operands of pair ph + 2 (its list id is in the ring)
    const int tB = ph + 2, sB = tB & 3;
    const bool B_on = tB >= 0 && tB < T;
    const int B_L = B_on ? m_L[sB] : -1;
    float B_x = 0.f, B_c = 0.f;
    int64_t B_lb = 0, B_le = 0;
    if (B_L >= 0) {
      if (tid < d) {
        B_x = __ldg(a.xq + m_q[sB] * d + tid);
        B_c = __ldg(a.coarse + (int64_t)B_L * d + tid);
      }
      if (tid == ST - 1) {
        B_lb = a.offsets[B_L];
        B_le = a.offsets[B_L + 1];
      }
    }
    // ---- pair ph: its first codes are requested before the table of pair ph + 1 is built
    const int s0 = ph & 3;
    const bool on0 = ph >= 0 && m_L[s0] >= 0 && m_len[s0] > 0;
    const int len0 = on0 ? m_len[s0] : 0;
    const int64_t lb0 = m_lb[s0];
    const uint8_t* cl = a.codes + lb0 * M;
    uint32_t nxt[MW] = {};
    if (warp * 32 + lane < len0) load_code<MW>(cl + (size_t)(warp * 32 + lane) * M, nxt);
    // ---- pair ph + 1: scale from the bound, then the fixed-point table
    const int t1 = ph + 1, s1 = t1 & 3;
    const bool on1 = t1 >= 0 && t1 < T && m_L[s1] >= 0 && m_len[s1] > 0;
    float inv1 = 1.f;
    if (on1) {
      const float* r1 = rr + (t1 & 1) * dpad;
      float rm[DSB];
      float n = 0.f;
#pragma unroll
      for (int j = 0; j < DSB; ++j) {
        rm[j] = (DS != 0 || j < dsub) ? r1[my_m * dsub + j] : 0.f;
        n = fmaf(rm[j], rm[j], n);
      }
      float u = sqrtf(n) + bmax[my_m];
      u = u * u * 1.001f;  // >= every entry of T_m as the float code below computes it
#pragma unroll
      for (int sft = 16; sft >= 1; sft >>= 1) u = fmaxf(u, __shfl_xor_sync(kFull, u, sft));
      int ex = 0;
      if (u > 0.f && u < 3.0e38f) frexpf(u, &ex);  // u < 2^ex
      int se = 27 - ex;                            // scaled entries < 2^27
      se = se > 100 ? 100 : (se < -100 ? -100 : se);
      const float scale = __uint_as_float((uint32_t)(127 + se) << 23);
      inv1 = __uint_as_float((uint32_t)(127 - se) << 23);
      uint32_t* lut = lut0 + (t1 & 1) * (256 * 32);
      for (int c0 = warp * REP; c0 < 256; c0 += SW * REP) {
        const int c = c0 + cofs;
        const float* b = cb + c * dp + my_m * dsub;
        float t = 0.f;
#pragma unroll
        for (int j = 0; j < DSB; ++j) {
          if (DS != 0 || j < dsub) {
            const float df = rm[j] - b[j];
            t = fmaf(df, df, t);
          }
        }
        const uint32_t v = __float2uint_rn(t * scale);
        // replica (rep + cofs) mod REP at store rep: the 32 lanes write 32 different banks
#pragma unroll
        for (int rep = 0; rep < REP; ++rep) lut[c * 32 + my_m + ((rep + cofs) % REP) * M] = v;
      }
    }
    // ---- pair ph: scan and select (C3 + C4)
    if (on0) {
      const uint32_t lutb = smem_addr(lut0 + (ph & 1) * (256 * 32));
      uint32_t base[M];
#pragma unroll
      for (int s = 0; s < M; ++s) base[s] = lutb + (((lane + s) & 31) << 2);
      for (int v0 = warp * 32; v0 < len0; v0 += ST) {
        const int v = v0 + lane;
        const bool ok = v < len0;
        uint32_t w[MW];
#pragma unroll
        for (int i = 0; i < MW; ++i) w[i] = nxt[i];
        if (v + ST < len0) load_code<MW>(cl + (size_t)(v + ST) * M, nxt);
        float dist = 0.f;
        if (ok) {
          rotate_bytes<MW>(w, rot);
          uint32_t acc = 0u;
          gather_all<0, M>(w, base, acc);
          dist = (float)acc * inv0;
        }
        // the item's K-th distance is <= every warp's K-th: the smallest published one bounds all
        const float bound = fminf(sel.thr_val, __uint_as_float(*reinterpret_cast<volatile uint32_t*>(ithr + (li & 1))));
        const bool cand = ok && !(dist > bound);
        if (__any_sync(kFull, cand)) {  // the exact key is only built when some lane may have a winner
          const uint64_t key = make_key(dist, (uint32_t)(lb0 + v));
          const uint64_t thr_before = sel.thr;
          sel.push(cand && sel.wants(key), key);
          if (sel.thr != thr_before && lane == 0) atomicMin(ithr + (li & 1), __float_as_uint(sel.thr_val));
        }
      }
      if (tid == 0) bytes += (unsigned long long)len0 * M;
    }
    // ---- item end: every warp's queue goes to global memory (merged by the C5 pass)
    if (ph >= 0 && pg == a.G - 1) {
      sel.finish();
      uint64_t* W = a.Wg + (((int64_t)blockIdx.x + (int64_t)li * gridDim.x) * SW + warp) * K;
#pragma unroll
      for (int rr_ = 0; rr_ < NQ; ++rr_) W[rr_ * 32 + lane] = sel.W[rr_];
      sel.reset();
    }
    // ---- the hops land: their values are first touched here, a whole phase after the loads
    asm volatile("" : "+r"(A_L), "+f"(B_x), "+f"(B_c), "+l"(B_lb), "+l"(B_le));
    if (A_on) {
      m_L[(ph + 3) & 3] = A_L;
      m_q[(ph + 3) & 3] = A_q;
      if (A_L >= 0 && a.out_probed) a.out_probed[A_q * a.nprobe + A_p] = (int32_t)A_L;
    }
    if (B_on) {
      if (tid < d) rr[(tB & 1) * dpad + tid] = B_x - B_c;
      if (tid == ST - 1) {
        m_lb[sB] = B_lb;
        m_len[sB] = B_L >= 0 ? (int)(B_le - B_lb) : 0;
      }
    }
    __syncthreads();
    inv0 = inv1;
    if (ph >= 0 && ++pg == a.G) {
      pg = 0;
      ++li;
    }
    if (++pgA == a.G) {
      pgA = 0;
      ++liA;
    }
  }
  if (tid == 0 && bytes) atomicAdd(a.scanned, bytes);
}

template <int NQ, int M, int DS>
int launch_scan3_t(const ScanArgs& a, int64_t nq, cudaStream_t s) {
  const size_t smem = scan3_smem(a.d, 32 * NQ).total;
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    FS_CUDA(cudaFuncSetAttribute(ivfpq_scan3_kernel<NQ, M, DS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_smem = smem;
  }
  const int64_t n_items = nq * a.ngroups;
  int64_t grid = sm_count();
  if (grid > n_items) grid = n_items;
  ivfpq_scan3_kernel<NQ, M, DS><<<(unsigned)grid, ST, smem, s>>>(a, n_items);
  FS_LAUNCHED();
  return FS_OK;
}

template <int M, int DS>
int launch_scan3_m(int kclass, const ScanArgs& a, int64_t nq, cudaStream_t s) {
  switch (kclass) {
    case 0: return launch_scan3_t<1, M, DS>(a, nq, s);
    case 1: return launch_scan3_t<2, M, DS>(a, nq, s);
    default: return launch_scan3_t<4, M, DS>(a, nq, s);
  }
}

}  // namespace

bool scan2_supported(int d, int M, int k) {
  // Opt-in (FS_IVFPQ_SCAN=persistent).  It removes what binds the per-pair kernel (one wavefront
  // per lookup, no codebook traffic) but 16 warps in step on one table issue only ~55 % of the
  // time and execute ~12 k instructions per pair: 53.9 ms against 40.1 ms at nprobe 256
  // (profiles/r01_ivfpq.md).  Kept as the base of the warp-decoupled version.
  static int on = -1;
  if (on < 0) {
    const char* e = getenv("FS_IVFPQ_SCAN");
    on = (e && strcmp(e, "persistent") == 0) ? 1 : 0;
  }
  if (!on) return false;
  if (!(M == 8 || M == 16)) return false;
  if (d % M != 0 || d / M > 16 || d > ST) return false;
  const int kc = k_class(k);
  if (kc > 2) return false;
  return scan3_smem(d, 32 << kc).total <= 227 * 1024;
}

int scan2_queues_per_item() { return SW; }

int launch_scan2(const ScanArgs& a, int64_t nq, int k, unsigned int* /*work*/, cudaStream_t s) {
  const int kc = k_class(k);
  if (a.M == 16) return a.dsub == 6 ? launch_scan3_m<16, 6>(kc, a, nq, s) : launch_scan3_m<16, 0>(kc, a, nq, s);
  return a.dsub == 12 ? launch_scan3_m<8, 12>(kc, a, nq, s) : launch_scan3_m<8, 0>(kc, a, nq, s);
}

}  // namespace fs
