// ivfpq.cu -- IVFADC index: object, quantizers, add path,
// inverted-file maintenance, export and the fs_ivfpq_* C ABI.
//
//   D1 coarse assign  q1(y) = argmin_c ||y - c||^2: the exact-search engine with
//                     k = 1 over the centroids (flat.cu)
//   D2 PQ encode      r = y - q1(y); code_m = argmin_c ||r^m - B[m][c]||^2, ties to
//                     the lower c; byte m = sub-quantizer m (Eq. 3)
//   D3 append         (code, id) staged in arrival order; finalise groups them by
//                     list with a STABLE radix sort on the list number, so every
//                     list keeps append order
#include "ivfpq.cuh"

#include "flat.cuh"
#include "select.cuh"

namespace fs {

// ---------------------------------------------------------------------------
// DevBuf
// ---------------------------------------------------------------------------
int DevBuf::ensure(size_t bytes, size_t keep, cudaStream_t s) {
  if (bytes <= cap) return FS_OK;
  size_t ncap = cap + cap / 2;
  if (ncap < bytes) ncap = bytes;
  ncap = align_up(ncap, 256);
  void* np = nullptr;
  cudaError_t e = cudaMalloc(&np, ncap);
  if (e != cudaSuccess) {
    // second chance: exactly what is needed
    ncap = align_up(bytes, 256);
    e = cudaMalloc(&np, ncap);
    if (e != cudaSuccess) {
      cudaGetLastError();
      return set_error(FS_ENOMEM, "cudaMalloc(%zu) failed: %s", ncap, cudaGetErrorString(e));
    }
  }
  if (keep > 0 && p != nullptr) {
    FS_CUDA(cudaMemcpyAsync(np, p, keep, cudaMemcpyDeviceToDevice, s));
  }
  FS_CUDA(cudaStreamSynchronize(s));
  if (p) cudaFree(p);
  p = np;
  cap = ncap;
  return FS_OK;
}
void DevBuf::release() {
  if (p) cudaFree(p);
  p = nullptr;
  cap = 0;
}

// ---------------------------------------------------------------------------
// D2: residual PQ encoding.
// CTA = 8 warps; a tile of TV = 32 vectors; sub-quantizers one after another:
// the 256 codewords of sub-quantizer m and the tile's residual sub-vectors sit in
// shared memory; a warp takes 4 vectors at a time, lane l owns codewords
// l, l+32, .., l+224 (4 x 8 accumulators), distances in the direct form
// sum_j (r_j - b_j)^2 in fp32; argmin over (distance, c) packed keys by shuffles.
// ---------------------------------------------------------------------------
namespace {
constexpr int ENC_WARPS = 8, ENC_TV = 32, ENC_VPW = 4;

__global__ void __launch_bounds__(ENC_WARPS * 32)
    pq_encode_kernel(const float* __restrict__ y, int64_t n, int d, int M, int dsub,
                     const float* __restrict__ coarse, const int64_t* __restrict__ assign,
                     const float* __restrict__ pq, uint8_t* __restrict__ codes_out,
                     uint32_t* __restrict__ list_out, float* __restrict__ s1_out) {
  extern __shared__ __align__(16) float enc_smem[];
  const int dsp = dsub | 1;                    // odd stride: conflict-free codeword reads
  float* cb = enc_smem;                        // [256][dsp]
  float* res = cb + 256 * dsp;                 // [TV][dsub]
  float* cen = res + ENC_TV * dsub;            // [TV][dsub] the centroid's sub-vector (for term 1)
  float* s1a = cen + ENC_TV * dsub;            // [TV] term 1 accumulated over the sub-quantizers
  uint8_t* cd = reinterpret_cast<uint8_t*>(s1a + ENC_TV);  // [TV][M]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t ntiles = (n + ENC_TV - 1) / ENC_TV;
  for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int64_t v0 = tile * ENC_TV;
    const int nv = (int)((n - v0) < ENC_TV ? (n - v0) : ENC_TV);
    __syncthreads();
    if (tid < ENC_TV) s1a[tid] = 0.f;
    for (int m = 0; m < M; ++m) {
      __syncthreads();
      for (int e = tid; e < 256 * dsub; e += ENC_WARPS * 32) {
        const int c = e / dsub, j = e - c * dsub;
        cb[c * dsp + j] = pq[((int64_t)m * 256 + c) * dsub + j];
      }
      for (int e = tid; e < ENC_TV * dsub; e += ENC_WARPS * 32) {
        const int v = e / dsub, j = e - v * dsub;
        float r = 0.f, cj = 0.f;
        if (v < nv) {
          const int64_t L = assign[v0 + v];
          cj = coarse[L * d + m * dsub + j];
          r = y[(v0 + v) * d + m * dsub + j] - cj;
        }
        res[e] = r;
        cen[e] = cj;
      }
      __syncthreads();
      // warp w: vectors w*4 .. w*4+3
      float acc[ENC_VPW][8];
#pragma unroll
      for (int v = 0; v < ENC_VPW; ++v)
#pragma unroll
        for (int c = 0; c < 8; ++c) acc[v][c] = 0.f;
      const float* rw = res + warp * ENC_VPW * dsub;
      for (int j = 0; j < dsub; ++j) {
        float b[8], r[ENC_VPW];
#pragma unroll
        for (int c = 0; c < 8; ++c) b[c] = cb[(c * 32 + lane) * dsp + j];
#pragma unroll
        for (int v = 0; v < ENC_VPW; ++v) r[v] = rw[v * dsub + j];
#pragma unroll
        for (int v = 0; v < ENC_VPW; ++v)
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            const float t = r[v] - b[c];
            acc[v][c] = fmaf(t, t, acc[v][c]);
          }
      }
#pragma unroll
      for (int v = 0; v < ENC_VPW; ++v) {
        uint64_t best = kSentinelKey;
#pragma unroll
        for (int c = 0; c < 8; ++c) best = umin64(best, make_key(acc[v][c], (uint32_t)(c * 32 + lane)));
#pragma unroll
        for (int s = 16; s >= 1; s >>= 1) best = umin64(best, shfl_xor64(best, s));
        const int cbest = (int)key_idx(best);
        if (lane == 0) cd[(warp * ENC_VPW + v) * M + m] = (uint8_t)cbest;
        // Eq. 11 term 1 of this sub-quantizer: ||B||^2 + 2 <c, B> = sum_j B_j (B_j + 2 c_j), in dimension
        // order by one lane (fixed order: the same vector always gets the same bits)
        if (lane == 0) {
          const float* bw = cb + cbest * dsp;
          const float* cw = cen + (warp * ENC_VPW + v) * dsub;
          float t = 0.f;
          for (int j = 0; j < dsub; ++j) t = fmaf(bw[j], bw[j] + 2.f * cw[j], t);
          s1a[warp * ENC_VPW + v] += t;
        }
      }
    }
    __syncthreads();
    for (int e = tid; e < nv * M; e += ENC_WARPS * 32) codes_out[v0 * M + e] = cd[e];
    if (tid < nv) {
      list_out[v0 + tid] = (uint32_t)assign[v0 + tid];
      s1_out[v0 + tid] = s1a[tid];
    }
  }
}
}  // namespace

int launch_pq_encode(const fs_ivfpq* ix, const float* y, int64_t n, const int64_t* assign,
                     uint8_t* codes_out, uint32_t* list_out, float* s1_out, cudaStream_t s) {
  if (n == 0) return FS_OK;
  const int dsub = ix->dsub, dsp = dsub | 1;
  const size_t smem = (size_t)(256 * dsp + 2 * ENC_TV * dsub + ENC_TV) * sizeof(float) + (size_t)ENC_TV * ix->M;
  FS_CUDA(cudaFuncSetAttribute(pq_encode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));  // per device
  const int64_t ntiles = ceil_div(n, ENC_TV);
  const int64_t maxg = (int64_t)sm_count() * 8;
  pq_encode_kernel<<<(unsigned)(ntiles < maxg ? ntiles : maxg), ENC_WARPS * 32, smem, s>>>(
      y, n, ix->d, ix->M, dsub, ix->coarse.as<float>(), assign, ix->pq.as<float>(), codes_out,
      list_out, s1_out);
  FS_LAUNCHED();
  return FS_OK;
}

// ---------------------------------------------------------------------------
// D3: stable LSD radix sort of (list number, arrival index), 8 bits per pass.
// Every WARP owns a contiguous range of the input and walks it 32 keys at a time:
// __match_any_sync gives each key its rank among the equal digits of the step, a
// per-warp table of 256 running offsets gives the rest -- no block-level
// synchronisation, and stability by construction.
// ---------------------------------------------------------------------------
namespace {
constexpr int RS_WARPS = 8;

__global__ void __launch_bounds__(RS_WARPS * 32)
    rs_hist_kernel(const uint32_t* __restrict__ keys, int64_t n, int shift, int64_t per_warp,
                   uint32_t* __restrict__ hist, int nwt) {
  __shared__ uint32_t h[RS_WARPS][256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t w = (int64_t)blockIdx.x * RS_WARPS + warp;
  for (int i = lane; i < 256; i += 32) h[warp][i] = 0;
  __syncwarp();
  const int64_t b = w * per_warp;
  int64_t e = b + per_warp;
  if (e > n) e = n;
  for (int64_t i0 = b; i0 < e; i0 += 32) {
    const int64_t i = i0 + lane;
    const bool ok = i < e;
    const uint32_t dig = ok ? ((keys[i] >> shift) & 255u) : (256u + lane);
    const unsigned peers = __match_any_sync(kFull, dig);
    if (ok && lane == __ffs(peers) - 1) h[warp][dig] += __popc(peers);
    __syncwarp();
  }
  for (int i = lane; i < 256; i += 32) hist[(int64_t)i * nwt + w] = h[warp][i];
}

// Exclusive scan in place, one CTA of 1024 threads.
__global__ void __launch_bounds__(1024) rs_scan_kernel(uint32_t* __restrict__ a, int64_t len) {
  __shared__ uint32_t part[1024];
  const int t = threadIdx.x;
  const int64_t per = (len + 1023) / 1024;
  const int64_t b = t * per;
  int64_t e = b + per;
  if (e > len) e = len;
  uint32_t sum = 0;
  for (int64_t i = b; i < e; ++i) sum += a[i];
  part[t] = sum;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    const uint32_t v = t >= off ? part[t - off] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  uint32_t run = part[t] - sum;
  for (int64_t i = b; i < e; ++i) {
    const uint32_t v = a[i];
    a[i] = run;
    run += v;
  }
}

__global__ void __launch_bounds__(RS_WARPS * 32)
    rs_scatter_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                      uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, int64_t n,
                      int shift, int64_t per_warp, const uint32_t* __restrict__ hist, int nwt) {
  __shared__ uint32_t off[RS_WARPS][256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t w = (int64_t)blockIdx.x * RS_WARPS + warp;
  for (int i = lane; i < 256; i += 32) off[warp][i] = hist[(int64_t)i * nwt + w];
  __syncwarp();
  const int64_t b = w * per_warp;
  int64_t e = b + per_warp;
  if (e > n) e = n;
  for (int64_t i0 = b; i0 < e; i0 += 32) {
    const int64_t i = i0 + lane;
    const bool ok = i < e;
    uint32_t key = 0, val = 0;
    if (ok) {
      key = keys_in[i];
      val = vals_in ? vals_in[i] : (uint32_t)i;
    }
    const uint32_t dig = ok ? ((key >> shift) & 255u) : (256u + lane);
    const unsigned peers = __match_any_sync(kFull, dig);
    uint32_t base = 0;
    if (ok) base = off[warp][dig];
    __syncwarp();
    if (ok) {
      const uint32_t pos = base + __popc(peers & ((1u << lane) - 1u));
      keys_out[pos] = key;
      vals_out[pos] = val;
      if (lane == __ffs(peers) - 1) off[warp][dig] = base + __popc(peers);
    }
    __syncwarp();
  }
}

// keys[a] = list number of CSR position a (old entries entering a re-finalise).
__global__ void csr_expand_kernel(const int64_t* __restrict__ offsets, int nlist, int64_t n,
                                  uint32_t* __restrict__ keys) {
  const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n) return;
  int lo = 0, hi = nlist;  // largest l with offsets[l] <= a
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (offsets[mid] <= a) lo = mid; else hi = mid;
  }
  keys[a] = (uint32_t)lo;
}

// offsets[l] = first sorted position whose list number is >= l.
__global__ void csr_offsets_kernel(const uint32_t* __restrict__ keys, int64_t n, int nlist,
                                   int64_t* __restrict__ offsets) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int64_t k1 = keys[p];
  const int64_t k0 = p > 0 ? (int64_t)keys[p - 1] : -1;
  for (int64_t l = k0 + 1; l <= k1; ++l) offsets[l] = p;
  if (p == n - 1)
    for (int64_t l = k1 + 1; l <= nlist; ++l) offsets[l] = n;
}

// Moves every vector to its CSR position p.  perm[p] = arrival index (old CSR entries first, then the
// staged ones); keys[p] = list number of position p.  With `permute` the code bytes are stored in the lane
// order of the fixed-point scan: byte i of the vector at position v of its list holds sub-quantizer
// i ^ (v mod M) (M = 8 / 16); old entries are moved from the order of their old position to the new one.
__global__ void csr_gather_kernel(const uint32_t* __restrict__ perm, const uint32_t* __restrict__ keys, int64_t n,
                                  int64_t n_old, int M, bool permute, const int64_t* __restrict__ old_offsets,
                                  const int64_t* __restrict__ new_offsets, const uint8_t* __restrict__ old_codes,
                                  const int64_t* __restrict__ old_ids, const float* __restrict__ old_s1,
                                  const uint8_t* __restrict__ st_codes, const int64_t* __restrict__ st_ids,
                                  const float* __restrict__ st_s1, uint8_t* __restrict__ codes,
                                  int64_t* __restrict__ ids, float* __restrict__ s1) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int64_t a = perm[p];
  const uint8_t* src;
  int r = 0;
  if (permute) {
    const int64_t L = keys[p];
    r = (int)((p - new_offsets[L]) & (M - 1));
    if (a < n_old) r ^= (int)((a - old_offsets[L]) & (M - 1));
  }
  if (a < n_old) {
    src = old_codes + a * M;
    ids[p] = old_ids[a];
    s1[p] = old_s1[a];
  } else {
    src = st_codes + (a - n_old) * M;
    ids[p] = st_ids[a - n_old];
    s1[p] = st_s1[a - n_old];
  }
  uint8_t* dst = codes + p * M;
  if (permute) {
    uint32_t w[4];
    for (int i = 0; i < M / 4; ++i) w[i] = reinterpret_cast<const uint32_t*>(src)[i];
    const uint32_t sel = 0x3210u ^ (0x1111u * (uint32_t)(r & 3));  // byte i <- byte i ^ (r & 3) of the same word
    for (int i = 0; i < M / 4; ++i) reinterpret_cast<uint32_t*>(dst)[i] = __byte_perm(w[i ^ (r >> 2)], 0u, sel);
  } else if ((M & 3) == 0) {
    for (int w = 0; w < M / 4; ++w)
      reinterpret_cast<uint32_t*>(dst)[w] = reinterpret_cast<const uint32_t*>(src)[w];
  } else {
    for (int b = 0; b < M; ++b) dst[b] = src[b];
  }
}

// Plain order of the stored codes of whole lists: block j copies list list_nos[j] (or list j) from the CSR
// arrays to dst + dst_offsets[j] * M, undoing the permutation of csr_gather_kernel.
__global__ void csr_unpermute_kernel(const uint8_t* __restrict__ codes, const int64_t* __restrict__ offsets,
                                     const int32_t* __restrict__ list_nos, const int64_t* __restrict__ dst_offsets,
                                     int M, uint8_t* __restrict__ dst) {
  const int64_t L = list_nos ? list_nos[blockIdx.x] : blockIdx.x;
  const int64_t b = offsets[L], len = offsets[L + 1] - b;
  uint8_t* out = dst + (dst_offsets ? dst_offsets[blockIdx.x] : b) * M;
  for (int64_t v = threadIdx.x; v < len; v += blockDim.x) {
    const int r = (int)(v & (M - 1));
    const uint32_t sel = 0x3210u ^ (0x1111u * (uint32_t)(r & 3));
    uint32_t w[4];
    for (int i = 0; i < M / 4; ++i) w[i] = reinterpret_cast<const uint32_t*>(codes + (b + v) * M)[i];
    for (int i = 0; i < M / 4; ++i) reinterpret_cast<uint32_t*>(out + v * M)[i] = __byte_perm(w[i ^ (r >> 2)], 0u, sel);
  }
}

__global__ void iota_ids_kernel(int64_t* ids, int64_t n, int64_t start) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) ids[i] = start + i;
}
}  // namespace

// Stable LSD radix sort of n 32-bit keys (values < 2^nbits) with their arrival indices as the values.
// keysA holds the input keys (overwritten); tmp must hold 3 * nb4 + hist bytes more (laid out as the
// caller of stable_sort_ws says).  On return *keys_sorted / *order point into the buffers.
size_t stable_sort_ws(int64_t n) {
  const size_t nb4 = align_up((size_t)n * sizeof(uint32_t), 256);
  int64_t grid = ceil_div(n, (int64_t)RS_WARPS * 32 * 64);
  const int64_t maxg = (int64_t)sm_count() * 4;
  if (grid > maxg) grid = maxg;
  if (grid < 1) grid = 1;
  return 4 * nb4 + align_up((size_t)256 * grid * RS_WARPS * sizeof(uint32_t), 256);
}

int stable_sort_by_key(char* t, int64_t n, int nbits, const uint32_t** keys_sorted, const uint32_t** order,
                       cudaStream_t s) {
  const size_t nb4 = align_up((size_t)n * sizeof(uint32_t), 256);
  const int passes = nbits <= 0 ? 1 : (nbits + 7) / 8;
  int64_t grid = ceil_div(n, (int64_t)RS_WARPS * 32 * 64);
  const int64_t maxg = (int64_t)sm_count() * 4;
  if (grid > maxg) grid = maxg;
  if (grid < 1) grid = 1;
  const int nwt = (int)grid * RS_WARPS;
  const int64_t per_warp = ceil_div(ceil_div(n, nwt), 32) * 32;
  uint32_t* kA = reinterpret_cast<uint32_t*>(t);
  uint32_t* vA = reinterpret_cast<uint32_t*>(t + nb4);
  uint32_t* kB = reinterpret_cast<uint32_t*>(t + 2 * nb4);
  uint32_t* vB = reinterpret_cast<uint32_t*>(t + 3 * nb4);
  uint32_t* hist = reinterpret_cast<uint32_t*>(t + 4 * nb4);
  const uint32_t* vin = nullptr;
  uint32_t *kin = kA, *kout = kB, *vout = vB, *vother = vA;
  for (int pass = 0; pass < passes; ++pass) {
    const int shift = 8 * pass;
    rs_hist_kernel<<<(unsigned)grid, RS_WARPS * 32, 0, s>>>(kin, n, shift, per_warp, hist, nwt);
    rs_scan_kernel<<<1, 1024, 0, s>>>(hist, (int64_t)256 * nwt);
    rs_scatter_kernel<<<(unsigned)grid, RS_WARPS * 32, 0, s>>>(kin, vin, kout, vout, n, shift, per_warp, hist, nwt);
    launch_counter() += 3;
    vin = vout;
    uint32_t* tk = kin; kin = kout; kout = tk;
    uint32_t* tv = vout; vout = vother; vother = tv;
  }
  if (cudaGetLastError() != cudaSuccess) return set_error(FS_ECUDA, "stable sort: launch failed");
  *keys_sorted = kin;
  *order = vin;
  return FS_OK;
}

int ivfpq_finalise(fs_ivfpq* ix, cudaStream_t s) {
  if (ix->n_staged == 0 && !ix->offsets_host.empty()) return FS_OK;
  const int64_t n = ix->n_csr + ix->n_staged;
  const int nlist = ix->nlist, M = ix->M;
  int rc;
  if (n >= (1LL << 32)) return set_error(FS_EUNSUPPORTED, "fs_ivfpq: more than 2^32-1 vectors");
  DevBuf noffsets, ncodes, nids, ns1;
  if ((rc = noffsets.ensure((size_t)(nlist + 1) * sizeof(int64_t), 0, s)) != FS_OK) return rc;
  if (n == 0) {
    FS_CUDA(cudaMemsetAsync(noffsets.p, 0, (size_t)(nlist + 1) * sizeof(int64_t), s));
  } else {
    // sort temporaries: keys/vals double-buffered
    DevBuf tmp;
    const size_t nb4 = align_up((size_t)n * sizeof(uint32_t), 256);
    int nbits = 0;
    while ((1LL << nbits) < nlist) ++nbits;
    const int passes = nbits == 0 ? 0 : (nbits + 7) / 8;
    int64_t grid = ceil_div(n, (int64_t)RS_WARPS * 32 * 64);
    const int64_t maxg = (int64_t)sm_count() * 4;
    if (grid > maxg) grid = maxg;
    if (grid < 1) grid = 1;
    const int nwt = (int)grid * RS_WARPS;
    const int64_t per_warp = ceil_div(ceil_div(n, nwt), 32) * 32;
    const size_t hist_b = align_up((size_t)256 * nwt * sizeof(uint32_t), 256);
    if ((rc = tmp.ensure(4 * nb4 + hist_b, 0, s)) != FS_OK) {
      noffsets.release();
      return rc;
    }
    char* t = tmp.as<char>();
    uint32_t* kA = reinterpret_cast<uint32_t*>(t);
    uint32_t* vA = reinterpret_cast<uint32_t*>(t + nb4);
    uint32_t* kB = reinterpret_cast<uint32_t*>(t + 2 * nb4);
    uint32_t* vB = reinterpret_cast<uint32_t*>(t + 3 * nb4);
    uint32_t* hist = reinterpret_cast<uint32_t*>(t + 4 * nb4);
    auto cleanup = [&]() {
      tmp.release();
      noffsets.release();
      ncodes.release();
      nids.release();
      ns1.release();
    };
    // keys in arrival order: old CSR entries (already grouped), then the staged ones
    if (ix->n_csr > 0) {
      csr_expand_kernel<<<(unsigned)ceil_div(ix->n_csr, 256), 256, 0, s>>>(
          ix->offsets.as<int64_t>(), nlist, ix->n_csr, kA);
      ++launch_counter();
    }
    if (ix->n_staged > 0)
      FS_CUDA(cudaMemcpyAsync(kA + ix->n_csr, ix->st_list.p, (size_t)ix->n_staged * sizeof(uint32_t),
                              cudaMemcpyDeviceToDevice, s));
    const uint32_t* vin = nullptr;
    uint32_t *kin = kA, *kout = kB, *vout = vB, *vother = vA;
    for (int pass = 0; pass < passes; ++pass) {
      const int shift = 8 * pass;
      rs_hist_kernel<<<(unsigned)grid, RS_WARPS * 32, 0, s>>>(kin, n, shift, per_warp, hist, nwt);
      rs_scan_kernel<<<1, 1024, 0, s>>>(hist, (int64_t)256 * nwt);
      rs_scatter_kernel<<<(unsigned)grid, RS_WARPS * 32, 0, s>>>(kin, vin, kout, vout, n, shift,
                                                                  per_warp, hist, nwt);
      launch_counter() += 3;
      vin = vout;
      uint32_t* tk = kin; kin = kout; kout = tk;
      uint32_t* tv = vout; vout = vother; vother = tv;
    }
    if (passes == 0) {  // nlist == 1: identity permutation
      rs_hist_kernel<<<(unsigned)grid, RS_WARPS * 32, 0, s>>>(kin, n, 0, per_warp, hist, nwt);
      rs_scan_kernel<<<1, 1024, 0, s>>>(hist, (int64_t)256 * nwt);
      rs_scatter_kernel<<<(unsigned)grid, RS_WARPS * 32, 0, s>>>(kin, nullptr, kout, vout, n, 0,
                                                                  per_warp, hist, nwt);
      launch_counter() += 3;
      vin = vout;
      kin = kout;
    }
    if (cudaGetLastError() != cudaSuccess) {
      cleanup();
      return set_error(FS_ECUDA, "fs_ivfpq finalise: sort launch failed");
    }
    if ((rc = ncodes.ensure((size_t)n * M, 0, s)) != FS_OK ||
        (rc = nids.ensure((size_t)n * sizeof(int64_t), 0, s)) != FS_OK ||
        (rc = ns1.ensure((size_t)n * sizeof(float), 0, s)) != FS_OK) {
      cleanup();
      return rc;
    }
    csr_offsets_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, s>>>(kin, n, nlist,
                                                                  noffsets.as<int64_t>());
    csr_gather_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, s>>>(
        vin, kin, n, ix->n_csr, M, ix->permuted(), ix->offsets.as<int64_t>(), noffsets.as<int64_t>(),
        ix->codes.as<uint8_t>(), ix->ids.as<int64_t>(), ix->s1.as<float>(), ix->st_codes.as<uint8_t>(),
        ix->st_ids.as<int64_t>(), ix->st_s1.as<float>(), ncodes.as<uint8_t>(), nids.as<int64_t>(), ns1.as<float>());
    launch_counter() += 2;
    cudaError_t e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) e = cudaGetLastError();
    tmp.release();
    if (e != cudaSuccess) {
      noffsets.release();
      ncodes.release();
      nids.release();
      ns1.release();
      return set_error(FS_ECUDA, "fs_ivfpq finalise failed: %s", cudaGetErrorString(e));
    }
  }
  ix->offsets.release();
  ix->codes.release();
  ix->ids.release();
  ix->s1.release();
  ix->offsets = noffsets;
  ix->codes = ncodes;
  ix->ids = nids;
  ix->s1 = ns1;
  ix->n_csr = n;
  ix->n_staged = 0;
  ix->st_list.release();
  ix->st_codes.release();
  ix->st_ids.release();
  ix->st_s1.release();
  ix->offsets_host.resize(nlist + 1);
  FS_CUDA(cudaMemcpyAsync(ix->offsets_host.data(), ix->offsets.p, (size_t)(nlist + 1) * sizeof(int64_t),
                          cudaMemcpyDeviceToHost, s));
  FS_CUDA(cudaStreamSynchronize(s));
  return FS_OK;
}

// ---------------------------------------------------------------------------
// D1: nearest centroid (k = 1 exact search), in chunks that bound the workspace.
// ---------------------------------------------------------------------------
int ivfpq_prepare_coarse(fs_ivfpq* ix, cudaStream_t s) {
  int rc = launch_row_norms(ix->coarse.as<float>(), ix->nlist, ix->d, ix->cnorm.as<float>(), s);
  if (rc != FS_OK) return rc;
  return flat_prepare_device(ix->coarse.as<float>(), ix->nlist, ix->d, ix->cprep.p, s);
}

int assign_nearest(const float* x, int64_t n, const float* cent, const float* cent_norm, int K,
                   int d, int64_t* assign, cudaStream_t s, const void* cent_prep) {
  if (n == 0) return FS_OK;
  FlatPrep view;
  if (cent_prep) view = flat_prep_view(cent_prep, K, d);
  const int64_t chunk = n < (1 << 20) ? n : (1 << 20);
  size_t need = flat_plan(chunk, K, d, 1).bytes;
  if (n % chunk != 0) {  // the smaller last chunk has its own plan
    const size_t tail = flat_plan(n % chunk, K, d, 1).bytes;
    if (tail > need) need = tail;
  }
  DevBuf ws, dist;
  int rc;
  if ((rc = ws.ensure(need, 0, s)) != FS_OK) return rc;
  if ((rc = dist.ensure((size_t)chunk * sizeof(float), 0, s)) != FS_OK) {
    ws.release();
    return rc;
  }
  for (int64_t b = 0; b < n && rc == FS_OK; b += chunk) {
    const int64_t m = (n - b) < chunk ? (n - b) : chunk;
    rc = flat_knn_device(x + b * d, m, cent, K, d, 1, cent_norm, dist.as<float>(), assign + b,
                         ws.p, s, cent_prep ? &view : nullptr);
  }
  cudaStreamSynchronize(s);
  ws.release();
  dist.release();
  return rc;
}

static int ivfpq_add_device(fs_ivfpq* ix, const float* xb, int64_t n, const int64_t* ids,
                            cudaStream_t s) {
  const int M = ix->M;
  const int64_t base = ix->n_staged;
  const int64_t first_id = ix->ntotal();
  int rc;
  if (ix->ntotal() + n >= (1LL << 32))
    return set_error(FS_EUNSUPPORTED, "fs_ivfpq_add: more than 2^32-1 vectors");
  if ((rc = ix->st_list.ensure((size_t)(base + n) * sizeof(uint32_t), (size_t)base * sizeof(uint32_t), s)) != FS_OK ||
      (rc = ix->st_codes.ensure((size_t)(base + n) * M, (size_t)base * M, s)) != FS_OK ||
      (rc = ix->st_ids.ensure((size_t)(base + n) * sizeof(int64_t), (size_t)base * sizeof(int64_t), s)) != FS_OK ||
      (rc = ix->st_s1.ensure((size_t)(base + n) * sizeof(float), (size_t)base * sizeof(float), s)) != FS_OK)
    return rc;
  DevBuf assign;
  if ((rc = assign.ensure((size_t)n * sizeof(int64_t), 0, s)) != FS_OK) return rc;
  rc = assign_nearest(xb, n, ix->coarse.as<float>(), ix->cnorm.as<float>(), ix->nlist, ix->d,
                      assign.as<int64_t>(), s, ix->cprep.p);
  if (rc == FS_OK)
    rc = launch_pq_encode(ix, xb, n, assign.as<int64_t>(), ix->st_codes.as<uint8_t>() + base * M,
                          ix->st_list.as<uint32_t>() + base, ix->st_s1.as<float>() + base, s);
  if (rc == FS_OK) {
    if (ids) {
      const cudaError_t e = cudaMemcpyAsync(ix->st_ids.as<int64_t>() + base, ids, (size_t)n * sizeof(int64_t),
                                            cudaMemcpyDeviceToDevice, s);
      if (e != cudaSuccess) rc = set_error(FS_ECUDA, "fs_ivfpq_add: copy of the ids failed: %s", cudaGetErrorString(e));
    } else {
      iota_ids_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, s>>>(ix->st_ids.as<int64_t>() + base, n,
                                                                first_id);
      ++launch_counter();
    }
  }
  cudaError_t e = cudaStreamSynchronize(s);
  assign.release();
  if (rc != FS_OK) return rc;
  if (e != cudaSuccess) return set_error(FS_ECUDA, "fs_ivfpq_add: %s", cudaGetErrorString(e));
  ix->n_staged += n;
  return FS_OK;
}

}  // namespace fs

// ---------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------
extern "C" {

int fs_ivfpq_create(fs_ivfpq** out, int d, int nlist, int M) {
  if (!out) return fs::set_error(FS_EINVAL, "fs_ivfpq_create: NULL out");
  *out = nullptr;
  if (d < 1 || nlist < 1 || M < 1) return fs::set_error(FS_EINVAL, "fs_ivfpq_create: d, nlist, M must be >= 1");
  if (d % M != 0) return fs::set_error(FS_EINVAL, "fs_ivfpq_create: d %% M != 0 (P:L86)");
  if (M > 64) return fs::set_error(FS_EUNSUPPORTED, "fs_ivfpq_create: M > 64 (P:L295)");
  if (d > 2048) return fs::set_error(FS_EUNSUPPORTED, "fs_ivfpq_create: d > 2048");
  if (d / M > 128) return fs::set_error(FS_EUNSUPPORTED, "fs_ivfpq_create: d / M > 128");
  fs_ivfpq* ix = new (std::nothrow) fs_ivfpq();
  if (!ix) return fs::set_error(FS_ENOMEM, "fs_ivfpq_create: out of host memory");
  ix->d = d;
  ix->nlist = nlist;
  ix->M = M;
  ix->dsub = d / M;
  int rc;
  if ((rc = ix->coarse.ensure((size_t)nlist * d * sizeof(float), 0, nullptr)) != FS_OK ||
      (rc = ix->cnorm.ensure((size_t)nlist * sizeof(float), 0, nullptr)) != FS_OK ||
      (rc = ix->cprep.ensure(fs::flat_prep_bytes(nlist, d), 0, nullptr)) != FS_OK ||
      (rc = ix->pq.ensure((size_t)256 * d * sizeof(float), 0, nullptr)) != FS_OK ||
      (rc = ix->scanned.ensure(sizeof(unsigned long long), 0, nullptr)) != FS_OK) {
    fs_ivfpq_destroy(ix);
    return rc;
  }
  cudaMemset(ix->scanned.p, 0, sizeof(unsigned long long));
  for (cudaEvent_t& e : ix->ev)
    if (cudaEventCreate(&e) != cudaSuccess) {
      fs_ivfpq_destroy(ix);
      return fs::set_error(FS_ECUDA, "fs_ivfpq_create: cudaEventCreate failed");
    }
  *out = ix;
  return FS_OK;
}

int fs_ivfpq_destroy(fs_ivfpq* ix) {
  if (!ix) return FS_OK;
  cudaDeviceSynchronize();
  fs::DevBuf* bufs[] = {&ix->coarse, &ix->cnorm, &ix->cprep, &ix->pq, &ix->offsets, &ix->codes, &ix->ids,
                        &ix->st_list, &ix->st_codes, &ix->st_ids, &ix->scanned, &ix->s1, &ix->st_s1};
  for (fs::DevBuf* b : bufs) b->release();
  for (cudaEvent_t e : ix->ev)
    if (e) cudaEventDestroy(e);
  delete ix;
  return FS_OK;
}

int fs_ivfpq_set_quantizers(fs_ivfpq* ix, const float* coarse, const float* pq, fs_stream stream) {
  if (!ix || !coarse || !pq) return fs::set_error(FS_EINVAL, "fs_ivfpq_set_quantizers: NULL pointer");
  if (ix->ntotal() > 0)
    return fs::set_error(FS_ESTATE, "fs_ivfpq_set_quantizers: index already holds vectors");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  FS_CUDA(cudaMemcpyAsync(ix->coarse.p, coarse, (size_t)ix->nlist * ix->d * sizeof(float),
                          cudaMemcpyDeviceToDevice, s));
  FS_CUDA(cudaMemcpyAsync(ix->pq.p, pq, (size_t)256 * ix->d * sizeof(float), cudaMemcpyDeviceToDevice, s));
  int rc = fs::ivfpq_prepare_coarse(ix, s);
  if (rc != FS_OK) return rc;
  ix->have_quantizers = true;
  return FS_OK;
}

int fs_ivfpq_get_quantizers(const fs_ivfpq* ix, float* coarse, float* pq, fs_stream stream) {
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_get_quantizers: NULL index");
  if (!ix->have_quantizers) return fs::set_error(FS_ESTATE, "fs_ivfpq_get_quantizers: no quantizers set or trained");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (coarse)
    FS_CUDA(cudaMemcpyAsync(coarse, ix->coarse.p, (size_t)ix->nlist * ix->d * sizeof(float),
                            cudaMemcpyDeviceToDevice, s));
  if (pq)
    FS_CUDA(cudaMemcpyAsync(pq, ix->pq.p, (size_t)256 * ix->d * sizeof(float), cudaMemcpyDeviceToDevice, s));
  return FS_OK;
}

int fs_ivfpq_add(fs_ivfpq* ix, const float* xb, int64_t n, const int64_t* ids, fs_stream stream) {
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_add: NULL index");
  if (n < 0 || (n > 0 && !xb)) return fs::set_error(FS_EINVAL, "fs_ivfpq_add: bad arguments");
  if (!ix->have_quantizers) return fs::set_error(FS_ESTATE, "fs_ivfpq_add: no quantizers set or trained");
  if (n == 0) return FS_OK;
  return fs::ivfpq_add_device(ix, xb, n, ids, static_cast<cudaStream_t>(stream));
}

int64_t fs_ivfpq_ntotal(const fs_ivfpq* ix) { return ix ? ix->ntotal() : 0; }

int64_t fs_ivfpq_last_scanned_codes(const fs_ivfpq* ix) {
  if (!ix) return 0;
  unsigned long long v = 0;
  cudaDeviceSynchronize();
  if (cudaMemcpy(&v, ix->scanned.p, sizeof v, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
  return (int64_t)v;
}

int fs_ivfpq_last_stage_ms(const fs_ivfpq* ix, float* ms) {
  if (!ix || !ms) return fs::set_error(FS_EINVAL, "fs_ivfpq_last_stage_ms: NULL pointer");
  if (!ix->ev_valid) return fs::set_error(FS_ESTATE, "fs_ivfpq_last_stage_ms: no search has run");
  FS_CUDA(cudaEventSynchronize(ix->ev[3]));
  for (int i = 0; i < 3; ++i) FS_CUDA(cudaEventElapsedTime(ms + i, ix->ev[i], ix->ev[i + 1]));
  return FS_OK;
}

int fs_ivfpq_list(const fs_ivfpq* cix, int list_no, const uint8_t** codes, const int64_t** ids,
                  int64_t* len) {
  fs_ivfpq* ix = const_cast<fs_ivfpq*>(cix);
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_list: NULL index");
  if (list_no < 0 || list_no >= ix->nlist) return fs::set_error(FS_EINVAL, "fs_ivfpq_list: list_no out of range");
  int rc = fs::ivfpq_finalise(ix, nullptr);
  if (rc != FS_OK) return rc;
  const int64_t b = ix->offsets_host[list_no], e = ix->offsets_host[list_no + 1];
  if (codes) *codes = ix->codes.as<uint8_t>() + b * ix->M;
  if (ids) *ids = ix->ids.as<int64_t>() + b;
  if (len) *len = e - b;
  return FS_OK;
}

int fs_ivfpq_export(const fs_ivfpq* cix, int64_t* offsets, uint8_t* codes, int64_t* ids,
                    fs_stream stream) {
  fs_ivfpq* ix = const_cast<fs_ivfpq*>(cix);
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_export: NULL index");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = fs::ivfpq_finalise(ix, s);
  if (rc != FS_OK) return rc;
  if (offsets)
    FS_CUDA(cudaMemcpyAsync(offsets, ix->offsets.p, (size_t)(ix->nlist + 1) * sizeof(int64_t),
                            cudaMemcpyDeviceToDevice, s));
  if (codes && ix->n_csr > 0) {
    if (ix->permuted()) {
      fs::csr_unpermute_kernel<<<(unsigned)ix->nlist, 128, 0, s>>>(ix->codes.as<uint8_t>(), ix->offsets.as<int64_t>(),
                                                                 nullptr, nullptr, ix->M, codes);
      FS_LAUNCHED();
    } else {
      FS_CUDA(cudaMemcpyAsync(codes, ix->codes.p, (size_t)ix->n_csr * ix->M, cudaMemcpyDeviceToDevice, s));
    }
  }
  if (ids && ix->n_csr > 0)
    FS_CUDA(cudaMemcpyAsync(ids, ix->ids.p, (size_t)ix->n_csr * sizeof(int64_t), cudaMemcpyDeviceToDevice, s));
  return FS_OK;
}

int fs_ivfpq_export_lists(const fs_ivfpq* cix, const int32_t* list_nos, int64_t n_lists, int64_t* offsets_host,
                          uint8_t* codes, int64_t* ids, fs_stream stream) {
  fs_ivfpq* ix = const_cast<fs_ivfpq*>(cix);
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_export_lists: NULL index");
  if (n_lists < 0 || !offsets_host || (n_lists > 0 && !list_nos))
    return fs::set_error(FS_EINVAL, "fs_ivfpq_export_lists: bad arguments");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = fs::ivfpq_finalise(ix, s);
  if (rc != FS_OK) return rc;
  int64_t total = 0;
  for (int64_t j = 0; j < n_lists; ++j) {
    const int L = list_nos[j];
    if (L < 0 || L >= ix->nlist) return fs::set_error(FS_EINVAL, "fs_ivfpq_export_lists: list %d out of range", L);
    offsets_host[j] = total;
    total += ix->offsets_host[L + 1] - ix->offsets_host[L];
  }
  offsets_host[n_lists] = total;
  if (!codes && !ids) return FS_OK;
  if (codes && ix->permuted() && total > 0) {
    // the lists' codes in plain byte order: one block per list, list numbers and output offsets uploaded
    int32_t* d_ln = nullptr;
    int64_t* d_off = nullptr;
    FS_CUDA(cudaMallocAsync(&d_ln, (size_t)n_lists * sizeof(int32_t), s));
    FS_CUDA(cudaMallocAsync(&d_off, (size_t)(n_lists + 1) * sizeof(int64_t), s));
    FS_CUDA(cudaMemcpyAsync(d_ln, list_nos, (size_t)n_lists * sizeof(int32_t), cudaMemcpyHostToDevice, s));
    FS_CUDA(cudaMemcpyAsync(d_off, offsets_host, (size_t)(n_lists + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, s));
    fs::csr_unpermute_kernel<<<(unsigned)n_lists, 128, 0, s>>>(ix->codes.as<uint8_t>(), ix->offsets.as<int64_t>(), d_ln,
                                                              d_off, ix->M, codes);
    FS_LAUNCHED();
    FS_CUDA(cudaFreeAsync(d_ln, s));
    FS_CUDA(cudaFreeAsync(d_off, s));
    FS_CUDA(cudaStreamSynchronize(s));  // list_nos / offsets_host are the caller's: copied before returning
    codes = nullptr;
  }
  // one copy per run of consecutive list numbers (their CSR ranges are adjacent)
  for (int64_t j = 0; j < n_lists;) {
    int64_t e = j + 1;
    while (e < n_lists && list_nos[e] == list_nos[e - 1] + 1) ++e;
    const int64_t src = ix->offsets_host[list_nos[j]], len = offsets_host[e] - offsets_host[j];
    if (len > 0) {
      if (codes)
        FS_CUDA(cudaMemcpyAsync(codes + offsets_host[j] * ix->M, ix->codes.as<uint8_t>() + src * ix->M,
                                (size_t)len * ix->M, cudaMemcpyDeviceToDevice, s));
      if (ids)
        FS_CUDA(cudaMemcpyAsync(ids + offsets_host[j], ix->ids.as<int64_t>() + src, (size_t)len * sizeof(int64_t),
                                cudaMemcpyDeviceToDevice, s));
    }
    j = e;
  }
  return FS_OK;
}

size_t fs_ivfpq_search_ws_bytes(const fs_ivfpq* ix, int64_t nq, int nprobe, int k) {
  if (!ix || nq < 0 || nprobe < 1 || nprobe > ix->nlist || nprobe > 1024 || k < 1 || k > FS_MAX_K) return 0;
  return fs::ivfpq_search_ws(ix, nq, nprobe, k);
}

int fs_ivfpq_search(fs_ivfpq* ix, const float* xq, int64_t nq, int nprobe, int k, float* out_dist,
                    int64_t* out_ids, int32_t* out_probed, void* ws, size_t ws_bytes,
                    fs_stream stream) {
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_search: NULL index");
  if (nq < 0 || (nq > 0 && (!xq || !out_dist || !out_ids)))
    return fs::set_error(FS_EINVAL, "fs_ivfpq_search: bad arguments");
  if (k < 1 || nprobe < 1) return fs::set_error(FS_EINVAL, "fs_ivfpq_search: k and nprobe must be >= 1");
  if (k > FS_MAX_K) return fs::set_error(FS_EUNSUPPORTED, "fs_ivfpq_search: k = %d > %d", k, FS_MAX_K);
  if (nprobe > ix->nlist || nprobe > 1024)
    return fs::set_error(FS_EINVAL, "fs_ivfpq_search: nprobe = %d > min(nlist, 1024)", nprobe);
  if (!ix->have_quantizers) return fs::set_error(FS_ESTATE, "fs_ivfpq_search: no quantizers set or trained");
  if (nq == 0) return FS_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = fs::ivfpq_finalise(ix, s);
  if (rc != FS_OK) return rc;
  fs::TempWs t;
  rc = t.acquire(ws, ws_bytes, fs::ivfpq_search_ws(ix, nq, nprobe, k), s);
  if (rc != FS_OK) return rc;
  return fs::ivfpq_search_device(ix, xq, nq, nprobe, k, out_dist, out_ids, out_probed, t.ptr, s);
}

int fs_ivfpq_knn_graph(fs_ivfpq* ix, const float* x, int64_t n, int nprobe, int k, int64_t batch,
                       float* out_dist, int64_t* out_ids, int32_t* out_probed, fs_stream stream) {
  if (!ix) return fs::set_error(FS_EINVAL, "fs_ivfpq_knn_graph: NULL index");
  if (n < 0 || batch < 0 || (n > 0 && (!x || !out_dist || !out_ids)))
    return fs::set_error(FS_EINVAL, "fs_ivfpq_knn_graph: bad arguments");
  if (k < 1 || k > FS_MAX_K) return fs::set_error(FS_EINVAL, "fs_ivfpq_knn_graph: k must be in 1..%d", FS_MAX_K);
  if (nprobe < 1 || nprobe > ix->nlist || nprobe > 1024)
    return fs::set_error(FS_EINVAL, "fs_ivfpq_knn_graph: nprobe = %d outside 1..min(nlist, 1024)", nprobe);
  if (!ix->have_quantizers) return fs::set_error(FS_ESTATE, "fs_ivfpq_knn_graph: no quantizers set or trained");
  if (n == 0) return FS_OK;
  if (batch == 0) batch = 65536;
  if (batch > n) batch = n;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = fs::ivfpq_finalise(ix, s);
  if (rc != FS_OK) return rc;
  // one workspace for every batch (the tail batch needs no more than a full one)
  fs::TempWs t;
  size_t need = fs::ivfpq_search_ws(ix, batch, nprobe, k);
  const int64_t tail = n % batch;
  if (tail) {
    const size_t nt = fs::ivfpq_search_ws(ix, tail, nprobe, k);
    need = nt > need ? nt : need;
  }
  if ((rc = t.acquire(nullptr, 0, need, s)) != FS_OK) return rc;
  for (int64_t b = 0; b < n; b += batch) {
    const int64_t nq = n - b < batch ? n - b : batch;
    rc = fs::ivfpq_search_device(ix, x + b * ix->d, nq, nprobe, k, out_dist + b * k, out_ids + b * k,
                                 out_probed ? out_probed + b * nprobe : nullptr, t.ptr, s);
    if (rc != FS_OK) return rc;
  }
  return FS_OK;
}

int fs_ivfpq_search_host(fs_ivfpq* ix, const float* xq_host, int64_t nq, int nprobe, int k,
                         float* out_dist_host, int64_t* out_ids_host) {
  if (!ix || nq < 0 || (nq > 0 && (!xq_host || !out_dist_host || !out_ids_host)))
    return fs::set_error(FS_EINVAL, "fs_ivfpq_search_host: bad arguments");
  if (nq == 0) return FS_OK;
  if (k < 1 || k > FS_MAX_K) return fs::set_error(FS_EINVAL, "fs_ivfpq_search_host: bad k");
  float *dq = nullptr, *dd = nullptr;
  int64_t* di = nullptr;
  cudaStream_t s = nullptr;
  const size_t qb = (size_t)nq * ix->d * sizeof(float), on = (size_t)nq * k;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) {
    if (e == cudaSuccess) e = r;
    return e == cudaSuccess;
  };
  int rc = FS_OK;
  ok(cudaMalloc(&dq, qb)) && ok(cudaMalloc(&dd, on * sizeof(float))) &&
      ok(cudaMalloc(&di, on * sizeof(int64_t))) &&
      ok(cudaMemcpyAsync(dq, xq_host, qb, cudaMemcpyHostToDevice, s));
  if (e == cudaSuccess) {
    rc = fs_ivfpq_search(ix, dq, nq, nprobe, k, dd, di, nullptr, nullptr, 0, s);
    if (rc == FS_OK) {
      ok(cudaMemcpyAsync(out_dist_host, dd, on * sizeof(float), cudaMemcpyDeviceToHost, s)) &&
          ok(cudaMemcpyAsync(out_ids_host, di, on * sizeof(int64_t), cudaMemcpyDeviceToHost, s));
    }
  }
  ok(cudaStreamSynchronize(s));
  cudaFree(dq);
  cudaFree(dd);
  cudaFree(di);
  if (rc == FS_OK && e != cudaSuccess)
    rc = fs::set_error(FS_ECUDA, "fs_ivfpq_search_host: %s", cudaGetErrorString(e));
  return rc;
}

}  // extern "C"
