// ivfpq_scan.cuh -- arguments of the list-scan kernels (ivfpq_search.cu: one CTA per
// (query, group of lists); ivfpq_scan.cu: persistent CTAs with a resident codebook and
// a bank-conflict-free table layout).
#pragma once

#include <cstdint>

#include "common.cuh"

namespace fs {

struct ScanArgs {
  const float* xq;
  const float* coarse;
  const float* pq;
  const float* pq_t;         // pq regrouped for vector loads (ivfpq_search.cu), or NULL
  const float* pq_r;         // pq regrouped for the rotated fixed-point kernel, or NULL
  const float* bmax;         // [M] max_c ||B[m][c]||, or NULL
  const float* term1;        // [nlist][M * 256] Eq. 11 term 1 in lane order, or NULL
  const int64_t* probe_ids;  // [nq][nprobe], ascending coarse distance
  const int64_t* offsets;    // [nlist+1]
  const uint8_t* codes;      // [ntotal][M]
  uint64_t* Wg;              // [nq][ngroups][K] partial queues (keys: distance, CSR position)
  unsigned long long* scanned;
  int32_t* out_probed;       // [nq][nprobe] or NULL
  int d, M, dsub, nprobe, G, ngroups, k;
  unsigned int* work;        // zeroed counter for the kernels that hand items out dynamically
  bool len32;                // every list is shorter than 2^31 vectors
};

// rotate the MW-word little-endian value w right by r bytes (r < 4 MW, per-lane constant)
template <int MW>
__device__ __forceinline__ void rotate_bytes(uint32_t (&w)[MW], int r) {
  if (MW > 1) {
#pragma unroll
    for (int bit = MW / 2; bit >= 1; bit >>= 1) {  // word rotation by (r >> 2), one bit at a time
      const bool on = ((r >> 2) & bit) != 0;
      uint32_t t[MW];
#pragma unroll
      for (int i = 0; i < MW; ++i) t[i] = on ? w[(i + bit) % MW] : w[i];
#pragma unroll
      for (int i = 0; i < MW; ++i) w[i] = t[i];
    }
  }
  const int sh = (r & 3) * 8;
  uint32_t t[MW];
#pragma unroll
  for (int i = 0; i < MW; ++i) t[i] = __funnelshift_r(w[i], w[(i + 1) % MW], sh);
#pragma unroll
  for (int i = 0; i < MW; ++i) w[i] = t[i];
}

// out byte i = in byte (i ^ r) of the MW-word little-endian value w (r < 4 MW, per-lane constant):
// the fixed-point kernels let lane l add sub-quantizer (s ^ l) mod M at step s (any order gives the
// same integer sum), so that step s reads bank l ^ s -- 32 different banks -- and the address is one
// XOR away from a per-lane constant.
template <int MW>
__device__ __forceinline__ void xor_permute_bytes(uint32_t (&w)[MW], int r) {
  const uint32_t sel = 0x3210u ^ (0x1111u * (uint32_t)(r & 3));  // nibble i -> i ^ (r & 3)
#pragma unroll
  for (int i = 0; i < MW; ++i) w[i] = __byte_perm(w[i], 0u, sel);
#pragma unroll
  for (int bit = 1; bit < MW; bit <<= 1) {
    const bool on = ((r >> 2) & bit) != 0;
    uint32_t t[MW];
#pragma unroll
    for (int i = 0; i < MW; ++i) t[i] = on ? w[i ^ bit] : w[i];
#pragma unroll
    for (int i = 0; i < MW; ++i) w[i] = t[i];
  }
}

// Packed fp32 pairs (sm_100 FADD2 / FFMA2): two lanes of a 64-bit register per instruction
__device__ __forceinline__ uint64_t f2_pack(float a, float b) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
  return r;
}
__device__ __forceinline__ uint64_t f2_sub(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ float f2_hsum(uint64_t v) {
  float a, b;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
  return a + b;
}

// One code = MW words.  Streaming loads (evict-first): the codes pass through L1 once, the
// codebook that every table build re-reads should stay there.
template <int MW>
__device__ __forceinline__ void load_code(const uint8_t* p, uint32_t (&w)[MW]) {
  if (MW == 2) {
    const uint2 t = __ldcs(reinterpret_cast<const uint2*>(p));
    w[0] = t.x;
    w[1] = t.y;
  } else {
#pragma unroll
    for (int i = 0; i < MW / 4; ++i) {
      const uint4 t = __ldcs(reinterpret_cast<const uint4*>(p) + i);
      w[4 * i] = t.x;
      w[4 * i + 1] = t.y;
      w[4 * i + 2] = t.z;
      w[4 * i + 3] = t.w;
    }
  }
}

// Persistent scan: M in {8, 16, 32}, queue class K <= 256, codebook + tables within 200 KB.
bool scan2_supported(int d, int M, int k);
int scan2_queues_per_item();  // partial queues it writes per (query, list group): Wg is [nq][ngroups][that][K]
int launch_scan2(const ScanArgs& a, int64_t nq, int k, unsigned int* work, cudaStream_t s);

}  // namespace fs
