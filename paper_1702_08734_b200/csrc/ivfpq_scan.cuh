// ivfpq_scan.cuh -- arguments and small helpers of the list-scan kernels (ivfpq_search.cu).
#pragma once

#include <cstdint>

#include "common.cuh"

namespace fs {

struct ScanArgs {
  const float* xq;
  const float* coarse;
  const float* pq;
  const int64_t* probe_ids;  // [nq][nprobe], ascending coarse distance
  const float* cdist;        // [nq][nprobe] C1's distances (Eq. 11 term 2)
  bool cd_partial;           // cdist lacks ||x||^2 (C1 through the distance matrix)
  const int64_t* offsets;    // [nlist+1]
  const uint8_t* codes;      // [ntotal][M] (M = 8 / 16: stored in the scan's lane order, ivfpq.cuh)
  const float* s1;           // [ntotal] Eq. 11 term 1 per stored vector
  uint64_t* Wg;              // [nq][ngroups][K] partial queues (keys: distance, CSR position)
  unsigned long long* scanned;
  int32_t* out_probed;       // [nq][nprobe] or NULL
  int d, M, dsub, nprobe, G, ngroups, k;
};

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

}  // namespace fs
