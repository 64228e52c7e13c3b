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
  const int64_t* probe_ids;  // [nq][nprobe], ascending coarse distance
  const int64_t* offsets;    // [nlist+1]
  const uint8_t* codes;      // [ntotal][M]
  uint64_t* Wg;              // [nq][ngroups][K] partial queues (keys: distance, CSR position)
  unsigned long long* scanned;
  int32_t* out_probed;       // [nq][nprobe] or NULL
  int d, M, dsub, nprobe, G, ngroups, k;
};

// Persistent scan: M in {8, 16, 32}, queue class K <= 256, codebook + tables within 200 KB.
bool scan2_supported(int d, int M, int k);
int launch_scan2(const ScanArgs& a, int64_t nq, int k, unsigned int* work, cudaStream_t s);

}  // namespace fs
