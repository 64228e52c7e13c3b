// flat.cuh -- internal interface of the exact-search engine (flat.cu), used by
// the public fs_flat_l2_knn and by the IVFPQ coarse quantizer / add path.
#pragma once

#include "common.cuh"
#include "select.cuh"

namespace fs {

struct FlatPlan {
  int kclass;    // queue class: K = 32 << kclass
  int K;
  int S;         // database splits (partial queues per query)
  int64_t chunk; // database vectors per split
  size_t off_ynorm, off_xnorm, off_W, bytes;  // workspace layout
};

FlatPlan flat_plan(int64_t nq, int64_t nb, int d, int k);

// ||row||^2 for n rows of x [n][d] (B1).
int launch_row_norms(const float* x, int64_t n, int d, float* out, cudaStream_t s);

// The database side of B1 done once (fs_flat_prepare; the ||y_j||^2 do not depend on the queries):
// views into the caller's prepared block.  Layout (flat_tc.cu): 256-byte header (word 0: some lo of the database
// is non-zero) | ||y||^2 with the tile padding of the tensor-core engine | tensor-core engine: the lo plane.
struct FlatPrep {
  const float* ynorm;        // [nb] (+ padding)
  const unsigned int* flag;  // tensor-core engine: the database's lo flag; NULL on the FFMA engine
  const float* blo;          // tensor-core engine: lo plane [nb][d] (zeros where x is a TF32 number)
};
size_t flat_prep_bytes(int64_t nb, int d);
int flat_prepare_device(const float* xb, int64_t nb, int d, void* prep, cudaStream_t s);
FlatPrep flat_prep_view(const void* prep, int64_t nb, int d);

// Exact k-NN on device buffers.  ynorm_opt: precomputed ||y||^2 [nb] or NULL (FFMA engine); prep: the
// prepared database or NULL (both engines).  ws must hold flat_plan(...).bytes.  nq > 0, nb > 0.
int flat_knn_device(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k,
                    const float* ynorm_opt, float* out_dist, int64_t* out_ids, void* ws,
                    cudaStream_t s, const FlatPrep* prep = nullptr);

// Tensor-core engine (flat_tc.cu): tcgen05 / TMEM / TMA, 3xTF32 split operands.
struct FlatTcPlan {
  int kclass, K, S, qtiles, qgroups, grid, KB, nstage, cap;
  int64_t chunk, chunk0;
  size_t smem;
  size_t off_ynorm, off_xnorm, off_flag, off_gbound, off_hbound, off_hclaim, off_W, off_cbuf, off_qhi, off_qlo, off_bhi, off_blo, bytes;
  // sampled bound (k >= 2, large databases): a strided sample of ns rows is searched first for the c-th distance
  int64_t ns, sstride;
  int c;
  size_t off_fail, off_failq, off_qfhi, off_qflo, off_sub;  // fail list, gathered failed queries, the sample pass's own plan
};
bool flat_tc_supported(int d);  // d % 4 == 0, 32 <= d <= 128, not disabled by FS_FLAT_ENGINE=ffma
FlatTcPlan flat_tc_plan(int64_t nq, int64_t nb, int d, int k);
// dout != NULL: distance-matrix mode -- no selection, dout[q * dld + j] = ||y_j||^2 - 2 <x_q, y_j>
// (dld % 4 == 0, dout 16-byte aligned); k, out_dist and out_ids are ignored, the workspace is that of k = 1.
int flat_knn_tc_device(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k, float* out_dist,
                       int64_t* out_ids, void* ws, cudaStream_t s, float* dout = nullptr, int64_t dld = 0,
                       const FlatPrep* prep = nullptr);

// B4: S partial queues per query -> k results (+||x||^2 if xnorm != NULL).
// Optional extras of the sampled-bound scheme of the tensor-core engine (flat_tc.cu):
struct FinishExtra {
  unsigned int* bound_out = nullptr;       // != NULL: no results; bound_out[q] = order image of the k-th smallest d'
  unsigned int* fail_cnt = nullptr;        // != NULL: queries whose queues hold fewer than `need` keys are appended
  int* fail_q = nullptr;                   //          to fail_q (the sampled bound was too tight for them)
  int need = 0;
  const unsigned int* nq_dev = nullptr;    // != NULL: number of rows, on the device (<= nq)
  const int* qmap = nullptr;               // != NULL: row i of Wg is query qmap[i] (xnorm and outputs are indexed by it)
  bool packed = false;                     // every queue holds its keys first, sentinels behind them: reading stops there
};
int launch_flat_finish(const uint64_t* Wg, int64_t nq, int S, int k, const float* xnorm,
                       float* out_dist, int64_t* out_ids, cudaStream_t s, const FinishExtra* extra = nullptr);

// Positions -> ids: ids_io[q][i] holds a position into table (or < 0); it becomes table[position], and
// entries of a query with bitwise-equal distance are put in ascending id order.
int launch_resolve_ids(float* dist, int64_t* ids_io, const int64_t* table, int64_t nq, int k, cudaStream_t s,
                       int64_t table_stride = 0);
// keys of the G partial lists of every query for launch_flat_finish: Wg [nq][G][K]
int launch_merge_pack(const float* dist, const int64_t* ids, int64_t nq, int G, int k, int K, uint64_t* Wg, cudaStream_t s);

}  // namespace fs
