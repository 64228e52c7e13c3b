/* fs.h -- C ABI of the B200-native hot path of arXiv 1702.08734
 * ("Billion-scale similarity search with GPUs"): per-query k-selection fused
 * with distance computation.
 *
 * Citations "P:L<n>" are line numbers of the paper text.
 *
 * General conventions (the paper is silent on all of them):
 *  - Every data pointer is a DEVICE pointer unless its comment says "host".
 *    The caller owns all inputs, outputs and workspaces; the library owns only
 *    the opaque fs_ivfpq object and the inverted lists inside it.
 *  - Work is enqueued on the given stream (a cudaStream_t cast to void*; NULL is
 *    the legacy default stream); outputs are valid once that stream is
 *    synchronised.  The *_host entry points are the exception: they take HOST
 *    pointers, copy in, run, copy out and synchronise before returning.
 *  - Every function returns FS_OK or an error code; nothing throws or aborts
 *    across the ABI.  Arguments are validated before any launch;
 *    fs_last_error() gives a thread-local detail string for the last failure.
 *  - Results are ascending by distance/value; ties by lower index/id.  When
 *    fewer than k candidates exist the tail is (+INF, -1) (the +inf sentinel
 *    convention of P:L220).  Distances are SQUARED L2 (D is squared, P:L52;
 *    Eq. 7/10).
 *  - Workspaces: if ws == NULL the library allocates and frees a stream-ordered
 *    temporary itself; otherwise ws must hold at least the matching *_ws_bytes.
 *  - Devices and threads: every call works on the CURRENT device of the calling thread (cudaSetDevice);
 *    pointers, streams and fs_ivfpq objects belong to the device they were created on.  The device entry
 *    points (fs_kselect, fs_flat_l2_knn, fs_merge_topk, fs_kmeans, fs_ivfpq_search) may run concurrently
 *    from several host threads on distinct streams with distinct workspaces; calls on one fs_ivfpq object
 *    are serialised by the caller (add / train / search change or read its lists and event records); the
 *    *_host entry points hold a process-wide lock (one staging arena).
 */
#ifndef FS_H_
#define FS_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define FS_API __attribute__((visibility("default")))
#else
#define FS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fs_ivfpq fs_ivfpq; /* opaque, library-owned */
typedef void* fs_stream;          /* cudaStream_t */

enum {
  FS_OK = 0,
  FS_EINVAL = 1,       /* bad argument (NULL pointer, negative size, ld < n, d % M != 0 ...) */
  FS_EUNSUPPORTED = 2, /* outside the supported range (k > 1024, d too large ...) */
  FS_ENOMEM = 3,       /* allocation failed or ws_bytes too small */
  FS_ECUDA = 4,        /* a CUDA call failed; fs_last_error() has the CUDA string */
  FS_ESTATE = 5        /* index not in the state the call needs (no quantizers ...) */
};

#define FS_MAX_K 1024 /* "it supports k <= 1024" */

FS_API const char* fs_last_error(void);
/* Library version and the SM architecture it was compiled for ("sm_100a"). */
FS_API const char* fs_version(void);
/* Which engine fs_flat_l2_knn's contraction runs on in this build:
 * "ffma-fp32" (CUDA cores) or "tcgen05-3xtf32" (tensor cores, split operands). */
FS_API const char* fs_flat_engine(void);
/* Number of kernel launches this thread's calls have enqueued since the last
 * fs_reset_launch_count(); used by bench.py to fill "gpu_launches". */
FS_API int64_t fs_launch_count(void);
FS_API void fs_reset_launch_count(void);

/* --------------------------------------------------------------------------
 * k-selection (WarpSelect, section 4.2; k = 1 is a
 * reduction; long rows by decomposition).
 * For each of n_rows arrays [a_i], i = 0..n-1, the k lowest values ascending
 * with their indices; ties broken by lower index, -0 == +0, NaN orders after
 * +INF (a NaN is returned only when fewer than k other values exist; rows with many
 * NaNs are answered exactly but by slower passes).  Bit-exact: out_val holds the
 * original fp32 bits.
 *   rows     device fp32 [n_rows][ld], row-major, ld >= n
 *   out_val  device fp32 [n_rows][k];  out_idx device int32 [n_rows][k]
 *   1 <= k <= FS_MAX_K; n < 2^31; k > n pads with (+INF, -1).
 * n_rows == 0 or n == 0 is valid (n == 0 writes only padding).
 * ------------------------------------------------------------------------ */
FS_API int fs_kselect(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
               int32_t* out_idx, void* ws, size_t ws_bytes, fs_stream stream);
/* The "other comparator" of P:L48 ("other comparators are sometimes desired"): the k HIGHEST values of
 * every array, descending, ties broken by LOWER index, -0 == +0, NaN after everything else (so a NaN is
 * returned only when fewer than k ordinary values exist); k > n pads with (-INF, -1).  Same arguments,
 * workspace (fs_kselect_ws_bytes) and error behaviour as fs_kselect; the same kernels run on the negated
 * values. */
FS_API int fs_kselect_largest(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                              int32_t* out_idx, void* ws, size_t ws_bytes, fs_stream stream);
FS_API size_t fs_kselect_ws_bytes(int64_t n_rows, int64_t n, int k);
/* Same with HOST buffers (pinned or pageable): rows are copied in, selected and copied out in up to
 * 8 slices on three internal streams (copy-in of a slice overlaps the selection of the previous one and
 * the copy-out of the one before); returns after everything has landed.  Device staging is a grow-only
 * allocation owned by the library (kept for the next call, one call at a time per process). */
FS_API int fs_kselect_host(const float* rows_host, int64_t n_rows, int64_t n, int64_t ld, int k,
                    float* out_val_host, int32_t* out_idx_host);
/* fs_kselect for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): same arguments, results and errors as fs_kselect, but the scratch memory of the
 * kernels (row counter; for few long rows the bound, survivor counts and survivor lists) is a
 * built-in __device__ array of FS_NOALLOC_SCRATCH_BYTES, which every GPU that loads the library holds
 * until the process exits.  The call allocates and frees nothing.  A call whose
 * fs_kselect_ws_bytes(n_rows, n, k) exceeds the array returns FS_EUNSUPPORTED (every batch of >= 75 rows
 * needs 256 bytes; one 2^27-element row at k = 1024 needs 0.8 MB).  The array is shared by all calls and
 * keeps the last call's contents; what must start at zero is cleared on `stream` before the kernels run,
 * so calls in stream order are independent.  Calls that OVERLAP on the GPU (several streams or host
 * threads on one device) race on the array: serialise them.  Device ordinals 0..63. */
#define FS_NOALLOC_SCRATCH_BYTES (4u << 20)
FS_API int fs_kselect_noalloc(const float* rows, int64_t n_rows, int64_t n, int64_t ld, int k, float* out_val,
                              int32_t* out_idx, fs_stream stream);
FS_API size_t fs_kselect_noalloc_max_scratch(void);

/* --------------------------------------------------------------------------
 * Exact squared-L2 k-NN (Eq. 1-2; computation layout 5.1):
 * norms (B1), the -2<x,y> tile contraction (B2), "+||y||^2 then k-select" as the
 * tile epilogue (B3: the nq x nb matrix never reaches HBM), merge of the partial
 * lists of database chunks and "+||x||^2" (B4).
 *   xq device fp32 [nq][d], xb device fp32 [nb][d], row-major, contiguous
 *   out_dist device fp32 [nq][k] (full squared distance, clamped at 0)
 *   out_ids  device int64 [nq][k]
 *   1 <= k <= FS_MAX_K; 1 <= d <= 2048; nb < 2^31.
 * Arithmetic: fp32 (FFMA) or 3xTF32-split tensor-core products with fp32
 * accumulation; |dist - exact| <= 1e-4 (||x||^2 + ||y||^2).
 * ------------------------------------------------------------------------ */
FS_API int fs_flat_l2_knn(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k,
                   float* out_dist, int64_t* out_ids, void* ws, size_t ws_bytes,
                   fs_stream stream);
FS_API size_t fs_flat_l2_knn_ws_bytes(int64_t nq, int64_t nb, int d, int k);
FS_API int fs_flat_l2_knn_host(const float* xq_host, int64_t nq, const float* xb_host, int64_t nb, int d,
                        int k, float* out_dist_host, int64_t* out_ids_host);

/* Prepared database.  The ||y_j||^2 of Eq. 2 do not depend on the queries (only the inner-product term
 * is computed per query batch), nor does the database's half of the operand split of the tensor-core engine:
 * fs_flat_prepare computes them once, fs_flat_l2_knn_prepared is fs_flat_l2_knn without that pass (0.45 ms of
 * a 4.4 - 5.6 ms cfg3 call).  Results are bit-identical to fs_flat_l2_knn's.
 *   prep  device memory of the CALLER's, 256-byte aligned, fs_flat_prepare_bytes(nb, d) bytes (the norms;
 *         for d on the tensor-core engine also a lo plane of nb * d floats); written by fs_flat_prepare on
 *         `stream`, only read by the search.  It describes xb's CONTENTS: prepare again after changing them.
 *   xb    the same array in both calls.  If xb is not 16-byte aligned on the tensor-core engine the
 *         prepared block is not used (the call then does what fs_flat_l2_knn does).
 * Errors as fs_flat_l2_knn; FS_EINVAL for a NULL / misaligned / too small prep. */
FS_API size_t fs_flat_prepare_bytes(int64_t nb, int d);
FS_API int fs_flat_prepare(const float* xb, int64_t nb, int d, void* prep, size_t prep_bytes, fs_stream stream);
FS_API int fs_flat_l2_knn_prepared(const float* xq, int64_t nq, const float* xb, const void* prep, size_t prep_bytes,
                            int64_t nb, int d, int k, float* out_dist, int64_t* out_ids, void* ws,
                            size_t ws_bytes, fs_stream stream);

/* --------------------------------------------------------------------------
 * Merge of partial results (database sharding, 5.4 P:L355-363: every shard answers the full query
 * set, "an additional round of k-selection is still required" to join the partial results).
 *   dist device fp32 [nq][G][k], ids device int64 [nq][G][k]: the G lists of every query (from
 *   fs_flat_l2_knn / fs_ivfpq_search on G shards, ids already global); entries with id < 0 are padding.
 *   out_dist [nq][k], out_ids [nq][k]: the k smallest (distance, id) pairs, ascending, ties by lower id,
 *   padded with (+INF, -1).  Distances are taken as they are (no arithmetic; negative values clamp at 0).
 *   Entries of equal distance always come out in ascending id order; which of several entries tied at the
 *   k-th place are kept is decided by (list number, place in the list), which is the id order when every
 *   list is sorted by (distance, id) and list g holds ids below those of list g + 1 -- contiguous id shards.
 * ------------------------------------------------------------------------ */
FS_API int fs_merge_topk(const float* dist, const int64_t* ids, int64_t nq, int G, int k, float* out_dist,
                  int64_t* out_ids, void* ws, size_t ws_bytes, fs_stream stream);
FS_API size_t fs_merge_topk_ws_bytes(int64_t nq, int G, int k);

/* --------------------------------------------------------------------------
 * IVFADC index with 8-bit residual product quantizer (Eq. 3-7, P:L59-90;
 * layout 5.2-5.3, Alg. 4).
 *   d % M == 0, 1 <= M <= 64, nlist >= 1, 256 codewords per
 *   sub-quantizer; sub-vector m = dimensions [m*d/M, (m+1)*d/M).
 * ------------------------------------------------------------------------ */
FS_API int fs_ivfpq_create(fs_ivfpq** out, int d, int nlist, int M);
FS_API int fs_ivfpq_destroy(fs_ivfpq* index);

/* Quantizers: coarse centroids [nlist][d] and PQ codebooks [M][256][d/M], device
 * fp32; copied in / out.  The oracle and the library share these arrays. */
FS_API int fs_ivfpq_set_quantizers(fs_ivfpq* index, const float* coarse, const float* pq,
                            fs_stream stream);
FS_API int fs_ivfpq_get_quantizers(const fs_ivfpq* index, float* coarse, float* pq, fs_stream stream);

/* k-means training of both quantizers on n device vectors x [n][d] (
 * assignment = exact search with k = 1).  Off the parity path: the
 * resulting arrays are what both sides use. */
FS_API int fs_ivfpq_train(fs_ivfpq* index, const float* x, int64_t n, int niter, uint64_t seed,
                   fs_stream stream);

/* Lloyd's k-means on n device vectors x [n][d] (section 6.2: the assignment step is the exact
 * search with k = 1).  centroids: device fp32 [K][d], in / out: with init != 0 they start as the evenly
 * strided input points x[floor(c n / K)], else as given.  niter iterations of (assign to the nearest centroid,
 * ties to the lower one; replace every centroid by the mean of its points -- summed in ascending point order
 * in double precision, so the result is deterministic; an empty cluster c at iteration it is re-seeded from
 * point mix(mix(seed + 0x9E3779B97F4A7C15 (it + 1)) + c) mod n, mix = the splitmix64 finaliser).
 * assign: device int64 [n] or NULL: the assignment the last update was computed from.  n >= K, n < 2^32. */
FS_API int fs_kmeans(const float* x, int64_t n, int d, int K, int niter, uint64_t seed, int init,
              float* centroids, int64_t* assign, fs_stream stream);

/* Add (D1-D3): coarse assignment q1(y) = argmin_c ||y - c||^2 by the flat
 * kernel with k = 1, residual PQ encoding (Eq. 3; byte
 * m = sub-quantizer m), append of (code, id) to list q1(y).
 *   xb device fp32 [n][d]; ids device int64 [n] or NULL (ids ntotal..ntotal+n-1).
 * Lists keep append order (ascending id when ids are added ascending).
 * Needs exclusive access to the index. */
FS_API int fs_ivfpq_add(fs_ivfpq* index, const float* xb, int64_t n, const int64_t* ids,
                 fs_stream stream);

/* Search (C1-C5, Alg. 4): coarse top-nprobe (Eq. 5); the ADC distance (Eq. 7) in the
 * decomposition of Eq. 11: term 1 was stored per vector at add time, term 2 = ||x - c_L||^2 is
 * one number per probed list, term 3 comes from ONE table per query (no per-list tables); inverted-list
 * code scan with fused pass-1 selection, pass-2 merge to k and id resolution for the winners
 * only.  Distances agree with Eq. 7 evaluated in double to ~1e-6 relative.
 *   xq device fp32 [nq][d]; 1 <= nprobe <= min(nlist, 1024); 1 <= k <= FS_MAX_K
 *   out_dist device fp32 [nq][k] (squared ADC distance), out_ids device int64 [nq][k]
 *   out_probed device int32 [nq][nprobe] ascending coarse distance, or NULL. */
FS_API int fs_ivfpq_search(fs_ivfpq* index, const float* xq, int64_t nq, int nprobe, int k,
                    float* out_dist, int64_t* out_ids, int32_t* out_probed, void* ws,
                    size_t ws_bytes, fs_stream stream);
FS_API size_t fs_ivfpq_search_ws_bytes(const fs_ivfpq* index, int64_t nq, int nprobe, int k);
FS_API int fs_ivfpq_search_host(fs_ivfpq* index, const float* xq_host, int64_t nq, int nprobe, int k,
                         float* out_dist_host, int64_t* out_ids_host);

/* All-vs-all k-NN graph (section 6.5: "the k-NN graph ... every vector of the collection is a
 * query"): row i of the output is fs_ivfpq_search's answer for query x_i, computed in batches of `batch`
 * queries (0: 65 536) with one workspace, all on `stream`.  x are normally the vectors the index holds;
 * nothing is special-cased for them: x_i's own id is returned like any other neighbour when its
 * quantised image is among the k nearest (P:L441 does not exclude it either).
 *   x device fp32 [n][d]; out_dist device fp32 [n][k]; out_ids device int64 [n][k];
 *   out_probed device int32 [n][nprobe] or NULL.  Arguments checked as in fs_ivfpq_search. */
FS_API int fs_ivfpq_knn_graph(fs_ivfpq* index, const float* x, int64_t n, int nprobe, int k, int64_t batch,
                       float* out_dist, int64_t* out_ids, int32_t* out_probed, fs_stream stream);

FS_API int64_t fs_ivfpq_ntotal(const fs_ivfpq* index);
/* Total code bytes the probed lists of the last fs_ivfpq_search held
 * (sum over (query, list) pairs of len * M): the scan's algorithmic bytes. */
FS_API int64_t fs_ivfpq_last_scanned_codes(const fs_ivfpq* index);
/* Device time of the three stages of the last fs_ivfpq_search on its stream (CUDA events the
 * search records): ms[0] = C1 coarse top-nprobe, ms[1] = C2-C4 (tables, list scan, pass-1
 * selection: the stage the scan roofline is quoted on), ms[2] = C5 merge + ids.  HOST float
 * [3]; waits for that search to finish. */
FS_API int fs_ivfpq_last_stage_ms(const fs_ivfpq* index, float* ms);
/* Read-only device views of one list, valid until the next add/destroy.  For M = 8 and 16 the scan's
 * storage order is what the view shows: byte i of the vector at list position p holds the index of
 * sub-quantizer i ^ (p mod M) (bank-conflict-free table reads); fs_ivfpq_export and
 * fs_ivfpq_export_lists return the codes in the paper's order (byte m = sub-quantizer m). */
FS_API int fs_ivfpq_list(const fs_ivfpq* index, int list_no, const uint8_t** codes, const int64_t** ids,
                  int64_t* len);
/* The whole inverted file in CSR form, copied to caller buffers (device):
 * offsets int64 [nlist+1], codes uint8 [ntotal][M], ids int64 [ntotal]; any of
 * the three may be NULL. */
FS_API int fs_ivfpq_export(const fs_ivfpq* index, int64_t* offsets, uint8_t* codes, int64_t* ids,
                    fs_stream stream);
/* The same for a subset of the lists (what a checker of a 10^9-vector index copies out: only the
 * lists some queries probed).  list_nos: HOST int32 [n_lists], each in [0, nlist).  offsets_host:
 * HOST int64 [n_lists + 1], always written: list j occupies [offsets_host[j], offsets_host[j+1])
 * of the outputs.  codes (uint8 [total][M]) and ids (int64 [total]) are DEVICE buffers of
 * total = offsets_host[n_lists] entries, or NULL (call once with NULL to size them). */
FS_API int fs_ivfpq_export_lists(const fs_ivfpq* index, const int32_t* list_nos, int64_t n_lists,
                          int64_t* offsets_host, uint8_t* codes, int64_t* ids, fs_stream stream);

#ifdef __cplusplus
}
#endif
#endif /* FS_H_ */
