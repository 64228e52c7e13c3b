// flat.cu -- fs_flat_l2_knn: exact squared-L2 k-NN with the k-selection fused
// into the distance tiles.
//
//   B1 norms        row_norms_kernel: ||y_i||^2, ||x_j||^2 in one pass
//   B2 contraction  flat_tile_kernel main loop: <x_j, y_i> on a TQ x TB tile
//   B3 epilogue     d' = ||y||^2 - 2<x,y> is staged in SHARED memory and each
//                   query row is k-selected right there by one warp (the paper's
//                   fused "+||y||^2 then k-select" kernel, reading the tile
//                   from shared memory instead of a D' matrix in global memory:
//                   the nq x nb matrix never reaches HBM)
//   B4 merge        flat_finish_kernel: the database is cut into S ranges
//                   ("can similarly be tiled over l"); the S partial
//                   queues of a query are selected again, ||x||^2 is added
//                   (not needed before selection) and clamped at 0.
//
// This file is the FFMA (fp32 CUDA-core) engine: exact fp32 products and sums.
// The tensor-core engine (flat_tc.cu) shares the epilogue and the finish pass.
#include "flat.cuh"

namespace fs {

// ---------------------------------------------------------------------------
// B1: squared norms, one warp per vector.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) row_norms_kernel(const float* __restrict__ x, int64_t n,
                                                        int d, float* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (row >= n) return;
  const float* p = x + row * d;
  float s = 0.f;
  for (int c = lane; c < d; c += 32) s = fmaf(p[c], p[c], s);
#pragma unroll
  for (int m = 16; m >= 1; m >>= 1) s += __shfl_xor_sync(kFull, s, m);
  if (lane == 0) out[row] = s;
}

int launch_row_norms(const float* x, int64_t n, int d, float* out, cudaStream_t s) {
  if (n == 0) return FS_OK;
  row_norms_kernel<<<(unsigned)ceil_div(n, 8), 256, 0, s>>>(x, n, d, out);
  FS_LAUNCHED();
  return FS_OK;
}

// ---------------------------------------------------------------------------
// B2 + B3: FFMA tile kernel with the selection epilogue.
// CTA = 256 threads, tile TQ=64 queries x TB=128 database vectors, BK=16.
// Thread (ty, tx) = (tid/16, tid%16) owns rows ty*4..+3 and columns tx*4..+3,
// 64+tx*4..+3.
// ---------------------------------------------------------------------------
namespace {
constexpr int TQ = 64, TB = 128, BK = 16, THREADS = 256;
constexpr int AS = TQ + 4, BS = TB + 4, DS = TB + 4;
constexpr int CBUF = 72;  // keys per row batch: 64 + padding of warp_flush<*, 2>

struct FlatSmem {
  float As[2][BK][AS];
  float Bs[2][BK][BS];
  float Dt[TQ][DS];        // staged d' tile
  float yn[TB];            // ||y||^2 of the tile's columns
  uint64_t buf[TQ][CBUF];  // per-row candidate batches
  uint64_t thr_key[TQ];
  float thr_val[TQ];
  int cnt[TQ];
};
}  // namespace

template <bool VEC>
__global__ void __launch_bounds__(THREADS, 2)
    flat_tile_kernel(const float* __restrict__ xq, int64_t nq, const float* __restrict__ xb,
                     int64_t nb, int d, const float* __restrict__ ynorm, int S,
                     int64_t chunk /* database vectors per split, multiple of TB */, int kclass,
                     uint64_t* __restrict__ Wg /* [nq][S][K] */) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  FlatSmem& sm = *reinterpret_cast<FlatSmem*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tx = tid & 15, ty = tid >> 4;
  const int64_t q0 = (int64_t)blockIdx.x * TQ;
  const int s = blockIdx.y;
  const int64_t b_begin = (int64_t)s * chunk;
  int64_t b_end = b_begin + chunk;
  if (b_end > nb) b_end = nb;
  const int K = 32 << kclass;

  // queue init (sentinels) for this CTA's rows and split
  for (int r = warp; r < TQ; r += THREADS / 32) {
    if (q0 + r < nq) {
      uint64_t* W = Wg + ((q0 + r) * S + s) * K;
      for (int i = lane; i < K; i += 32) W[i] = kSentinelKey;
    }
  }
  if (tid < TQ) {
    sm.thr_key[tid] = kSentinelKey;
    sm.thr_val[tid] = __uint_as_float(0x7FFFFFFFu);
    sm.cnt[tid] = 0;
  }
  __syncthreads();

  // global -> register fetch of one BK slab: A: 1 x 4 floats, B: 2 x 4 floats per thread
  const int lrow = tid >> 2, lk = (tid & 3) * 4;
  auto fetch4 = [&](const float* base, int64_t row, int64_t nrows, int k0, float (&v)[4]) {
    if (row < nrows) {
      const float* p = base + row * d + k0;
      if (VEC) {
        if (k0 + 3 < d) {
          const float4 t = *reinterpret_cast<const float4*>(p);
          v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
          return;
        }
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) v[i] = (k0 + i < d) ? p[i] : 0.f;
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i) v[i] = 0.f;
    }
  };

  for (int64_t b0 = b_begin; b0 < b_end; b0 += TB) {
    float acc[4][8];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;

    float ra[4], rb0[4], rb1[4];
    fetch4(xq, q0 + lrow, nq, lk, ra);
    fetch4(xb, b0 + lrow, b_end, lk, rb0);
    fetch4(xb, b0 + 64 + lrow, b_end, lk, rb1);
    if (tid < TB) sm.yn[tid] = (b0 + tid < b_end) ? ynorm[b0 + tid] : 0.f;
    int cur = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      sm.As[0][lk + i][lrow] = ra[i];
      sm.Bs[0][lk + i][lrow] = rb0[i];
      sm.Bs[0][lk + i][64 + lrow] = rb1[i];
    }
    __syncthreads();
    for (int k0 = 0; k0 < d; k0 += BK) {
      const bool more = k0 + BK < d;
      if (more) {
        fetch4(xq, q0 + lrow, nq, k0 + BK + lk, ra);
        fetch4(xb, b0 + lrow, b_end, k0 + BK + lk, rb0);
        fetch4(xb, b0 + 64 + lrow, b_end, k0 + BK + lk, rb1);
      }
#pragma unroll
      for (int kk = 0; kk < BK; ++kk) {
        const float4 a = *reinterpret_cast<const float4*>(&sm.As[cur][kk][ty * 4]);
        const float4 bl = *reinterpret_cast<const float4*>(&sm.Bs[cur][kk][tx * 4]);
        const float4 bh = *reinterpret_cast<const float4*>(&sm.Bs[cur][kk][64 + tx * 4]);
        const float av[4] = {a.x, a.y, a.z, a.w};
        const float bv[8] = {bl.x, bl.y, bl.z, bl.w, bh.x, bh.y, bh.z, bh.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
      }
      if (more) {
        const int nxt = cur ^ 1;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          sm.As[nxt][lk + i][lrow] = ra[i];
          sm.Bs[nxt][lk + i][lrow] = rb0[i];
          sm.Bs[nxt][lk + i][64 + lrow] = rb1[i];
        }
        __syncthreads();
        cur = nxt;
      }
    }
    // B3 part 1: d' = ||y||^2 - 2 <x, y> staged in shared memory
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float4 lo, hi;
      lo.x = fmaf(-2.f, acc[i][0], sm.yn[tx * 4 + 0]);
      lo.y = fmaf(-2.f, acc[i][1], sm.yn[tx * 4 + 1]);
      lo.z = fmaf(-2.f, acc[i][2], sm.yn[tx * 4 + 2]);
      lo.w = fmaf(-2.f, acc[i][3], sm.yn[tx * 4 + 3]);
      hi.x = fmaf(-2.f, acc[i][4], sm.yn[64 + tx * 4 + 0]);
      hi.y = fmaf(-2.f, acc[i][5], sm.yn[64 + tx * 4 + 1]);
      hi.z = fmaf(-2.f, acc[i][6], sm.yn[64 + tx * 4 + 2]);
      hi.w = fmaf(-2.f, acc[i][7], sm.yn[64 + tx * 4 + 3]);
      *reinterpret_cast<float4*>(&sm.Dt[ty * 4 + i][tx * 4]) = lo;
      *reinterpret_cast<float4*>(&sm.Dt[ty * 4 + i][64 + tx * 4]) = hi;
    }
    __syncthreads();
    // B3 part 2: one warp k-selects each row of the staged tile (lane j owns
    // columns 4j..4j+3), state carried across tiles in shared/global memory
    const int ncols = (int)((b_end - b0) < TB ? (b_end - b0) : TB);
    for (int r = warp; r < TQ; r += THREADS / 32) {
      if (q0 + r >= nq) continue;
      const float4 x = *reinterpret_cast<const float4*>(&sm.Dt[r][lane * 4]);
      float thr_val = sm.thr_val[r];
      const int c0 = lane * 4;
      const bool any = (c0 < ncols) && (!(x.x > thr_val) | !(x.y > thr_val) | !(x.z > thr_val) |
                                        !(x.w > thr_val));
      if (!__any_sync(kFull, any)) continue;
      uint64_t thr = sm.thr_key[r];
      int cnt = sm.cnt[r];
      uint64_t* buf = sm.buf[r];
#pragma unroll 1
      for (int t = 0; t < 4; ++t) {
        const float xv = t == 0 ? x.x : t == 1 ? x.y : t == 2 ? x.z : x.w;
        const uint64_t key = make_key(xv, (uint32_t)(b0 + c0 + t));
        const bool pred = (c0 + t < ncols) && !(xv > thr_val) && key < thr;
        const unsigned m = __ballot_sync(kFull, pred);
        if (m == 0) continue;
        if (pred) buf[cnt + __popc(m & ((1u << lane) - 1u))] = key;
        cnt += __popc(m);
        if (cnt > 32) {
          thr = warp_flush_b64(kclass, Wg + ((q0 + r) * S + s) * K + lane, 32, buf, cnt);
          thr_val = key_val(thr);
          cnt = 0;
        }
      }
      if (lane == 0) {
        sm.thr_key[r] = thr;
        sm.thr_val[r] = thr_val;
        sm.cnt[r] = cnt;
      }
    }
    __syncthreads();
  }
  // drain the batches
  for (int r = warp; r < TQ; r += THREADS / 32) {
    if (q0 + r >= nq) continue;
    const int cnt = sm.cnt[r];
    if (cnt > 0) warp_flush_b64(kclass, Wg + ((q0 + r) * S + s) * K + lane, 32, sm.buf[r], cnt);
  }
}

// ---------------------------------------------------------------------------
// B4: select again over the S partial queues of each query, add ||x||^2, clamp,
// widen ids.  One warp per query.  xnorm may be NULL (adds nothing).
// ---------------------------------------------------------------------------
template <int NQ>
__global__ void __launch_bounds__(128) flat_finish_kernel(const uint64_t* __restrict__ Wg,
                                                          int64_t nq, int S, int k,
                                                          const float* __restrict__ xnorm,
                                                          float* __restrict__ out_dist,
                                                          int64_t* __restrict__ out_ids, const FinishExtra ex) {
  extern __shared__ __align__(16) uint64_t smem_keys[];
  constexpr int NB = NQ < 4 ? NQ : 4;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t q = (int64_t)blockIdx.x * 4 + warp;
  if (ex.nq_dev) nq = (int64_t)*ex.nq_dev < nq ? (int64_t)*ex.nq_dev : nq;
  if (q >= nq) return;
  const int64_t oq = ex.qmap ? (int64_t)ex.qmap[q] : q;  // the query this row belongs to
  constexpr int K = 32 * NQ;
  WarpSelect<NQ, NB> sel;
  sel.init(smem_keys + warp * warp_select_smem_keys<NB>(), lane);
  const uint64_t* src = Wg + q * S * K;
  if (S == 1) {
#pragma unroll
    for (int r = 0; r < NQ; ++r) sel.W[r] = src[r * 32 + lane];
  } else {
    // ex.packed: a partial queue holds its keys first and sentinels behind them, so the first 32 slots that
    // hold only sentinels end the queue (with tight bounds most queues are nearly empty)
    for (int sq = 0; sq < S; ++sq) {
      const uint64_t* qs = src + (int64_t)sq * K;
      for (int e0 = 0; e0 < K; e0 += 32) {
        const uint64_t key = qs[e0 + lane];
        if (ex.packed && __all_sync(kFull, key == kSentinelKey)) break;
        sel.push(key < sel.thr, key);  // sentinels never pass: thr <= sentinel
      }
    }
    sel.finish();
  }
  if (ex.bound_out) {  // the sample pass: only the k-th smallest d' is wanted, as a bound
    sort_blocked<NQ>(sel.W, lane);
#pragma unroll
    for (int r = 0; r < NQ; ++r)
      if (lane * NQ + r == k - 1) ex.bound_out[oq] = (unsigned int)(sel.W[r] >> 32);
    return;
  }
  if (ex.fail_cnt) {  // fewer keys than the query must have: its sampled bound was too tight
    int have = 0;
#pragma unroll
    for (int r = 0; r < NQ; ++r) have += sel.W[r] != kSentinelKey;
    have = __reduce_add_sync(kFull, have);
    if (have < ex.need && lane == 0) ex.fail_q[atomicAdd(ex.fail_cnt, 1u)] = (int)q;
  }
  // Final value = d' + ||x||^2, clamped at 0.  Rounding (and the clamp) can make
  // distinct d' equal, so order again on the final (value, id) keys: ascending,
  // ties by lower id.  The lane-stride registers are read as a blocked array
  // (any bijection is fine before a full sort); sorted element e = lane*NQ + r.
  const float xn = xnorm ? xnorm[oq] : 0.f;
#pragma unroll
  for (int r = 0; r < NQ; ++r) {
    const uint64_t key = sel.W[r];
    if (key != kSentinelKey) {
      const float dv = key_val(key) + xn;
      sel.W[r] = make_key(dv > 0.f ? dv : 0.f, key_idx(key));
    }
  }
  sort_blocked<NQ>(sel.W, lane);
#pragma unroll
  for (int r = 0; r < NQ; ++r) {
    const int i = lane * NQ + r;
    if (i < k) {
      const uint64_t key = sel.W[r];
      if (key == kSentinelKey) {
        out_dist[oq * k + i] = __uint_as_float(0x7F800000u);
        out_ids[oq * k + i] = -1;
      } else {
        out_dist[oq * k + i] = key_val(key);
        out_ids[oq * k + i] = (int64_t)key_idx(key);
      }
    }
  }
}

template <int NQ>
static int launch_finish_t(const uint64_t* Wg, int64_t nq, int S, int k, const float* xnorm,
                           float* out_dist, int64_t* out_ids, cudaStream_t s, const FinishExtra& ex) {
  constexpr int NB = NQ < 4 ? NQ : 4;
  const size_t smem = 4 * warp_select_smem_keys<NB>() * sizeof(uint64_t);
  flat_finish_kernel<NQ><<<(unsigned)ceil_div(nq, 4), 128, smem, s>>>(Wg, nq, S, k, xnorm,
                                                                      out_dist, out_ids, ex);
  FS_LAUNCHED();
  return FS_OK;
}

// ---------------------------------------------------------------------------
// Positions -> ids after a selection on (distance, position) keys (IVFPQ C5, shard merge).
// ---------------------------------------------------------------------------
// C5 second half: positions -> ids; entries with bitwise-equal distance are put
// in ascending id order (positions order them by list and append order, which is
// ascending id only inside a list filled in ascending id order).  One warp per query.
__global__ void __launch_bounds__(128)
    resolve_ids_kernel(float* __restrict__ dist, int64_t* __restrict__ ids_io,
                       const int64_t* __restrict__ ids_all, int64_t table_stride, int64_t nq, int k) {
  extern __shared__ __align__(16) unsigned char res_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t q = (int64_t)blockIdx.x * 4 + warp;
  if (q >= nq) return;
  const int64_t* ids = ids_all + q * table_stride;  // per-query table (shard merge) or one table (stride 0)
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

int launch_resolve_ids(float* dist, int64_t* ids_io, const int64_t* table, int64_t nq, int k, cudaStream_t s,
                       int64_t table_stride) {
  if (nq == 0) return FS_OK;
  const size_t smem = (size_t)4 * k * (sizeof(int64_t) + sizeof(float));
  resolve_ids_kernel<<<(unsigned)ceil_div(nq, 4), 128, smem, s>>>(dist, ids_io, table, table_stride, nq, k);
  FS_LAUNCHED();
  return FS_OK;
}

// ---------------------------------------------------------------------------
// Merge of G partial results per query (database shards: "an additional round of
// k-selection is still required"): (distance, id) pairs -> keys (distance image, position in the
// query's G * k candidates), padded to the queue class.
// ---------------------------------------------------------------------------
__global__ void merge_pack_kernel(const float* __restrict__ dist, const int64_t* __restrict__ ids, int64_t nq, int G, int k,
                                  int K, uint64_t* __restrict__ Wg) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // over [nq][G][K]
  if (e >= nq * G * K) return;
  const int i = (int)(e % K);
  const int64_t qg = e / K;  // q * G + g
  uint64_t key = kSentinelKey;
  if (i < k) {
    const int64_t src = qg * k + i;
    const int g = (int)(qg % G);
    if (ids[src] >= 0) key = make_key(dist[src], (uint32_t)(g * k + i));
  }
  Wg[e] = key;
}

int launch_merge_pack(const float* dist, const int64_t* ids, int64_t nq, int G, int k, int K, uint64_t* Wg, cudaStream_t s) {
  const int64_t n = nq * G * K;
  if (n == 0) return FS_OK;
  merge_pack_kernel<<<(unsigned)ceil_div(n, 256), 256, 0, s>>>(dist, ids, nq, G, k, K, Wg);
  FS_LAUNCHED();
  return FS_OK;
}

int launch_flat_finish(const uint64_t* Wg, int64_t nq, int S, int k, const float* xnorm,
                       float* out_dist, int64_t* out_ids, cudaStream_t s, const FinishExtra* extra) {
  if (nq == 0) return FS_OK;
  const FinishExtra ex = extra ? *extra : FinishExtra();
  switch (k_class(k)) {
    case 0: return launch_finish_t<1>(Wg, nq, S, k, xnorm, out_dist, out_ids, s, ex);
    case 1: return launch_finish_t<2>(Wg, nq, S, k, xnorm, out_dist, out_ids, s, ex);
    case 2: return launch_finish_t<4>(Wg, nq, S, k, xnorm, out_dist, out_ids, s, ex);
    case 3: return launch_finish_t<8>(Wg, nq, S, k, xnorm, out_dist, out_ids, s, ex);
    case 4: return launch_finish_t<16>(Wg, nq, S, k, xnorm, out_dist, out_ids, s, ex);
    default: return launch_finish_t<32>(Wg, nq, S, k, xnorm, out_dist, out_ids, s, ex);
  }
}

// ---------------------------------------------------------------------------
// Host driver
// ---------------------------------------------------------------------------
FlatPlan flat_plan(int64_t nq, int64_t nb, int d, int k) {
  FlatPlan p;
  p.kclass = k_class(k);
  p.K = 32 << p.kclass;
  const int64_t qtiles = ceil_div(nq, TQ);
  const int64_t btiles = ceil_div(nb, TB);
  // Database splits: fill the GPU (2 CTAs per SM) with as few partial queues as
  // possible, preferring counts that leave the last wave nearly full.
  const int64_t slots = (int64_t)sm_count() * 2;
  int64_t best_S = 1;
  double best_score = -1.0;
  const int64_t max_S = btiles < 64 ? btiles : 64;
  for (int64_t S = 1; S <= max_S; ++S) {
    const int64_t per = ceil_div(btiles, S);
    if (S > 1 && per < 8) break;  // at least 8 tiles (1024 vectors) per split
    const int64_t realS = ceil_div(btiles, per);
    const int64_t ctas = qtiles * realS;
    const double eff = (double)ctas / (double)(ceil_div(ctas, slots) * slots);
    const double score = eff - 0.004 * (double)realS;  // fewer splits on near-ties
    if (score > best_score) {
      best_score = score;
      best_S = realS;
    }
  }
  const int64_t per = ceil_div(btiles > 0 ? btiles : 1, best_S);
  p.chunk = per * TB;
  p.S = (int)(nb > 0 ? ceil_div(nb, p.chunk) : 1);
  p.off_ynorm = 0;
  p.off_xnorm = align_up((size_t)nb * sizeof(float), 256);
  p.off_W = p.off_xnorm + align_up((size_t)nq * sizeof(float), 256);
  p.bytes = p.off_W + align_up((size_t)nq * p.S * p.K * sizeof(uint64_t), 256);
  if (flat_tc_supported(d) && nq > 0 && nb > 0) {  // the tensor-core engine lays out its own workspace
    const size_t tb = flat_tc_plan(nq, nb, d, k).bytes;
    if (tb > p.bytes) p.bytes = tb;
  }
  return p;
}

int flat_knn_device(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k,
                    const float* ynorm_opt, float* out_dist, int64_t* out_ids, void* ws,
                    cudaStream_t s, const FlatPrep* prep) {
  if (flat_tc_supported(d)) return flat_knn_tc_device(xq, nq, xb, nb, d, k, out_dist, out_ids, ws, s, nullptr, 0, prep);
  if (prep != nullptr && ynorm_opt == nullptr) ynorm_opt = prep->ynorm;
  const FlatPlan p = flat_plan(nq, nb, d, k);
  char* w = static_cast<char*>(ws);
  float* ynorm = reinterpret_cast<float*>(w + p.off_ynorm);
  float* xnorm = reinterpret_cast<float*>(w + p.off_xnorm);
  uint64_t* Wg = reinterpret_cast<uint64_t*>(w + p.off_W);
  int rc;
  if (ynorm_opt == nullptr) {
    if ((rc = launch_row_norms(xb, nb, d, ynorm, s)) != FS_OK) return rc;
  }
  if ((rc = launch_row_norms(xq, nq, d, xnorm, s)) != FS_OK) return rc;
  const float* yn = ynorm_opt ? ynorm_opt : ynorm;

  const bool vec = (d % 4 == 0) && (((uintptr_t)xq | (uintptr_t)xb) % 16 == 0);
  const dim3 grid((unsigned)ceil_div(nq, TQ), (unsigned)p.S);
  const size_t smem = sizeof(FlatSmem);
  // (function attributes are per device: set on every call, it costs about a microsecond)
  FS_CUDA(cudaFuncSetAttribute(flat_tile_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  FS_CUDA(cudaFuncSetAttribute(flat_tile_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  if (vec)
    flat_tile_kernel<true><<<grid, THREADS, smem, s>>>(xq, nq, xb, nb, d, yn, p.S, p.chunk, p.kclass, Wg);
  else
    flat_tile_kernel<false><<<grid, THREADS, smem, s>>>(xq, nq, xb, nb, d, yn, p.S, p.chunk, p.kclass, Wg);
  FS_LAUNCHED();
  return launch_flat_finish(Wg, nq, p.S, k, xnorm, out_dist, out_ids, s);
}

__global__ void fill_padding_kernel(float* dist, int64_t* ids, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    dist[i] = __uint_as_float(0x7F800000u);
    ids[i] = -1;
  }
}

int flat_validate(const void* xq, int64_t nq, const void* xb, int64_t nb, int d, int k,
                  const void* od, const void* oi) {
  if (nq < 0 || nb < 0) return set_error(FS_EINVAL, "fs_flat_l2_knn: negative size");
  if (d < 1 || k < 1) return set_error(FS_EINVAL, "fs_flat_l2_knn: d and k must be >= 1");
  if (k > FS_MAX_K) return set_error(FS_EUNSUPPORTED, "fs_flat_l2_knn: k = %d > %d", k, FS_MAX_K);
  if (d > 2048) return set_error(FS_EUNSUPPORTED, "fs_flat_l2_knn: d = %d > 2048", d);
  if (nb >= (1LL << 31)) return set_error(FS_EUNSUPPORTED, "fs_flat_l2_knn: nb must be < 2^31");
  if (ceil_div(nq, TQ) > 0x7fffffffLL) return set_error(FS_EUNSUPPORTED, "fs_flat_l2_knn: nq too large");
  if (nq > 0 && (!xq || !od || !oi || (nb > 0 && !xb)))
    return set_error(FS_EINVAL, "fs_flat_l2_knn: NULL pointer");
  return FS_OK;
}

}  // namespace fs

extern "C" {

const char* fs_flat_engine(void) {
  return fs::flat_tc_supported(128) ? "tcgen05-3xtf32 (d % 4 == 0, 32 <= d <= 128; ffma-fp32 otherwise)" : "ffma-fp32";
}

size_t fs_flat_l2_knn_ws_bytes(int64_t nq, int64_t nb, int d, int k) {
  if (nq < 0 || nb < 0 || d < 1 || k < 1 || k > FS_MAX_K) return 0;
  return fs::flat_plan(nq, nb, d, k).bytes;
}

static int flat_l2_knn_entry(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k, float* out_dist,
                             int64_t* out_ids, void* ws, size_t ws_bytes, fs_stream stream, const void* prep) {
  int rc = fs::flat_validate(xq, nq, xb, nb, d, k, out_dist, out_ids);
  if (rc != FS_OK) return rc;
  if (nq == 0) return FS_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (nb == 0) {
    const int64_t n = nq * k;
    fs::fill_padding_kernel<<<(unsigned)fs::ceil_div(n, 256), 256, 0, s>>>(out_dist, out_ids, n);
    FS_LAUNCHED();
    return FS_OK;
  }
  fs::TempWs t;
  rc = t.acquire(ws, ws_bytes, fs::flat_plan(nq, nb, d, k).bytes, s);
  if (rc != FS_OK) return rc;
  fs::FlatPrep view;
  if (prep) view = fs::flat_prep_view(prep, nb, d);
  return fs::flat_knn_device(xq, nq, xb, nb, d, k, nullptr, out_dist, out_ids, t.ptr, s, prep ? &view : nullptr);
}

int fs_flat_l2_knn(const float* xq, int64_t nq, const float* xb, int64_t nb, int d, int k,
                   float* out_dist, int64_t* out_ids, void* ws, size_t ws_bytes, fs_stream stream) {
  return flat_l2_knn_entry(xq, nq, xb, nb, d, k, out_dist, out_ids, ws, ws_bytes, stream, nullptr);
}

size_t fs_flat_prepare_bytes(int64_t nb, int d) {
  if (nb < 0 || d < 1 || d > 2048 || nb >= (1LL << 31)) return 0;
  return fs::flat_prep_bytes(nb, d);
}

int fs_flat_prepare(const float* xb, int64_t nb, int d, void* prep, size_t prep_bytes, fs_stream stream) {
  if (nb < 0 || d < 1) return fs::set_error(FS_EINVAL, "fs_flat_prepare: nb >= 0 and d >= 1");
  if (d > 2048 || nb >= (1LL << 31)) return fs::set_error(FS_EUNSUPPORTED, "fs_flat_prepare: d <= 2048, nb < 2^31");
  if (!prep || (nb > 0 && !xb)) return fs::set_error(FS_EINVAL, "fs_flat_prepare: NULL pointer");
  if ((reinterpret_cast<uintptr_t>(prep) & 255u) != 0) return fs::set_error(FS_EINVAL, "fs_flat_prepare: prep must be 256-byte aligned");
  if (prep_bytes < fs::flat_prep_bytes(nb, d))
    return fs::set_error(FS_EINVAL, "fs_flat_prepare: prep holds %zu bytes, %zu needed", prep_bytes, fs::flat_prep_bytes(nb, d));
  return fs::flat_prepare_device(xb, nb, d, prep, static_cast<cudaStream_t>(stream));
}

int fs_flat_l2_knn_prepared(const float* xq, int64_t nq, const float* xb, const void* prep, size_t prep_bytes, int64_t nb,
                            int d, int k, float* out_dist, int64_t* out_ids, void* ws, size_t ws_bytes,
                            fs_stream stream) {
  if (!prep) return fs::set_error(FS_EINVAL, "fs_flat_l2_knn_prepared: prep is NULL");
  if ((reinterpret_cast<uintptr_t>(prep) & 255u) != 0)
    return fs::set_error(FS_EINVAL, "fs_flat_l2_knn_prepared: prep must be 256-byte aligned");
  if (nb >= 0 && d >= 1 && d <= 2048 && nb < (1LL << 31) && prep_bytes < fs::flat_prep_bytes(nb, d))
    return fs::set_error(FS_EINVAL, "fs_flat_l2_knn_prepared: prep holds %zu bytes, %zu needed", prep_bytes,
                         fs::flat_prep_bytes(nb, d));
  return flat_l2_knn_entry(xq, nq, xb, nb, d, k, out_dist, out_ids, ws, ws_bytes, stream, prep);
}

size_t fs_merge_topk_ws_bytes(int64_t nq, int G, int k) {
  if (nq < 0 || G < 1 || k < 1 || k > FS_MAX_K) return 0;
  return fs::align_up((size_t)nq * G * (32 << fs::k_class(k)) * sizeof(uint64_t), 256);
}

int fs_merge_topk(const float* dist, const int64_t* ids, int64_t nq, int G, int k, float* out_dist,
                  int64_t* out_ids, void* ws, size_t ws_bytes, fs_stream stream) {
  if (nq < 0 || G < 1) return fs::set_error(FS_EINVAL, "fs_merge_topk: need nq >= 0, G >= 1");
  if (k < 1) return fs::set_error(FS_EINVAL, "fs_merge_topk: k must be >= 1");
  if (k > FS_MAX_K) return fs::set_error(FS_EUNSUPPORTED, "fs_merge_topk: k = %d > %d", k, FS_MAX_K);
  if ((int64_t)G * k >= (1LL << 31)) return fs::set_error(FS_EUNSUPPORTED, "fs_merge_topk: G * k too large");
  if (nq > 0 && (!dist || !ids || !out_dist || !out_ids)) return fs::set_error(FS_EINVAL, "fs_merge_topk: NULL pointer");
  if (nq == 0) return FS_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  fs::TempWs t;
  int rc = t.acquire(ws, ws_bytes, fs_merge_topk_ws_bytes(nq, G, k), s);
  if (rc != FS_OK) return rc;
  uint64_t* Wg = static_cast<uint64_t*>(t.ptr);
  const int K = 32 << fs::k_class(k);
  if ((rc = fs::launch_merge_pack(dist, ids, nq, G, k, K, Wg, s)) != FS_OK) return rc;
  if ((rc = fs::launch_flat_finish(Wg, nq, G, k, nullptr, out_dist, out_ids, s)) != FS_OK) return rc;
  // positions in the query's G * k candidates -> ids; equal distances in ascending id order
  return fs::launch_resolve_ids(out_dist, out_ids, ids, nq, k, s, (int64_t)G * k);
}

int fs_flat_l2_knn_host(const float* xq_host, int64_t nq, const float* xb_host, int64_t nb, int d,
                        int k, float* out_dist_host, int64_t* out_ids_host) {
  int rc = fs::flat_validate(xq_host, nq, xb_host, nb, d, k, out_dist_host, out_ids_host);
  if (rc != FS_OK) return rc;
  if (nq == 0) return FS_OK;
  float *dq = nullptr, *db = nullptr, *dd = nullptr;
  int64_t* di = nullptr;
  cudaStream_t s = nullptr;
  const size_t qb = (size_t)nq * d * sizeof(float), bb = (size_t)nb * d * sizeof(float);
  const size_t on = (size_t)nq * k;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) {
    if (e == cudaSuccess) e = r;
    return e == cudaSuccess;
  };
  ok(cudaMalloc(&dq, qb)) && ok(cudaMalloc(&db, bb ? bb : 16)) &&
      ok(cudaMalloc(&dd, on * sizeof(float))) && ok(cudaMalloc(&di, on * sizeof(int64_t))) &&
      ok(cudaMemcpyAsync(dq, xq_host, qb, cudaMemcpyHostToDevice, s)) &&
      (bb == 0 || ok(cudaMemcpyAsync(db, xb_host, bb, cudaMemcpyHostToDevice, s)));
  if (e == cudaSuccess) {
    rc = fs_flat_l2_knn(dq, nq, db, nb, d, k, dd, di, nullptr, 0, s);
    if (rc == FS_OK) {
      ok(cudaMemcpyAsync(out_dist_host, dd, on * sizeof(float), cudaMemcpyDeviceToHost, s)) &&
          ok(cudaMemcpyAsync(out_ids_host, di, on * sizeof(int64_t), cudaMemcpyDeviceToHost, s));
    }
  }
  ok(cudaStreamSynchronize(s));
  cudaFree(dq);
  cudaFree(db);
  cudaFree(dd);
  cudaFree(di);
  if (rc == FS_OK && e != cudaSuccess)
    rc = fs::set_error(FS_ECUDA, "fs_flat_l2_knn_host: %s", cudaGetErrorString(e));
  return rc;
}

}  // extern "C"
