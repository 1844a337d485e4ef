// sx_api.cu -- the C ABI of include/sparsex.h: argument validation, workspace carve-up, TMA
// descriptor construction and stage sequencing. All arithmetic of the method is in the kernels.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <mutex>

#include "sx_internal.h"

namespace sx {

static thread_local char g_err[512] = "";

sx_status set_error(sx_status st, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return st;
}

static std::atomic<uint64_t> g_launches{0};  // diagnostic only (sx_launch_count)

sx_status check_launch(const char *what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SX_OK;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

WsLayout ws_layout(const sx_pool *pool, const sx_batch *b) {
  WsLayout w;
  size_t off = 0;
  w.rope_table = off;
  off = align_up(off + sizeof(float2) * 64 * (size_t)(b->num_segments > 0 ? b->num_segments : 1), 256);
  w.page_desc = off;
  off = align_up(off + sizeof(int4) * (size_t)(b->total_seg_pages > 0 ? b->total_seg_pages : 1), 256);
  w.lse_new = off;
  off = align_up(off + 8 * sizeof(float) * (size_t)(b->total_new > 0 ? b->total_new : 1) * pool->num_q_heads, 256);
  w.partial = off;
  off = align_up(off + sizeof(float) * (size_t)pool->num_kv_heads * b->total_tokens, 256);
  w.scores = off;
  off = align_up(off + sizeof(float) * (size_t)b->total_tokens, 256);
  w.col_tab = off;
  off = align_up(off + colsum_tab_bytes(pool, b), 256);
  w.rows_tmp = off;
  off = align_up(off + sizeof(int32_t) * (size_t)b->total_tokens, 256);
  w.rows_cnt = off;
  off = align_up(off + sizeof(int32_t) * (size_t)b->num_reqs, 256);
  w.attn_part = off;
  off = align_up(off + attn_part_bytes(), 256);
  w.sel_scratch = off;
  off = align_up(off + select_scratch_bytes(b), 256);
  w.small_part = off;
  off = align_up(off + small_ws_bytes(b->num_reqs, pool->num_kv_heads, pool->num_q_heads / pool->num_kv_heads), 256);
  w.page_seg = off;
  off = align_up(off + sizeof(int32_t) * (size_t)b->num_reqs * b->max_pages_per_req, 256);
  w.total = off;
  return w;
}

static bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

static sx_status validate(const sx_pool *pool, const sx_batch *b) {
  if (!pool || !b) return set_error(SX_ERR_INVALID_ARG, "pool or batch is NULL");
  if (!pool->k || !pool->v) return set_error(SX_ERR_INVALID_ARG, "pool.k / pool.v is NULL");
  if (pool->head_dim != kHeadDim) return set_error(SX_ERR_UNSUPPORTED, "head_dim must be 128 (got %d)", pool->head_dim);
  if (pool->block_size != kPage) return set_error(SX_ERR_UNSUPPORTED, "block_size must be 16 (got %d)", pool->block_size);
  if (pool->num_blocks <= 0 || pool->num_kv_heads <= 0 || pool->num_q_heads <= 0)
    return set_error(SX_ERR_INVALID_ARG, "pool sizes must be positive");
  if (pool->num_q_heads % pool->num_kv_heads != 0 || pool->num_q_heads / pool->num_kv_heads > 128)
    return set_error(SX_ERR_UNSUPPORTED, "num_q_heads must be a multiple of num_kv_heads with group <= 128");
  if ((int64_t)pool->num_blocks * pool->num_kv_heads * kPage >= (int64_t)1 << 31)
    return set_error(SX_ERR_UNSUPPORTED, "pool too large for 32-bit TMA row coordinates");
  if (b->num_reqs <= 0 || b->num_segments < 0 || b->max_pages_per_req <= 0 || b->total_tokens <= 0 ||
      b->total_new < 0 || b->total_seg_pages < 0 || b->max_seq_len <= 0)
    return set_error(SX_ERR_INVALID_ARG, "batch sizes out of range");
  if (b->max_seq_len > b->max_pages_per_req * kPage)
    return set_error(SX_ERR_INVALID_ARG, "max_seq_len exceeds max_pages_per_req * 16");
  if (!b->seq_len || !b->tok_off || !b->k_block_table || !b->v_block_table || !b->new_off)
    return set_error(SX_ERR_INVALID_ARG, "a required batch array is NULL");
  if (b->num_segments > 0 && (!b->segments || !b->src_blocks))
    return set_error(SX_ERR_INVALID_ARG, "segments / src_blocks is NULL");
  if (b->total_new > 0 && !b->new_idx) return set_error(SX_ERR_INVALID_ARG, "new_idx is NULL");
  if (b->rope_style != 0 && b->rope_style != 1)
    return set_error(SX_ERR_UNSUPPORTED, "rope_style must be 0 (half-split) or 1 (interleaved)");
  if (!(b->rope_theta > 1.0)) return set_error(SX_ERR_INVALID_ARG, "rope_theta must be > 1");
  if (b->zero_copy != 0 && b->zero_copy != 1) return set_error(SX_ERR_INVALID_ARG, "zero_copy must be 0 or 1");
  if (misaligned(pool->k) || misaligned(pool->v)) return set_error(SX_ERR_MISALIGNED, "pool.k / pool.v not 16-B aligned");
  return SX_OK;
}

// zero-copy mode: build the rotation table and the page classification in the workspace (one small launch)
static sx_status zc_prepare(const sx_pool *pool, const sx_batch *b, void *ws, cudaStream_t s, ZcArgs *zc) {
  *zc = ZcArgs();
  if (!b->zero_copy || b->num_segments == 0) return SX_OK;
  const WsLayout w = ws_layout(pool, b);
  float2 *table = reinterpret_cast<float2 *>(static_cast<char *>(ws) + w.rope_table);
  int32_t *page_seg = reinterpret_cast<int32_t *>(static_cast<char *>(ws) + w.page_seg);
  zc->style = b->rope_style;
  zc->table = table;
  zc->page_seg = page_seg;
  return launch_zc_prepare(b, table, page_seg, s);
}

static sx_status validate_ws(const sx_pool *pool, const sx_batch *b, const void *ws, size_t ws_bytes) {
  WsLayout w = ws_layout(pool, b);
  if (!ws) return set_error(SX_ERR_INVALID_ARG, "workspace is NULL");
  if ((reinterpret_cast<uintptr_t>(ws) & 255u) != 0) return set_error(SX_ERR_MISALIGNED, "workspace not 256-B aligned");
  if (ws_bytes < w.total) return set_error(SX_ERR_WORKSPACE, "workspace too small: %zu < %zu", ws_bytes, w.total);
  return SX_OK;
}

// ------------------------------------------------------------------------------------ tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

static sx_status get_encode(EncodeTiledFn *fn) {
  static std::once_flag once;
  static EncodeTiledFn cached = nullptr;
  static cudaError_t err = cudaSuccess;
  std::call_once(once, [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    err = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q);
    if (err == cudaSuccess && q == cudaDriverEntryPointSuccess) cached = reinterpret_cast<EncodeTiledFn>(p);
  });
  if (!cached) {
    cudaGetLastError();
    return set_error(SX_ERR_CUDA, "cuTensorMapEncodeTiled unavailable: %s", cudaGetErrorString(err));
  }
  *fn = cached;
  return SX_OK;
}

// Encoded tensor maps are a pure function of (base pointer, shape): a small process-wide cache keyed by exactly
// those values saves the three driver encodes per stage call (visible on launch-bound configs such as C1). The
// only state the library keeps besides the last-error text and the launch counter; nothing in it can go stale.
struct TmapKey {
  const void *base;
  int a, b, c, d;  // pool: (num_blocks, Hkv, -1, -1); q: (total_rows, Hq, group, rows_per_tile)
  bool operator==(const TmapKey &o) const { return base == o.base && a == o.a && b == o.b && c == o.c && d == o.d; }
};
constexpr int kTmapCache = 256;
static std::mutex g_tmap_mu;
static TmapKey g_tmap_key[kTmapCache];
static CUtensorMap g_tmap_val[kTmapCache];
static int g_tmap_n = 0, g_tmap_next = 0;

static bool tmap_lookup(const TmapKey &k, CUtensorMap *out) {
  std::lock_guard<std::mutex> lk(g_tmap_mu);
  for (int i = 0; i < g_tmap_n; ++i)
    if (g_tmap_key[i] == k) {
      *out = g_tmap_val[i];
      return true;
    }
  return false;
}
static void tmap_store(const TmapKey &k, const CUtensorMap &v) {
  std::lock_guard<std::mutex> lk(g_tmap_mu);
  const int i = g_tmap_n < kTmapCache ? g_tmap_n++ : (g_tmap_next++ % kTmapCache);
  g_tmap_key[i] = k;
  g_tmap_val[i] = v;
}

// Pool viewed as a 2-D bf16 matrix [num_blocks*Hkv*16 rows][128]; box = 64 columns x 16 rows (one
// half of one (page, head) tile), 128-B swizzle: lands as two 8-row x 128-B swizzle atoms.
sx_status make_tmap_pool(CUtensorMap *out, const void *base, int num_blocks, int num_kv_heads) {
  const TmapKey key{base, num_blocks, num_kv_heads, -1, -1};
  if (tmap_lookup(key, out)) return SX_OK;
  EncodeTiledFn enc;
  sx_status st = get_encode(&enc);
  if (st != SX_OK) return st;
  cuuint64_t dims[2] = {(cuuint64_t)kHeadDim, (cuuint64_t)num_blocks * num_kv_heads * kPage};
  cuuint64_t strides[1] = {(cuuint64_t)kHeadDim * 2};
  cuuint32_t box[2] = {64, (cuuint32_t)kPage};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_error(SX_ERR_CUDA, "cuTensorMapEncodeTiled(pool) failed: %d", (int)r);
  tmap_store(key, *out);
  return SX_OK;
}

// Query rows [total_rows][Hq][128] viewed as 3-D (d, head, row); box = 64 d x g heads x rows_per_tile
// rows: the g query heads of one KV group for rows_per_tile consecutive rows land as (row, head)-
// ordered 128-B lines = the GQA-packed M (or N) dimension of a tile. Rows beyond total_rows are
// zero-filled by the TMA unit.
sx_status make_tmap_q(CUtensorMap *out, const void *base, int total_rows, int num_q_heads, int group,
                      int rows_per_tile) {
  const TmapKey key{base, total_rows, num_q_heads, group, rows_per_tile};
  if (tmap_lookup(key, out)) return SX_OK;
  EncodeTiledFn enc;
  sx_status st = get_encode(&enc);
  if (st != SX_OK) return st;
  cuuint64_t dims[3] = {(cuuint64_t)kHeadDim, (cuuint64_t)num_q_heads, (cuuint64_t)total_rows};
  cuuint64_t strides[2] = {(cuuint64_t)kHeadDim * 2, (cuuint64_t)kHeadDim * 2 * num_q_heads};
  cuuint32_t box[3] = {64, (cuuint32_t)group, (cuuint32_t)rows_per_tile};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(base), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return set_error(SX_ERR_CUDA, "cuTensorMapEncodeTiled(q) failed: %d", (int)r);
  tmap_store(key, *out);
  return SX_OK;
}

}  // namespace sx

using namespace sx;

extern "C" {

const char *sx_last_error(void) { return g_err; }

const char *sx_version(void) { return "sparsex-b200 0.3 (sm_100a; tcgen05/TMEM/TMA)"; }

uint64_t sx_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

sx_status sx_probe_pipe(int32_t pipe, int32_t iters, uint64_t *cycles, int32_t num_ctas, sx_stream stream) {
  if (!cycles || iters <= 0 || num_ctas <= 0) return set_error(SX_ERR_INVALID_ARG, "probe: bad arguments");
  return launch_probe(pipe, iters, reinterpret_cast<unsigned long long *>(cycles), num_ctas,
                      reinterpret_cast<cudaStream_t>(stream));
}

sx_status sx_check_batch(const sx_pool *pool, const sx_batch *batch, void *ws, size_t ws_bytes, sx_stream stream) {
  sx_status st = validate(pool, batch);
  if (st != SX_OK) return st;
  st = validate_ws(pool, batch, ws, ws_bytes);
  if (st != SX_OK) return st;
  return run_check_batch(pool, batch, ws, reinterpret_cast<cudaStream_t>(stream));
}

sx_status sx_check_rows(const sx_pool *pool, const sx_batch *batch, const int32_t *rows, const int32_t *rows_off,
                        int32_t max_rows, void *ws, size_t ws_bytes, sx_stream stream) {
  sx_status st = validate(pool, batch);
  if (st != SX_OK) return st;
  st = validate_ws(pool, batch, ws, ws_bytes);
  if (st != SX_OK) return st;
  if (!rows_off || max_rows < 0 || (max_rows > 0 && !rows)) return set_error(SX_ERR_INVALID_ARG, "check_rows: NULL array");
  return run_check_rows(batch, rows, rows_off, max_rows, ws, reinterpret_cast<cudaStream_t>(stream));
}

sx_status sx_workspace_size(const sx_pool *pool, const sx_batch *batch, size_t *bytes) {
  if (!bytes) return set_error(SX_ERR_INVALID_ARG, "bytes is NULL");
  if (!pool || !batch) return set_error(SX_ERR_INVALID_ARG, "pool or batch is NULL");
  if (pool->num_kv_heads <= 0 || pool->num_q_heads <= 0 || batch->total_tokens <= 0 || batch->num_segments < 0 ||
      batch->total_new < 0)
    return set_error(SX_ERR_INVALID_ARG, "sizes out of range");
  *bytes = ws_layout(pool, batch).total;
  return SX_OK;
}

sx_status sx_rope_realign_layers(const sx_pool *pools, int32_t num_layers, const sx_batch *batch, void *ws,
                                 size_t ws_bytes, sx_stream stream) {
  if (!pools || num_layers <= 0) return set_error(SX_ERR_INVALID_ARG, "pools is NULL or num_layers <= 0");
  // Copy-on-write state lives in the batch's v_block_table, page CONTENTS are per layer: after layer 0's scatter has
  // flipped an entry to the private page, the other layers' private pages would never be filled. A descriptor with
  // cow_private therefore describes the tables of ONE layer (one sx_batch per layer under COW).
  if (batch && batch->cow_private && num_layers > 1)
    return set_error(SX_ERR_UNSUPPORTED,
                     "copy-on-write tables are per layer: call sx_rope_realign with one sx_batch per layer");
  if (batch && batch->zero_copy)
    return set_error(SX_ERR_INVALID_ARG, "zero-copy mode: nothing to re-align (K is rotated as it is read)");
  for (int l = 0; l < num_layers; ++l) {
    sx_status st = validate(&pools[l], batch);
    if (st != SX_OK) return st;
    if (pools[l].num_kv_heads != pools[0].num_kv_heads || pools[l].num_blocks != pools[0].num_blocks)
      return set_error(SX_ERR_INVALID_ARG, "layer %d: pool shape differs from layer 0", l);
  }
  sx_status st = validate_ws(&pools[0], batch, ws, ws_bytes);
  if (st != SX_OK) return st;
  if (batch->num_segments == 0 || batch->total_seg_pages == 0) return SX_OK;
  WsLayout w = ws_layout(&pools[0], batch);
  return launch_realign(pools, num_layers, batch, reinterpret_cast<float2 *>(static_cast<char *>(ws) + w.rope_table),
                        reinterpret_cast<int4 *>(static_cast<char *>(ws) + w.page_desc),
                        reinterpret_cast<cudaStream_t>(stream));
}

sx_status sx_rope_realign(const sx_pool *pool, const sx_batch *batch, void *ws, size_t ws_bytes, sx_stream stream) {
  return sx_rope_realign_layers(pool, 1, batch, ws, ws_bytes, stream);
}

sx_status sx_scatter_kv(const sx_pool *pool, const sx_batch *batch, const void *k_fresh, const void *v_fresh,
                        const int32_t *rows, const int32_t *rows_off, int32_t max_rows, sx_stream stream) {
  sx_status st = validate(pool, batch);
  if (st != SX_OK) return st;
  if (max_rows < 0) return set_error(SX_ERR_INVALID_ARG, "max_rows < 0");
  if (max_rows == 0) return SX_OK;
  if (!k_fresh || !v_fresh || !rows || !rows_off) return set_error(SX_ERR_INVALID_ARG, "scatter: NULL array");
  if (misaligned(k_fresh) || misaligned(v_fresh)) return set_error(SX_ERR_MISALIGNED, "k_fresh / v_fresh not 16-B aligned");
  if (batch->zero_copy && !batch->cow_private)
    return set_error(SX_ERR_INVALID_ARG, "zero-copy mode: scatter needs cow_private (shared source pages are never written)");
  return launch_scatter(pool, batch, k_fresh, v_fresh, rows, rows_off, max_rows, reinterpret_cast<cudaStream_t>(stream));
}

sx_status sx_score_select_ex(const sx_pool *pool, const sx_batch *batch, const void *q_new, const float *lse_new,
                             int32_t lse_by_token, const int32_t *sel_off, const int32_t *rows_off,
                             int32_t overflow_blocks, int32_t tail_tokens, float *scores, int32_t *sel_idx,
                             int32_t *rows_R, int32_t *rows_off_out, void *ws, size_t ws_bytes, sx_stream stream) {
  sx_status st = validate(pool, batch);
  if (st != SX_OK) return st;
  st = validate_ws(pool, batch, ws, ws_bytes);
  if (st != SX_OK) return st;
  if (!sel_off || !rows_off || !sel_idx || !rows_R) return set_error(SX_ERR_INVALID_ARG, "score_select: NULL array");
  if (overflow_blocks < 0 || tail_tokens < 0)
    return set_error(SX_ERR_INVALID_ARG, "overflow_blocks / tail_tokens must be >= 0");
  if ((overflow_blocks > 0 || tail_tokens > 0) && !rows_off_out)
    return set_error(SX_ERR_INVALID_ARG, "rows_off_out is required with overflow / tail fallback (|R| is data dependent)");
  if (batch->total_new > 0 && !q_new) return set_error(SX_ERR_INVALID_ARG, "q_new is NULL");
  if (q_new && misaligned(q_new)) return set_error(SX_ERR_MISALIGNED, "q_new not 16-B aligned");
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  WsLayout w = ws_layout(pool, batch);
  char *base = static_cast<char *>(ws);
  float *partial = reinterpret_cast<float *>(base + w.partial);
  const float *lse = lse_new;
  if (lse_by_token != 0 && lse_by_token != 1) return set_error(SX_ERR_INVALID_ARG, "lse_by_token must be 0 or 1");
  int lse_splits = 1;
  ZcArgs zc;
  if (batch->total_new > 0) {
    st = zc_prepare(pool, batch, ws, s, &zc);
    if (st != SX_OK) return st;
    if (!lse) {  // sweep 1: row normaliser of Eq. (1) for the Sparse-Q rows
      float *lse_ws = reinterpret_cast<float *>(base + w.lse_new);
      lse_splits = sx::lse_splits(pool, batch);
      st = launch_lse(pool, batch, q_new, lse_ws, lse_splits, zc, s);
      if (st != SX_OK) return st;
      lse = lse_ws;
      lse_by_token = 0;
    }
    // sweep 2: column sums of A_sq (Eq. 2), one partial vector per KV head
    st = launch_colsum(pool, batch, q_new, lse, lse_by_token, lse_splits, partial,
                       reinterpret_cast<float2 *>(base + w.col_tab), zc, s);
    if (st != SX_OK) return st;
  } else {
    cudaError_t e = cudaMemsetAsync(partial, 0, sizeof(float) * (size_t)pool->num_kv_heads * batch->total_tokens, s);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "memset: %s", cudaGetErrorString(e));
  }
  float *sc = scores ? scores : reinterpret_cast<float *>(base + w.scores);
  return launch_select(pool, batch, partial, sel_off, rows_off, sc, sel_idx, rows_R, overflow_blocks, tail_tokens,
                       reinterpret_cast<int32_t *>(base + w.rows_tmp), reinterpret_cast<int32_t *>(base + w.rows_cnt),
                       rows_off_out, reinterpret_cast<int *>(base + w.sel_scratch), s);
}

sx_status sx_score_select(const sx_pool *pool, const sx_batch *batch, const void *q_new, const float *lse_new,
                          int32_t lse_by_token, const int32_t *sel_off, const int32_t *rows_off, float *scores, int32_t *sel_idx,
                          int32_t *rows_R, void *ws, size_t ws_bytes, sx_stream stream) {
  return sx_score_select_ex(pool, batch, q_new, lse_new, lse_by_token, sel_off, rows_off, 0, 0, scores, sel_idx, rows_R,
                            nullptr, ws, ws_bytes, stream);
}

sx_status sx_sparse_attn(const sx_pool *pool, const sx_batch *batch, int32_t mode, const void *q,
                         const int32_t *rows_R, const int32_t *rows_off, int32_t total_rows, void *out, float *lse,
                         void *ws, size_t ws_bytes, sx_stream stream) {
  sx_status st = validate(pool, batch);
  if (st != SX_OK) return st;
  if (mode < 0 || mode > 15)
    return set_error(SX_ERR_INVALID_ARG, "mode must be 0 (sparse rows) or 1 (full), optionally | SX_ATTN_* flags");
  const bool want_cuda_core = (mode & SX_ATTN_CUDA_CORE) != 0;
  // 2-CTA clusters: forced by a flag, else for batches of one request (measured: +1-2 % there, -5 % on batches)
  const bool want_cta_pair =
      (mode & SX_ATTN_CTA_PAIR) != 0 || ((mode & SX_ATTN_SINGLE_CTA) == 0 && batch->num_reqs == 1);
  const int mode_flags = mode;
  mode &= 1;
  if (total_rows < 0) return set_error(SX_ERR_INVALID_ARG, "total_rows < 0");
  if (total_rows == 0) return SX_OK;
  if (!q || !out) return set_error(SX_ERR_INVALID_ARG, "q / out is NULL");
  if (misaligned(q) || misaligned(out)) return set_error(SX_ERR_MISALIGNED, "q / out not 16-B aligned");
  cudaStream_t s = reinterpret_cast<cudaStream_t>(stream);
  if (mode == 1) {
    if (total_rows != batch->total_tokens)
      return set_error(SX_ERR_INVALID_ARG, "full mode: total_rows must equal total_tokens");
    rows_R = nullptr;
    rows_off = batch->tok_off;
  } else if (!rows_R || !rows_off) {
    return set_error(SX_ERR_INVALID_ARG, "rows_R / rows_off is NULL");
  }
  // Dispatch. BASELINE.json north_star asks for tcgen05 tiles only where GQA packing gives at least 64 query
  // rows per KV head and CUDA-core FMA paths below that. Measured on B200 (bench.py S6, S10) the padded
  // tensor-core tile with key splits is faster even at 4 pairs per KV head (52 us against 62 / 104 / 243 us for
  // 4 / 8 / 32 pairs over a 32K context), so it is the default for every row set; mode | SX_ATTN_CUDA_CORE
  // selects the CUDA-core kernels by the north_star rule (fewer than 64 pairs per KV head on average over the batch).
  const int g = pool->num_q_heads / pool->num_kv_heads;
  const bool allow_small = want_cuda_core;
  if (batch->zero_copy && batch->num_segments > 0) {
    // K tiles are rotated in shared memory by the softmax warpgroups of the single-CTA kernel: no CTA pairs
    if (want_cuda_core || (mode_flags & SX_ATTN_CTA_PAIR))
      return set_error(SX_ERR_UNSUPPORTED, "zero-copy mode: CUDA-core kernels / CTA pairs are not available");
    st = validate_ws(pool, batch, ws, ws_bytes);
    if (st != SX_OK) return st;
    ZcArgs zc;
    st = zc_prepare(pool, batch, ws, s, &zc);
    if (st != SX_OK) return st;
    // two query tiles per CTA fill the machine without key splits -> the shared-rotation form; else one tile per CTA
    int splits = attn_pv_splits(pool, batch, total_rows, 2);
    if (splits > 1) splits = attn_pv_splits(pool, batch, total_rows, 1);
    float *part = splits > 1 ? reinterpret_cast<float *>(static_cast<char *>(ws) + ws_layout(pool, batch).attn_part) : nullptr;
    return launch_attn(pool, batch, q, rows_R, rows_off, total_rows, out, lse, splits, part, false, zc, s);
  }
  if (allow_small && g <= 32 && (int64_t)total_rows * g < (int64_t)64 * batch->num_reqs) {
    st = validate_ws(pool, batch, ws, ws_bytes);
    if (st != SX_OK) return st;
    WsLayout w = ws_layout(pool, batch);
    return launch_attn_small(pool, batch, q, rows_R, rows_off, total_rows, out, lse,
                             reinterpret_cast<float *>(static_cast<char *>(ws) + w.small_part), s);
  }
  const int splits = attn_pv_splits(pool, batch, total_rows, 2);
  float *part = nullptr;
  if (splits > 1) {
    st = validate_ws(pool, batch, ws, ws_bytes);
    if (st != SX_OK) return st;
    part = reinterpret_cast<float *>(static_cast<char *>(ws) + ws_layout(pool, batch).attn_part);
  }
  return launch_attn(pool, batch, q, rows_R, rows_off, total_rows, out, lse, splits, part, want_cta_pair, ZcArgs(), s);
}

sx_status sx_sparse_attn_noalloc(const sx_pool *pool, const sx_batch *batch, const void *q, const int32_t *rows_R,
                                 const int32_t *rows_off, int32_t total_rows, void *out, float *lse,
                                 sx_stream stream) {
  sx_status st = validate(pool, batch);
  if (st != SX_OK) return st;
  if (total_rows < 0) return set_error(SX_ERR_INVALID_ARG, "total_rows < 0");
  if (total_rows == 0) return SX_OK;
  if (!q || !out || !rows_R || !rows_off) return set_error(SX_ERR_INVALID_ARG, "q / out / rows_R / rows_off is NULL");
  if (misaligned(q) || misaligned(out)) return set_error(SX_ERR_MISALIGNED, "q / out not 16-B aligned");
  if (batch->zero_copy && batch->num_segments > 0)
    return set_error(SX_ERR_UNSUPPORTED, "sx_sparse_attn_noalloc: zero-copy batches need the workspace (sx_sparse_attn)");
  return launch_attn_noalloc(pool, batch, q, rows_R, rows_off, total_rows, out, lse,
                             reinterpret_cast<cudaStream_t>(stream));
}

}  // extern "C"
